// gemm_tma.cu -- TMA-fed variant of the persistent 128x128 tensor-GEMM tile (gemm_p.cu) for operands that a
// rank-2 FP64 tensor map describes: A row-major [M][K] (k contiguous), B row-major [K][N] (n contiguous),
// C through its maps.  Same tile, same warp layout (16 warps x (32 x 32)), same BK = 32 x 3 stages; the
// difference is the producer: one thread issues cp.async.bulk.tensor copies (10 boxes
// per stage: A as two 128 x 16 boxes, B as eight 32 x 16 boxes, inner extent 128 bytes = the span of
// CU_TENSOR_MAP_SWIZZLE_128B) and arms the stage's "full" mbarrier with the byte count, instead of every
// thread issuing four 16-byte cp.async per operand with its own address arithmetic; a stage is refilled by
// the last warp that leaves it (a shared counter per stage instead of an "empty" mbarrier).
//
// Shared-memory layout = what the TMA unit writes under SWIZZLE_128B: inside a box, row i (128 bytes)
// holds its eight 16-byte chunks at chunk ^ (i & 7).  The fragment loads stay LDS.128 and conflict free by
// the choice of which tile row / column a lane's fragment element stands for (free, as in gemm_p.cu):
//   A box [row][16 k]:  fragment i, lane row lr  <->  tile row 8 i + pi(lr), pi(lr) = 4 (lr & 1) + (lr >> 1)
//                       (the two lane rows of a 16-byte phase differ in bit 2 of the row, hence in the chunk group)
//   B box [k][16 n]:    fragments 2 jj, 2 jj + 1, lane row lr  <->  columns 16 jj + 2 lr + {0, 1} of the warp tile
//                       (chunk lr of the k line; k = 8 g + 2 (lane % 4) + e supplies the XOR)
// PAPER.md:88-92 Eqs. 13-14 (the contraction these tiles serve); measured against the cp.async producer in
// profiles/r2_gemm_tma_vs_cpasync.md.
#include <cuda.h>

#include <algorithm>

#include "common.h"

namespace tatrg {

namespace {

constexpr int BM = 128, BN = 128, BK = 32, STAGES = 3, NT = 512;
constexpr int A_STAGE_BYTES = BM * BK * 8, B_STAGE_BYTES = BK * BN * 8;
constexpr int RASTER_W = 12;

__device__ __forceinline__ void mbar_init(unsigned bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n"
        " .reg .pred p;\n"
        "WAIT_%=:\n"
        " mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        " @p bra DONE_%=;\n"
        " bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d(unsigned dst, const CUtensorMap *map, int c0, int c1, unsigned bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::"r"(dst),
                 "l"(map), "r"(c0), "r"(c1), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void lds128(double &x, double &y, unsigned addr)
{
    const double2 v = *reinterpret_cast<const double2 *>(__cvta_shared_to_generic(addr));
    x = v.x;
    y = v.y;
}
__device__ __forceinline__ void dmma(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

__global__ void __launch_bounds__(NT, 1)
    tgemm_tma_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB,
                     const __grid_constant__ GemmParams p, const int total_tiles, const int c_vec)
{
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    __shared__ unsigned long long bars[STAGES];
    __shared__ int done[STAGES];
    // SWIZZLE_128B wants 1024-byte aligned boxes
    const unsigned base = ((unsigned)__cvta_generic_to_shared(smem_raw) + 1023u) & ~1023u;
    const unsigned As = base, Bs = base + STAGES * A_STAGE_BYTES;
    const unsigned full0 = (unsigned)__cvta_generic_to_shared(bars);

    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const int tiles_m = (p.M + BM - 1) / BM;
    if (t == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full0 + 8 * s, 1);
            done[s] = 0;
        }
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
    }
    __syncthreads();

    const int wm0 = (warp & 3) * 32, wn0 = (warp >> 2) * 32;
    const int lr = lane >> 2, lk = lane & 3;
    const int pi = 4 * (lr & 1) + (lr >> 1);
    // A: byte = h * 16384 + row * 128 + ((kk >> 1) ^ (row & 7)) * 16, row = wm0 + 8 i + pi, k pair (8 g + 2 lk): h = g >> 1,
    //    kk >> 1 = 4 (g & 1) + lk
    const unsigned a_row = (unsigned)(wm0 + pi) * 128u;
    // B: byte = (wn0 / 16 + jj) * 4096 + k * 128 + (lr ^ (k & 7)) * 16, k = 8 g + 2 lk + e
    const unsigned b_box = (unsigned)(wn0 >> 4) * 4096u;

    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    auto tile_coord = [&](int tile, int &m0, int &n0) {
        const int band = tile / (RASTER_W * p.tiles_n);
        const int in_band = tile - band * (RASTER_W * p.tiles_n);
        const int w = min(RASTER_W, tiles_m - band * RASTER_W);
        const int tn = in_band / w;
        n0 = tn * BN;
        m0 = (band * RASTER_W + (in_band - tn * w)) * BM;
    };
    const int nkt = (p.K + BK - 1) / BK;

    // ---- producer: the stage an item was read from is refilled, with the item STAGES ahead, by whichever warp
    // leaves it last (a shared counter per stage; no "empty" mbarrier, nobody waits): the copies go out the
    // moment the slot is free, two full k tiles before they are needed.  Every thread keeps the cursor.
    int p_tile = blockIdx.x, p_kt = 0, p_m0 = 0, p_n0 = 0;
    if (p_tile < total_tiles) tile_coord(p_tile, p_m0, p_n0);
    auto issue = [&](unsigned slot) {   // one thread
        const unsigned bar = full0 + 8 * slot;
        mbar_expect_tx(bar, A_STAGE_BYTES + B_STAGE_BYTES);
        const int k0 = p_kt * BK;
        tma_load_2d(As + slot * A_STAGE_BYTES, &mapA, k0, p_m0, bar);
        tma_load_2d(As + slot * A_STAGE_BYTES + 16384, &mapA, k0 + 16, p_m0, bar);
#pragma unroll
        for (int b = 0; b < 8; ++b) tma_load_2d(Bs + slot * B_STAGE_BYTES + b * 4096, &mapB, p_n0 + 16 * b, k0, bar);
    };
    auto advance = [&]() {
        if (++p_kt == nkt) {
            p_kt = 0;
            p_tile += gridDim.x;
            if (p_tile < total_tiles) tile_coord(p_tile, p_m0, p_n0);
        }
    };
#pragma unroll 1
    for (int s = 0; s < STAGES; ++s) {
        if (p_tile < total_tiles) {
            if (t == 0) issue(s);
            advance();
        }
    }

    unsigned it = 0;
    for (int c_tile = blockIdx.x; c_tile < total_tiles; c_tile += gridDim.x) {
        int m0, n0;
        tile_coord(c_tile, m0, n0);
#pragma unroll 1
        for (int kt = 0; kt < nkt; ++kt, ++it) {
            const unsigned slot = it % STAGES;
            mbar_wait(full0 + 8 * slot, (it / STAGES) & 1u);
            const unsigned as = As + slot * A_STAGE_BYTES + a_row, bs = Bs + slot * B_STAGE_BYTES + b_box;
#pragma unroll
            for (int g = 0; g < BK / 8; ++g) {
                double a[4][2];
#pragma unroll
                for (int i = 0; i < 4; ++i)
                    lds128(a[i][0], a[i][1], as + (g >> 1) * 16384 + i * 1024 + ((unsigned)((4 * (g & 1) + lk) ^ pi) << 4));
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    double b[4];
                    const int k = 8 * g + 2 * lk + e;
                    const unsigned boff = (unsigned)k * 128u + ((unsigned)(lr ^ (k & 7)) << 4);
                    lds128(b[0], b[1], bs + boff);
                    lds128(b[2], b[3], bs + 4096 + boff);
#pragma unroll
                    for (int i = 0; i < 4; ++i)
#pragma unroll
                        for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i][e], b[j]);
                }
            }
            // this warp is done with the stage; the last of the 16 warps refills it with item it + STAGES
            __syncwarp();
            if (p_tile < total_tiles) {
                if (lane == 0) {
                    __threadfence_block();
                    if (atomicAdd(&done[slot], 1) == NT / 32 - 1) {
                        done[slot] = 0;
                        __threadfence_block();
                        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
                        issue(slot);
                    }
                }
                advance();
            }
        }
        // ---- epilogue: acc (i, j, e) <-> m = m0 + wm0 + 8 i + pi, n = n0 + wn0 + 16 (j >> 1) + 4 lk + 2 e + (j & 1)
        double *Cb = p.C;
        long long cno[4];
        int nfirst[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {   // u = 2 jj + e: the pair (j = 2 jj, 2 jj + 1; e)
            nfirst[u] = n0 + wn0 + 16 * (u >> 1) + 4 * lk + 2 * (u & 1);
            cno[u] = nfirst[u] < p.N ? (p.cn.n0 == TATRG_RADIX_INF ? (long long)nfirst[u] * p.cn.s0 : map_off(p.cn, nfirst[u])) : 0;
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int m = m0 + wm0 + 8 * i + pi;
            if (m < p.M) {
                double *Cr = Cb + (p.cm.n0 == TATRG_RADIX_INF ? (long long)m * p.cm.s0 : map_off(p.cm, m));
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const double v0 = acc[i][2 * (u >> 1)][u & 1], v1 = acc[i][2 * (u >> 1) + 1][u & 1];
                    if (c_vec && nfirst[u] + 1 < p.N) {
                        double2 *c = reinterpret_cast<double2 *>(Cr + cno[u]);
                        double2 w = make_double2(p.alpha * v0, p.alpha * v1);
                        if (p.accumulate) {
                            const double2 o = *c;
                            w.x += o.x;
                            w.y += o.y;
                        }
                        *c = w;
                    } else {
                        if (nfirst[u] < p.N) {
                            double *c = Cr + cno[u];
                            double w = p.alpha * v0;
                            if (p.accumulate) w += *c;
                            *c = w;
                        }
                        if (nfirst[u] + 1 < p.N) {
                            double *c = Cr + map_off(p.cn, nfirst[u] + 1);
                            double w = p.alpha * v1;
                            if (p.accumulate) w += *c;
                            *c = w;
                        }
                    }
                }
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
        }
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void *f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
            return nullptr;
        fn = (EncodeTiledFn)f;
    }
    return fn;
}

bool single_level(const Map4 &m) { return m.n0 == TATRG_RADIX_INF; }

}  // namespace

// true if the launch was taken: A [M][K] with leading dimension lda (k contiguous), B [K][N] with ldb (n
// contiguous), no batch, no split-K, everything 16-byte aligned
bool tensor_gemm_tma(const GemmParams &p_in, int num_sms)
{
    const GemmParams &q = p_in;
    if (q.batch != 1 || q.ksplit > 1 || q.lower_only) return false;
    if (!single_level(q.am) || !single_level(q.ak) || !single_level(q.bk) || !single_level(q.bn)) return false;
    if (q.ak.s0 != 1 || q.bn.s0 != 1) return false;
    const long long lda = q.am.s0, ldb = q.bk.s0;
    if (lda < q.K || ldb < q.N || (lda & 1) || (ldb & 1)) return false;
    if (((uintptr_t)q.A & 15) || ((uintptr_t)q.B & 15)) return false;
    EncodeTiledFn enc = encode_fn();
    if (!enc) return false;
    CUtensorMap mapA, mapB;
    {
        cuuint64_t dims[2] = {(cuuint64_t)q.K, (cuuint64_t)q.M}, strides[1] = {(cuuint64_t)lda * 8};
        cuuint32_t box[2] = {16, 128}, estr[2] = {1, 1};
        if (enc(&mapA, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void *)q.A, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return false;
    }
    {
        cuuint64_t dims[2] = {(cuuint64_t)q.N, (cuuint64_t)q.K}, strides[1] = {(cuuint64_t)ldb * 8};
        cuuint32_t box[2] = {16, 32}, estr[2] = {1, 1};
        if (enc(&mapB, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, (void *)q.B, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return false;
    }
    constexpr size_t smem = (size_t)STAGES * (A_STAGE_BYTES + B_STAGE_BYTES) + 1024;
    static bool attr_done = false;
    if (!attr_done) {
        TATRG_CUDA_CHECK(cudaFuncSetAttribute(tgemm_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_done = true;
    }
    GemmParams p = p_in;
    p.tiles_n = (p.N + BN - 1) / BN;
    const long long tiles = (long long)((p.M + BM - 1) / BM) * p.tiles_n;
    if (tiles > 0x7fffffffLL) return false;
    const bool even_cn = p.cn.n0 == TATRG_RADIX_INF || !(p.cn.n0 & 1u);
    const int c_vec = (((uintptr_t)p.C & 15) == 0 && p.cn.s0 == 1 && even_cn && !(p.cn.s1 & 1) && !(p.cn.s2 & 1) && !(p.cn.s3 & 1) &&
                       !(p.cm.s0 & 1) && !(p.cm.s1 & 1) && !(p.cm.s2 & 1) && !(p.cm.s3 & 1))
                          ? 1
                          : 0;
    const unsigned grid = (unsigned)std::min<long long>(tiles, num_sms);
    const int slot = prof_begin(gemm_flops(p), 1);
    tgemm_tma_kernel<<<grid, NT, smem, stream()>>>(mapA, mapB, p, (int)tiles, c_vec);
    prof_end(slot);
    TATRG_LAUNCH_CHECK();
    count_launch();
    return true;
}

}  // namespace tatrg
