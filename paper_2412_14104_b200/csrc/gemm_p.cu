// gemm_p.cu -- the persistent 128x128 CTA tile of the tensor-GEMM (see gemm.cu for the operation):
//   C[b][cm(m)+cn(n)] (+)= alpha * sum_k A[b][am(m)+ak(k)] * B[b][bk(k)+bn(n)]
// on the FP64 tensor pipe (mma.sync m8n8k4 -> DMMA.8x8x4).  This is the kernel the bond swap
// (Table 1) and the O(r^2 chi^7) triad contraction (Eqs. 13-14) run on.
//
// One CTA per SM (16 warps, warp tile 32 x 32, 32 FP64 accumulators per thread) walks over output tiles
// blockIdx.x, blockIdx.x + gridDim.x, ...; the 3-stage cp.async pipeline (BK = 32, per-stage "full" /
// "empty" mbarriers) runs across tile boundaries, so the first operand tiles of the next output tile are
// in flight while the accumulators of the current one are written back: no pipeline fill / drain per
// output tile.
//
// Shared-memory layout of an operand tile (no padding, XOR swizzle on 16-byte chunks, chosen so that both
// the 16-byte cp.async writes and the 16-byte fragment reads are bank-conflict free):
//   k contiguous in global memory ("KF"):   [row][k], 32 doubles per row,
//                                           chunk (k/2) stored at (k/2) ^ ((row & 1) << 2)
//   free index contiguous ("FF"):           [k][row], 128 doubles per k line,
//                                           chunk (row/2) stored at (row/2) ^ h(k), h = bit1(k) | bit2(k) << 2
// Fragments are read with LDS.128, two DMMA operands per load (0.25 shared loads per DMMA instead of 0.5):
//   - DMMA number kk of a k group of 8 uses k = 8 g + 2 (lane % 4) + (kk % 2) -- the order of the summed
//     index is free --, so a KF row holds the operands of two consecutive DMMAs side by side;
//   - an FF tile assigns rows wm0 + 4 (lane / 4) + i to fragment i -- the assignment of tile rows to
//     fragment rows is free as long as the epilogue uses the same one --, so one k line holds the
//     operands of fragments i, i + 1 side by side.
#include <math.h>
#include <stdlib.h>

#include <algorithm>

#include "common.h"
#include "ctx.h"

namespace tatrg {

namespace {

constexpr int BM = 128, BN = 128, BK = 32, STAGES = 3, NT = 512;
constexpr int TILE = 128 * BK;   // doubles per operand stage
constexpr int RASTER_W = 12;

__device__ __forceinline__ void cp_async16(unsigned dst, const double *gsrc, int bytes)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(gsrc), "r"(bytes));
}
__device__ __forceinline__ void cp_async8(unsigned dst, const double *gsrc, int bytes)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(gsrc), "r"(bytes));
}
__device__ __forceinline__ void mbar_init(unsigned bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned bar)
{
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_on_cp_async(unsigned bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"(bar) : "memory");
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
// plain (non-volatile) 16-byte shared load: the compiler is free to hoist it above the DMMAs of the
// previous k group (the mbarrier wait / arrive asms carry a memory clobber and fence it in)
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

// offsets in doubles inside one operand stage
__device__ __forceinline__ int kf_off(int row, int k) { return row * BK + ((((k >> 1) ^ ((row & 1) << 2))) << 1) + (k & 1); }
__device__ __forceinline__ int ff_hash(int k) { return ((k >> 1) & 1) | (((k >> 2) & 1) << 2); }
__device__ __forceinline__ int ff_off(int k, int row) { return k * 128 + ((((row >> 1) ^ ff_hash(k))) << 1) + (row & 1); }

// Loader of one 128 x BK operand tile by the 512 threads.  KF: k is the contiguous index in global memory.
// VEC: 16-byte copies (pairs along the contiguous index), else 8-byte copies.
template <bool KF, bool VEC>
struct Loader {
    static constexpr int PER = VEC ? 4 : 8;   // copies per thread per tile
    // copy j of a thread lands DELTA * j doubles after copy 0 (the swizzle term does not depend on j)
    static constexpr int DELTA = KF ? (VEC ? 32 * BK : 16 * BK) : (VEC ? 32 : 16);
    unsigned fix[PER];                        // offsets of the free index (fixed over the k tiles of an output tile);
                                              // 32 bits: the host routes operands spanning >= 2^32 elements elsewhere
    const double *base;
    unsigned valid;                           // 2 bits per copy: valid elements along the free index (FF) / row valid (KF)
    int kl;                                   // this thread's (first) k inside the tile
    unsigned soff0;                           // byte offset of copy 0 inside a stage
    bool interior;                            // every copy of this thread is fully inside the operand along the free index

    // thread -> (k, free) coordinates of copy j
    __device__ __forceinline__ static int k_of(int t) { return KF ? (VEC ? (t & 15) * 2 : (t & 31)) : (t >> 4); }
    __device__ __forceinline__ static int f_of(int t, int j)
    {
        if (KF) return VEC ? (t >> 4) + 32 * j : (t >> 5) + 16 * j;
        return VEC ? ((t & 15) + 16 * j) * 2 : (t & 15) + 16 * j;
    }

    __device__ __forceinline__ void init_thread(int t)
    {
        kl = k_of(t);
        soff0 = 8u * (unsigned)(KF ? kf_off(f_of(t, 0), kl) : ff_off(kl, f_of(t, 0)));
    }

    __device__ __forceinline__ void init(const double *b, const Map4 &mfree, int f0, int F, int t)
    {
        base = b;
        valid = 0;
        interior = true;
#pragma unroll
        for (int j = 0; j < PER; ++j) {
            const int left = F - (f0 + f_of(t, j));
            const unsigned v = left <= 0 ? 0u : ((!KF && VEC) ? (left >= 2 ? 2u : 1u) : 1u);
            interior = interior && (v == ((!KF && VEC) ? 2u : 1u));
            valid |= v << (2 * j);
            fix[j] = v ? (unsigned)map_off(mfree, f0 + f_of(t, j)) : 0u;
        }
    }

    // kshift >= 0: the summed index is a composite of two legs, the faster one a power of two (2^kshift): shift and
    // mask instead of the integer divisions of map_off, which otherwise sit in front of every k tile's copies (2 % of
    // the kernel's time on the contraction shapes, whose summed index is such a composite).  (The same treatment of
    // the free-index and output maps, evaluated once per output tile, measured no gain.)
    __device__ __forceinline__ void load(unsigned stage_addr, const Map4 &mk, int kshift, int k0, int k_end) const
    {
        const int k_left = k_end - (k0 + kl);
        const unsigned kk = (unsigned)(k0 + kl);
        long long ko = 0;
        if (k_left > 0) {
            if (mk.n0 == TATRG_RADIX_INF)
                ko = (long long)kk * mk.s0;
            else if (kshift >= 0)
                ko = (long long)(kk & (mk.n0 - 1u)) * mk.s0 + (long long)(kk >> kshift) * mk.s1;
            else
                ko = map_off(mk, kk);
        }
        const unsigned dst0 = stage_addr + soff0;
        if (interior && k_left >= (KF && VEC ? 2 : 1)) {
            const double *src = base + ko;
#pragma unroll
            for (int j = 0; j < PER; ++j) {
                if (VEC)
                    cp_async16(dst0 + 8u * DELTA * j, src + fix[j], 16);
                else
                    cp_async8(dst0 + 8u * DELTA * j, src + fix[j], 8);
            }
            return;
        }
#pragma unroll
        for (int j = 0; j < PER; ++j) {
            const int v = (valid >> (2 * j)) & 3;
            int n;   // valid elements of this copy
            if (KF)
                n = v ? min(k_left, VEC ? 2 : 1) : 0;
            else
                n = k_left > 0 ? v : 0;
            n = max(n, 0);
            const double *src = n > 0 ? base + fix[j] + ko : base;
            if (VEC)
                cp_async16(dst0 + 8u * DELTA * j, src, n * 8);
            else
                cp_async8(dst0 + 8u * DELTA * j, src, n * 8);
        }
    }
};

struct TileCoord {
    int m0, n0, bz, split;
};

// per_z: live tiles of one (split, batch) slice.  lower_only (symmetric output, M = N): only the tiles on
// or below the diagonal are enumerated, row by row: index l -> (tm, tn <= tm), l = tm (tm + 1) / 2 + tn
template <bool TRI>
__device__ __forceinline__ TileCoord decode_tile(const GemmParams &p, int tile, int tiles_m, int per_z)
{
    TileCoord c;
    const int z = tile / per_z;
    const int r = tile - z * per_z;
    if (TRI) {
        // triangular B: column tile tn costs tn + 1 units.  Tiles come in pairs (tn, tiles_n - 1 - tn) of one
        // row band, every pair the same work; a CTA takes whole pairs (see next_tile in the kernel)
        const int half = p.tiles_n >> 1, q = r >> 1;
        const int tm = q / half, jp = q - tm * half;
        c.m0 = tm * BM;
        c.n0 = ((r & 1) ? p.tiles_n - 1 - jp : jp) * BN;
    } else if (p.lower_only) {
        int tm = (int)((sqrtf(8.0f * (float)r + 1.0f) - 1.0f) * 0.5f);
        while ((tm + 1) * (tm + 2) / 2 <= r) ++tm;
        while (tm * (tm + 1) / 2 > r) --tm;
        c.m0 = tm * BM;
        c.n0 = (r - tm * (tm + 1) / 2) * BN;
    } else {
        const int band = r / (RASTER_W * p.tiles_n);
        const int in_band = r - band * (RASTER_W * p.tiles_n);
        const int w = min(RASTER_W, tiles_m - band * RASTER_W);
        const int tn = in_band / w;
        c.n0 = tn * BN;
        c.m0 = (band * RASTER_W + (in_band - tn * w)) * BM;
    }
    c.split = z / p.batch;
    c.bz = z - c.split * p.batch;
    return c;
}

template <bool A_KF, bool B_KF, bool VEC, bool TRI>
__global__ void __launch_bounds__(NT, 1) tgemm_p_kernel(const __grid_constant__ GemmParams p, const int total_tiles, const int c_flags)
{
    extern __shared__ __align__(128) double smem[];
    __shared__ unsigned long long bars[2 * STAGES];
    const unsigned As = (unsigned)__cvta_generic_to_shared(smem);
    const unsigned Bs = As + STAGES * TILE * 8;
    const unsigned full0 = (unsigned)__cvta_generic_to_shared(bars);
    const unsigned empty0 = full0 + 8 * STAGES;

    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const int tiles_m = (p.M + BM - 1) / BM;
    const int per_z = p.lower_only ? tiles_m * (tiles_m + 1) / 2 : tiles_m * p.tiles_n;
    if (t == 0) {
#pragma unroll
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(full0 + 8 * s, NT);
            mbar_init(empty0 + 8 * s, NT);
        }
    }
    __syncthreads();

    const int wm0 = (warp & 3) * 32, wn0 = (warp >> 2) * 32;
    const int lr = lane >> 2, lk = lane & 3;
    // fragment read offsets (bytes) inside a stage, without the k-group term
    //   KF: row = w0 + 8 i + lr, chunk = (4 g + lk) ^ ((row & 1) << 2)  -> byte = row * 256 + ((32 g) ^ ((lr & 1) << 5)) * 2 + 16 lk ... folded below
    //   FF: k = 8 g + 2 lk + e, rows w0 + 4 lr + {0, 2}: chunk = (w0 / 2 + 2 lr + u) ^ h(lk)
    unsigned a_rd[2], b_rd[2];
    unsigned a_sx = 0, b_sx = 0;
    if (A_KF) {
        a_rd[0] = (unsigned)((wm0 + lr) * BK + 2 * lk) * 8u;
        a_rd[1] = 0;
        a_sx = (unsigned)(lr & 1) << 6;   // chunk bit 2 -> byte bit 6
    } else {
        const int h = (lk & 1) | ((lk >> 1) << 2);
        a_rd[0] = (unsigned)(2 * lk * 128 + ((((wm0 >> 1) + 2 * lr) ^ h) << 1)) * 8u;
        a_rd[1] = (unsigned)(2 * lk * 128 + ((((wm0 >> 1) + 2 * lr + 1) ^ h) << 1)) * 8u;
    }
    if (B_KF) {
        b_rd[0] = (unsigned)((wn0 + lr) * BK + 2 * lk) * 8u;
        b_rd[1] = 0;
        b_sx = (unsigned)(lr & 1) << 6;
    } else {
        const int h = (lk & 1) | ((lk >> 1) << 2);
        b_rd[0] = (unsigned)(2 * lk * 128 + ((((wn0 >> 1) + 2 * lr) ^ h) << 1)) * 8u;
        b_rd[1] = (unsigned)(2 * lk * 128 + ((((wn0 >> 1) + 2 * lr + 1) ^ h) << 1)) * 8u;
    }

    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    // ---- producer cursor
    auto pow2_shift = [](const Map4 &m) {
        return (m.n0 != TATRG_RADIX_INF && m.n1 == TATRG_RADIX_INF && (m.n0 & (m.n0 - 1u)) == 0u) ? __ffs((int)m.n0) - 1 : -1;
    };
    const int a_kshift = pow2_shift(p.ak), b_kshift = pow2_shift(p.bk);
    Loader<A_KF, VEC> la;
    Loader<B_KF, VEC> lb;
    la.init_thread(t);
    lb.init_thread(t);
    int p_tile = 0, p_kt = 0, p_nkt = 0, p_kbeg = 0, p_kend = 0;
    unsigned p_it = 0;
    auto k_range = [&](const TileCoord &c, int &kb, int &ke) {
        kb = 0;
        ke = p.K;
        if (p.ksplit > 1) {
            kb = min(p.K, c.split * p.ktiles_per_split * 16);
            ke = min(p.K, kb + p.ktiles_per_split * 16);
        }
        if (TRI) ke = min(ke, c.n0 + BN);   // B[k][n] = 0 for k > n
    };
    // tile walk of this CTA: blockIdx.x, + gridDim.x, ...; with a triangular B whole pairs (2 q, 2 q + 1)
    const int tile_first = TRI ? 2 * (int)blockIdx.x : (int)blockIdx.x;
    auto next_tile = [&](int tile) {
        if (TRI) return (tile & 1) ? tile + 2 * (int)gridDim.x - 1 : tile + 1;
        return tile + (int)gridDim.x;
    };
    auto prod_setup = [&]() {
        if (p_tile >= total_tiles) return;
        const TileCoord c = decode_tile<TRI>(p, p_tile, tiles_m, per_z);
        k_range(c, p_kbeg, p_kend);
        p_nkt = (p_kend - p_kbeg + BK - 1) / BK;
        p_kt = 0;
        la.init(p.A + map_off(p.ab, c.bz), p.am, c.m0, p.M, t);
        lb.init(p.B + map_off(p.bb, c.bz), p.bn, c.n0, p.N, t);
    };
    auto produce = [&]() {
        if (p_tile >= total_tiles) return;
        const unsigned slot = p_it % STAGES, use = p_it / STAGES;
        if (use >= 1) mbar_wait(empty0 + 8 * slot, (use - 1) & 1u);
        la.load(As + slot * (TILE * 8), p.ak, a_kshift, p_kbeg + p_kt * BK, p_kend);
        lb.load(Bs + slot * (TILE * 8), p.bk, b_kshift, p_kbeg + p_kt * BK, p_kend);
        mbar_arrive_on_cp_async(full0 + 8 * slot);
        ++p_it;
        if (++p_kt == p_nkt) {
            p_tile = next_tile(p_tile);
            prod_setup();
        }
    };
    p_tile = tile_first;
    prod_setup();
#pragma unroll 1
    for (int s = 0; s < STAGES - 1; ++s) produce();

    // ---- consumer
    unsigned it = 0;
    for (int c_tile = tile_first; c_tile < total_tiles; c_tile = next_tile(c_tile)) {
        const TileCoord tc = decode_tile<TRI>(p, c_tile, tiles_m, per_z);
        int kb, ke;
        k_range(tc, kb, ke);
        const int nkt = (ke - kb + BK - 1) / BK;
#pragma unroll 1
        for (int kt = 0; kt < nkt; ++kt, ++it) {
            const unsigned slot = it % STAGES;
            mbar_wait(full0 + 8 * slot, (it / STAGES) & 1u);
            const unsigned as = As + slot * (TILE * 8), bs = Bs + slot * (TILE * 8);
#pragma unroll
            for (int g = 0; g < BK / 8; ++g) {
                // operands are fetched in the order that keeps the fewest of them live (the register file is
                // full: 512 threads x 128): an FF tile one k at a time, a KF tile (which delivers two k per
                // load) whole for A and one fragment at a time for B
                if (A_KF) {
                    double a[4][2];
#pragma unroll
                    for (int i = 0; i < 4; ++i)
                        lds128(a[i][0], a[i][1], as + a_rd[0] + i * (8 * BK * 8) + (((unsigned)g << 6) ^ a_sx));
                    if (B_KF) {
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            double b0, b1;
                            lds128(b0, b1, bs + b_rd[0] + j * (8 * BK * 8) + (((unsigned)g << 6) ^ b_sx));
#pragma unroll
                            for (int i = 0; i < 4; ++i) dmma(acc[i][j][0], acc[i][j][1], a[i][0], b0);
#pragma unroll
                            for (int i = 0; i < 4; ++i) dmma(acc[i][j][0], acc[i][j][1], a[i][1], b1);
                        }
                    } else {
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            double b[4];
                            lds128(b[0], b[1], bs + b_rd[0] + (8 * g + e) * 1024);
                            lds128(b[2], b[3], bs + b_rd[1] + (8 * g + e) * 1024);
#pragma unroll
                            for (int i = 0; i < 4; ++i)
#pragma unroll
                                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i][e], b[j]);
                        }
                    }
                } else {
                    if (B_KF) {
                        double b[4][2];
#pragma unroll
                        for (int j = 0; j < 4; ++j)
                            lds128(b[j][0], b[j][1], bs + b_rd[0] + j * (8 * BK * 8) + (((unsigned)g << 6) ^ b_sx));
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            double a[4];
                            lds128(a[0], a[1], as + a_rd[0] + (8 * g + e) * 1024);
                            lds128(a[2], a[3], as + a_rd[1] + (8 * g + e) * 1024);
#pragma unroll
                            for (int i = 0; i < 4; ++i)
#pragma unroll
                                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j][e]);
                        }
                    } else {
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            double a[4], b[4];
                            lds128(a[0], a[1], as + a_rd[0] + (8 * g + e) * 1024);
                            lds128(a[2], a[3], as + a_rd[1] + (8 * g + e) * 1024);
                            lds128(b[0], b[1], bs + b_rd[0] + (8 * g + e) * 1024);
                            lds128(b[2], b[3], bs + b_rd[1] + (8 * g + e) * 1024);
#pragma unroll
                            for (int i = 0; i < 4; ++i)
#pragma unroll
                                for (int j = 0; j < 4; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
                        }
                    }
                }
            }
            mbar_arrive(empty0 + 8 * slot);   // this thread is done with the stage
            produce();                         // refill the slot of item it - 1 with item it + STAGES - 1
        }

        // ---- epilogue (the next tile's first stages are already in flight)
        // accumulator (i, j, e) <-> m = m0 + wm0 + (A_KF ? 8 i + lr : 4 lr + i),
        //                            n = n0 + wn0 + (B_KF ? 8 j + 2 lk + e : 8 lk + 4 e + j)
        // so a thread holds pairs of consecutive n: (j; e = 0, 1) for a KF B tile, (j = 2 u, 2 u + 1; e) for an FF
        // B tile -> 16-byte stores when C is contiguous along n (c_vec, checked on the host)
        double *Cb;
        Map4 cm, cn;
        double alpha = p.alpha;
        int accumulate = p.accumulate;
        bool vec = (c_flags & 1) != 0;
        if (p.ksplit > 1) {
            Cb = p.partial + ((long long)tc.split * p.batch + tc.bz) * (long long)p.M * p.N;
            cm = Map4{TATRG_RADIX_INF, TATRG_RADIX_INF, TATRG_RADIX_INF, 0, (long long)p.N, 0, 0, 0};
            cn = Map4{TATRG_RADIX_INF, TATRG_RADIX_INF, TATRG_RADIX_INF, 0, 1, 0, 0, 0};
            alpha = 1.0;
            accumulate = 0;
            vec = (c_flags & 2) != 0;
        } else {
            Cb = p.C + map_off(p.cb, tc.bz);
            cm = p.cm;
            cn = p.cn;
        }
        long long cno[4];   // offsets of the four column pairs of this thread
        int nfirst[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            nfirst[u] = tc.n0 + wn0 + (B_KF ? 8 * u + 2 * lk : 8 * lk + 4 * (u >> 1) + 2 * (u & 1));
            cno[u] = nfirst[u] < p.N ? (cn.n0 == TATRG_RADIX_INF ? (long long)nfirst[u] * cn.s0 : map_off(cn, nfirst[u])) : 0;
        }
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int m = tc.m0 + wm0 + (A_KF ? 8 * i + lr : 4 * lr + i);
            if (m < p.M) {
                double *Cr = Cb + (cm.n0 == TATRG_RADIX_INF ? (long long)m * cm.s0 : map_off(cm, m));
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    // the pair u of this thread: (v0, v1) at n = nfirst[u], nfirst[u] + 1
                    const double v0 = B_KF ? acc[i][u][0] : acc[i][2 * (u & 1)][u >> 1];
                    const double v1 = B_KF ? acc[i][u][1] : acc[i][2 * (u & 1) + 1][u >> 1];
                    if (vec && nfirst[u] + 1 < p.N) {
                        double2 *c = reinterpret_cast<double2 *>(Cr + cno[u]);
                        double2 w = make_double2(alpha * v0, alpha * v1);
                        if (accumulate) {
                            const double2 o = *c;
                            w.x += o.x;
                            w.y += o.y;
                        }
                        *c = w;
                    } else {
                        if (nfirst[u] < p.N) {
                            double *c = Cr + cno[u];
                            double w = alpha * v0;
                            if (accumulate) w += *c;
                            *c = w;
                        }
                        if (nfirst[u] + 1 < p.N) {
                            double *c = Cr + (vec ? cno[u] + 1 : map_off(cn, nfirst[u] + 1));
                            double w = alpha * v1;
                            if (accumulate) w += *c;
                            *c = w;
                        }
                    }
                }
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
        }
    }
    asm volatile("cp.async.wait_all;\n" ::);
}

bool even_or_inf(unsigned n) { return n == TATRG_RADIX_INF || (n & 1u) == 0; }
bool even(long long s) { return (s & 1LL) == 0; }
bool upper_even(const Map4 &m) { return even(m.s1) && even(m.s2) && even(m.s3); }
bool all_even(const Map4 &m) { return even(m.s0) && upper_even(m); }

template <bool A_KF, bool B_KF, bool VEC, bool TRI>
void launch_p(const GemmParams &p_in, int num_sms)
{
    constexpr size_t smem = (size_t)STAGES * 2 * TILE * sizeof(double);
    static bool attr_done = false;
    auto kern = tgemm_p_kernel<A_KF, B_KF, VEC, TRI>;
    if (!attr_done) {
        TATRG_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_done = true;
    }
    GemmParams p = p_in;
    const double flops = gemm_flops(p);
    p.tiles_n = (p.N + BN - 1) / BN;
    const long long tm = (p.M + BM - 1) / BM;
    if (p.lower_only && tm != p.tiles_n) fail(-22, "tensor_gemm: a symmetric (lower_only) output needs M = N");
    p.tri_b = TRI ? 1 : 0;
    const long long tiles = (p.lower_only ? tm * (tm + 1) / 2 : tm * p.tiles_n) * p.batch * (p.ksplit > 1 ? p.ksplit : 1);
    if (tiles > 0x3fffffffLL) fail(-22, "tensor_gemm: too many tiles");
    // while independent chains of small kernels run beside the step's big products, some SMs are left to them
    const unsigned grid = (unsigned)std::min<long long>(TRI ? tiles / 2 : tiles, std::max(1, num_sms - ctx().sm_reserve));
    // 16-byte stores of column pairs: bit 0 for C through its maps, bit 1 for the split-K partial sums
    int c_flags = 0;
    if (((uintptr_t)p.C & 15) == 0 && p.cn.s0 == 1 && even_or_inf(p.cn.n0) && upper_even(p.cn) && all_even(p.cm) && all_even(p.cb))
        c_flags |= 1;
    if ((p.N & 1) == 0 && ((uintptr_t)p.partial & 15) == 0) c_flags |= 2;
    const int slot = prof_begin(flops, 1);
    kern<<<grid, NT, smem, stream()>>>(p, (int)tiles, c_flags);
    prof_end(slot);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

// 16-byte copies along the contiguous index `fast` of an operand (the other index is `slow`)
bool vec_ok(const double *base, const Map4 &fast, const Map4 &slow, const Map4 &batch)
{
    return ((uintptr_t)base & 15) == 0 && fast.s0 == 1 && even_or_inf(fast.n0) && upper_even(fast) && all_even(slow) &&
           all_even(batch);
}

}  // namespace

// upper bound of map_off(m, i) over i < count (non-negative strides); < 0: a negative stride
static double map_span(const Map4 &m, long long count)
{
    if (m.s0 < 0 || m.s1 < 0 || m.s2 < 0 || m.s3 < 0) return -1.0;
    double span = 0.0, left = (double)count;
    const unsigned n[3] = {m.n0, m.n1, m.n2};
    const long long s[4] = {m.s0, m.s1, m.s2, m.s3};
    for (int l = 0; l < 4; ++l) {
        const double ext = (l < 3 && n[l] != TATRG_RADIX_INF && (double)n[l] < left) ? (double)n[l] : left;
        span += (ext - 1.0) * (double)s[l];
        if (l == 3 || n[l] == TATRG_RADIX_INF || (double)n[l] >= left) break;
        left = ceil(left / (double)n[l]);
    }
    return span;
}

bool tensor_gemm_persistent(const GemmParams &p, int num_sms)
{
    // the loader keeps the free-index offsets of an operand in 32 bits
    // the TMA-fed producer (gemm_tma.cu) is within 1-2 % of the cp.async producer but not ahead of it
    // (profiles/r2_gemm_tma_vs_cpasync.md): opt-in through tatrg_set_routes
    if ((ctx().routes & ROUTE_TMA_PRODUCER) && tensor_gemm_tma(p, num_sms)) return true;
    const double sa = map_span(p.am, p.M), sb = map_span(p.bn, p.N);
    if (sa < 0 || sb < 0 || sa >= 4294967295.0 || sb >= 4294967295.0) return false;
    const bool akf = p.a_kfast != 0, bkf = p.b_kfast != 0;
    const bool va = akf ? vec_ok(p.A, p.ak, p.am, p.ab) : vec_ok(p.A, p.am, p.ak, p.ab);
    const bool vb = bkf ? vec_ok(p.B, p.bk, p.bn, p.bb) : vec_ok(p.B, p.bn, p.bk, p.bb);
    // 16-byte copies along k need the k ranges of the split-K parts to start at even k: they do (units of 16)
    const bool vec = va && vb;
    // the triangular-B hint is taken (16-byte copy variants only) when the column tiles pair up; else the zeros
    // are multiplied as usual
    const bool tri = p.tri_b && vec && !p.lower_only && p.ksplit <= 1 && (((p.N + BN - 1) / BN) & 1) == 0;
    if (tri) {
        if (akf)
            bkf ? launch_p<true, true, true, true>(p, num_sms) : launch_p<true, false, true, true>(p, num_sms);
        else
            bkf ? launch_p<false, true, true, true>(p, num_sms) : launch_p<false, false, true, true>(p, num_sms);
        return true;
    }
    if (akf) {
        if (bkf)
            vec ? launch_p<true, true, true, false>(p, num_sms) : launch_p<true, true, false, false>(p, num_sms);
        else
            vec ? launch_p<true, false, true, false>(p, num_sms) : launch_p<true, false, false, false>(p, num_sms);
    } else {
        if (bkf)
            vec ? launch_p<false, true, true, false>(p, num_sms) : launch_p<false, true, false, false>(p, num_sms);
        else
            vec ? launch_p<false, false, true, false>(p, num_sms) : launch_p<false, false, false, false>(p, num_sms);
    }
    return true;
}

}  // namespace tatrg
