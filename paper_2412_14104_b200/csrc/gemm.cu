// gemm.cu -- the tensor-GEMM: one strided, batched FP64 contraction kernel on the sm_100a
// FP64 tensor pipe (mma.sync m8n8k4 -> SASS DMMA.8x8x4; tcgen05 has no f64 kind).
//
//   C[b][cm(m)+cn(n)] (+)= alpha * sum_k A[b][am(m)+ak(k)] * B[b][bk(k)+bn(n)]
//
// Every index (m, n, k, batch) is a mixed-radix composite of up to four tensor legs with
// arbitrary strides (Map4), so the leg permutations of the paper's contractions
// (PAPER.md:58-67 Eqs. 4-7, :90 Eqs. 13-14, the bond swap of :37) are folded into the
// cp.async gather addresses: no transpose kernel runs.  Operand tiles are staged in shared
// memory as [k][m] / [k][n] with a leading dimension = 4 (mod 16) doubles, which makes the
// 8-byte DMMA fragment loads bank-conflict free, through a STAGES-deep cp.async pipeline.
#include <math.h>
#include <stdlib.h>

#include <algorithm>

#include "common.h"

namespace tatrg {

namespace {

constexpr int BK = 16;
constexpr int RASTER_W = 12;

__device__ __forceinline__ void cp_async8(double *smem_dst, const double *gsrc, bool valid)
{
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    int sz = valid ? 8 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(d), "l"(gsrc), "r"(sz));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

__device__ __forceinline__ void dmma(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

template <int BM, int BN, int WM, int WN, int STAGES>
__global__ void __launch_bounds__((BM / WM) * (BN / WN) * 32)
    tgemm_kernel(const __grid_constant__ GemmParams p)
{
    constexpr int NW = (BM / WM) * (BN / WN), NT = NW * 32;
    constexpr int LDA = BM + 4, LDB = BN + 4;
    constexpr int A_PT = BM * BK / NT, B_PT = BN * BK / NT;
    constexpr int FM = WM / 8, FN = WN / 8;
    static_assert(NT % BM == 0 && NT % BN == 0 && NT % BK == 0, "loader layout");
    extern __shared__ double smem[];
    double *As = smem;
    double *Bs = smem + STAGES * BK * LDA;

    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    // tile order: bands of RASTER_W row tiles, row tile fastest inside a band, so that the CTAs
    // resident at one time cover a compact block of C and their operand tiles are shared in L2
    int tile_m, tile_n;
    {
        const int tiles_m = (p.M + BM - 1) / BM;
        const int band = blockIdx.x / (RASTER_W * p.tiles_n);
        const int in_band = blockIdx.x - band * (RASTER_W * p.tiles_n);
        const int w = min(RASTER_W, tiles_m - band * RASTER_W);
        tile_n = in_band / w;
        tile_m = band * RASTER_W + (in_band - tile_n * w);
    }
    const int m0 = tile_m * BM, n0 = tile_n * BN;
    if (p.lower_only && n0 >= m0 + BM) return;   // tile strictly above the diagonal of a symmetric output
    int bz = blockIdx.z;
    const int split = bz / p.batch;
    bz -= split * p.batch;

    const double *Ab = p.A + map_off(p.ab, bz);
    const double *Bb = p.B + map_off(p.bb, bz);

    int kt0 = 0, kt1 = (p.K + BK - 1) / BK;
    if (p.ksplit > 1) {
        kt0 = split * p.ktiles_per_split;
        kt1 = min(kt1, kt0 + p.ktiles_per_split);
    }
    const int nkt = max(kt1 - kt0, 0);

    // ---- loader state: (fast, slow) local tile coordinates of the elements this thread moves
    // A tile is BM x BK; a_kfast: fast = k (BK), slow = m; else fast = m (BM), slow = k.
    long long a_fix[A_PT];   // offsets that do not change with the k tile (a_kfast: rows)
    bool a_ok[A_PT];
    long long a_base = 0;    // !a_kfast: am(row) of this thread
    bool a_base_ok = true;
    if (p.a_kfast) {
#pragma unroll
        for (int u = 0; u < A_PT; ++u) {
            int ml = t / BK + (NT / BK) * u;
            a_ok[u] = (m0 + ml) < p.M;
            a_fix[u] = a_ok[u] ? map_off(p.am, m0 + ml) : 0;
        }
    } else {
        int ml = t % BM;
        a_base_ok = (m0 + ml) < p.M;
        a_base = a_base_ok ? map_off(p.am, m0 + ml) : 0;
    }
    long long b_fix[B_PT];
    bool b_ok[B_PT];
    long long b_base = 0;
    bool b_base_ok = true;
    if (p.b_kfast) {
#pragma unroll
        for (int u = 0; u < B_PT; ++u) {
            int nl = t / BK + (NT / BK) * u;
            b_ok[u] = (n0 + nl) < p.N;
            b_fix[u] = b_ok[u] ? map_off(p.bn, n0 + nl) : 0;
        }
    } else {
        int nl = t % BN;
        b_base_ok = (n0 + nl) < p.N;
        b_base = b_base_ok ? map_off(p.bn, n0 + nl) : 0;
    }

    auto load_tile = [&](int stage, int kt) {
        const int k0 = kt * BK;
        double *as = As + stage * BK * LDA;
        double *bs = Bs + stage * BK * LDB;
        if (p.a_kfast) {
            int kl = t % BK;
            bool kok = (k0 + kl) < p.K;
            long long ko = kok ? map_off_k(p.ak, k0 + kl) : 0;
#pragma unroll
            for (int u = 0; u < A_PT; ++u) {
                int ml = t / BK + (NT / BK) * u;
                bool ok = kok && a_ok[u];
                cp_async8(as + kl * LDA + ml, ok ? Ab + a_fix[u] + ko : p.A, ok);
            }
        } else {
            int ml = t % BM;
#pragma unroll
            for (int u = 0; u < A_PT; ++u) {
                int kl = t / BM + (NT / BM) * u;
                bool ok = a_base_ok && (k0 + kl) < p.K;
                long long ko = ok ? map_off_k(p.ak, k0 + kl) : 0;
                cp_async8(as + kl * LDA + ml, ok ? Ab + a_base + ko : p.A, ok);
            }
        }
        if (p.b_kfast) {
            int kl = t % BK;
            bool kok = (k0 + kl) < p.K;
            long long ko = kok ? map_off_k(p.bk, k0 + kl) : 0;
#pragma unroll
            for (int u = 0; u < B_PT; ++u) {
                int nl = t / BK + (NT / BK) * u;
                bool ok = kok && b_ok[u];
                cp_async8(bs + kl * LDB + nl, ok ? Bb + b_fix[u] + ko : p.B, ok);
            }
        } else {
            int nl = t % BN;
#pragma unroll
            for (int u = 0; u < B_PT; ++u) {
                int kl = t / BN + (NT / BN) * u;
                bool ok = b_base_ok && (k0 + kl) < p.K;
                long long ko = ok ? map_off_k(p.bk, k0 + kl) : 0;
                cp_async8(bs + kl * LDB + nl, ok ? Bb + b_base + ko : p.B, ok);
            }
        }
    };

    double acc[FM][FN][2];
#pragma unroll
    for (int i = 0; i < FM; ++i)
#pragma unroll
        for (int j = 0; j < FN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    const int wm0 = (warp % (BM / WM)) * WM, wn0 = (warp / (BM / WM)) * WN;
    const int lr = lane >> 2, lk = lane & 3;

#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nkt) load_tile(s, kt0 + s);
        cp_async_commit();
    }
    for (int it = 0; it < nkt; ++it) {
        cp_async_wait<STAGES - 2>();
        __syncthreads();
        {
            int nx = it + STAGES - 1;
            if (nx < nkt) load_tile(nx % STAGES, kt0 + nx);
            cp_async_commit();
        }
        const double *as = As + (it % STAGES) * BK * LDA + wm0 + lr;
        const double *bs = Bs + (it % STAGES) * BK * LDB + wn0 + lr;
#pragma unroll
        for (int kk = 0; kk < BK / 4; ++kk) {
            double a[FM], b[FN];
#pragma unroll
            for (int i = 0; i < FM; ++i) a[i] = as[(kk * 4 + lk) * LDA + i * 8];
#pragma unroll
            for (int j = 0; j < FN; ++j) b[j] = bs[(kk * 4 + lk) * LDB + j * 8];
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    cp_async_wait<0>();

    // ---- epilogue
    if (p.ksplit > 1) {
        double *P = p.partial + ((long long)split * p.batch + bz) * (long long)p.M * p.N;
#pragma unroll
        for (int i = 0; i < FM; ++i) {
            int m = m0 + wm0 + i * 8 + lr;
            if (m >= p.M) continue;
#pragma unroll
            for (int j = 0; j < FN; ++j) {
                int n = n0 + wn0 + j * 8 + lk * 2;
                if (n < p.N) P[(long long)m * p.N + n] = acc[i][j][0];
                if (n + 1 < p.N) P[(long long)m * p.N + n + 1] = acc[i][j][1];
            }
        }
        return;
    }
    double *Cb = p.C + map_off(p.cb, bz);
    long long cno[FN][2];
#pragma unroll
    for (int j = 0; j < FN; ++j) {
        int n = n0 + wn0 + j * 8 + lk * 2;
        cno[j][0] = n < p.N ? map_off(p.cn, n) : -1;
        cno[j][1] = n + 1 < p.N ? map_off(p.cn, n + 1) : -1;
    }
#pragma unroll
    for (int i = 0; i < FM; ++i) {
        int m = m0 + wm0 + i * 8 + lr;
        if (m >= p.M) continue;
        double *Cr = Cb + map_off(p.cm, m);
#pragma unroll
        for (int j = 0; j < FN; ++j) {
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                if (cno[j][e] < 0) continue;
                double v = p.alpha * acc[i][j][e];
                if (p.accumulate) v += Cr[cno[j][e]];
                Cr[cno[j][e]] = v;
            }
        }
    }
}

// partial[ksplit][batch][M][N] -> C via the maps
__global__ void splitk_reduce_kernel(const __grid_constant__ GemmParams p)
{
    long long total = (long long)p.batch * p.M * p.N;
    long long mn = (long long)p.M * p.N;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x) {
        double s = 0.0;
        for (int k = 0; k < p.ksplit; ++k) s += p.partial[k * total + i];
        int b = (int)(i / mn);
        long long r = i - b * mn;
        int m = (int)(r / p.N), n = (int)(r - (long long)m * p.N);
        double *c = p.C + map_off(p.cb, b) + map_off(p.cm, m) + map_off(p.cn, n);
        double v = p.alpha * s;
        if (p.accumulate) v += *c;
        *c = v;
    }
}

template <int BM, int BN, int WM, int WN, int STAGES>
void launch_cfg(const GemmParams &p_in)
{
    constexpr int NT = (BM / WM) * (BN / WN) * 32;
    constexpr size_t smem = (size_t)STAGES * BK * ((BM + 4) + (BN + 4)) * sizeof(double);
    static bool attr_done = false;
    auto kern = tgemm_kernel<BM, BN, WM, WN, STAGES>;
    if (!attr_done) {
        TATRG_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_done = true;
    }
    GemmParams p = p_in;
    p.tiles_n = (p.N + BN - 1) / BN;
    const long long tiles = (long long)((p.M + BM - 1) / BM) * p.tiles_n;
    if (tiles > 0x7fffffffLL) fail(-22, "tensor_gemm: too many tiles");
    dim3 grid((unsigned)tiles, 1, p.batch * (p.ksplit > 1 ? p.ksplit : 1));
    const int slot = prof_begin(gemm_flops(p), BM == 128);
    kern<<<grid, NT, smem, stream()>>>(p);
    prof_end(slot);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

}  // namespace

static int g_num_sms = 0;

void tensor_gemm(GemmParams p)
{
    if (p.M <= 0 || p.N <= 0 || p.batch <= 0) return;
    if (p.K <= 0) fail(-22, "tensor_gemm: K must be >= 1");
    if (!g_num_sms) {
        int dev = 0;
        TATRG_CUDA_CHECK(cudaGetDevice(&dev));
        TATRG_CUDA_CHECK(cudaDeviceGetAttribute(&g_num_sms, cudaDevAttrMultiProcessorCount, dev));
    }
    count_flops(gemm_flops(p));
    if (tensor_gemm_ts(p)) return;   // tall-and-skinny: streaming kernels (HBM-bound)
    // tile choice: 128x128 when it fills the machine (with split-K when the summed index is long),
    // 128x64 for outputs at most 64 columns wide with enough rows, else the 64x64 tile
    int ktiles = (p.K + BK - 1) / BK;
    long long big_tiles = (long long)((p.M + 127) / 128) * ((p.N + 127) / 128) * p.batch;
    const int max_split = ktiles / 8 < 512 ? ktiles / 8 : 512;
    bool big = p.M >= 96 && p.N >= 96 &&
               (big_tiles * 5 >= 4LL * g_num_sms || big_tiles * (long long)(max_split > 1 ? max_split : 1) >= 2LL * g_num_sms);
    // a short summed index (one or two k tiles) never fills the pipeline: two co-resident 128x64 CTAs per
    // SM hide each other's load and store phases (measured 0.37 -> 0.30 ms on the K = 32 product E M^(4))
    if (big && p.K <= 64) big = false;
    const bool mid = !big && p.N >= 17 && p.M >= 96 && (p.N <= 64 || p.K <= 64);
    long long tiles = big ? big_tiles
                          : mid ? (long long)((p.M + 127) / 128) * ((p.N + 63) / 64) * p.batch
                                : (long long)((p.M + 63) / 64) * ((p.N + 63) / 64) * p.batch;
    if (p.lower_only) {   // only the tiles that touch the lower triangle do work
        const int bm = (big || mid) ? 128 : 64, bn = big ? 128 : 64;
        const int tn = (p.N + bn - 1) / bn;
        long long cnt = 0;
        for (int m0 = 0; m0 < p.M; m0 += bm) cnt += std::min(tn, (m0 + bm - 1) / bn + 1);
        tiles = cnt * p.batch;
    }
    p.ksplit = 1;
    p.ktiles_per_split = ktiles;
    p.partial = nullptr;
    size_t mark = ws_mark();
    // split-K: the number of splits that minimises a simple cost model, in units of one k tile of 16:
    // waves of resident CTAs x (k tiles per CTA + a fixed per-CTA cost for the pipeline fill and the
    // epilogue) + the second pass over the partial sums
    const long long slots = (long long)g_num_sms * (big ? 1 : mid ? 2 : 3);
    if (max_split > 1) {
        const double fixed = 4.0, reduce_per_split = (double)p.M * p.N * p.batch / 2.0e6;
        auto cost = [&](int ks) {
            const double waves = ceil((double)tiles * ks / (double)slots);
            return waves * (ceil((double)ktiles / ks) + fixed) + (ks > 1 ? ks * reduce_per_split + 2.0 : 0.0);
        };
        int ks = 1;
        double best = cost(1);
        for (int c = 2; c <= max_split; ++c) {
            const double e = cost(c);
            if (e < best * 0.97) {
                best = e;
                ks = c;
            }
        }
        if (ks > 1) {
            p.ktiles_per_split = (ktiles + ks - 1) / ks;
            p.ksplit = (ktiles + p.ktiles_per_split - 1) / p.ktiles_per_split;
            if ((long long)p.batch * p.ksplit > 65535) fail(-22, "tensor_gemm: batch*ksplit too large");
            p.partial = ws_doubles((long long)p.ksplit * p.batch * p.M * p.N);
        }
    }
    if ((long long)p.batch * p.ksplit > 65535) fail(-22, "tensor_gemm: batch too large for grid.z");
    prof_shape(p.M, p.N, p.K, p.batch, p.ksplit);
    if (big) {
        if (!tensor_gemm_persistent(p, g_num_sms)) tensor_gemm_big(p, 128);
    }
    else if (mid)
        tensor_gemm_big(p, 64);
    else
        launch_cfg<64, 64, 32, 32, 4>(p);
    if (p.ksplit > 1) {
        long long total = (long long)p.batch * p.M * p.N;
        int blocks = (int)((total + 255) / 256 < 4LL * g_num_sms ? (total + 255) / 256 : 4LL * g_num_sms);
        splitk_reduce_kernel<<<blocks, 256, 0, stream()>>>(p);
        TATRG_LAUNCH_CHECK();
        count_launch();
    }
    ws_release(mark);
}

// ---------------------------------------------------------------------------------------
// FP64 peak probe: register-resident loops, no memory traffic.
// mode 0: DMMA.8x8x4 only, 1: DFMA only, 2: both interleaved.
__global__ void __launch_bounds__(256) probe_kernel(int mode, int iters, double *sink)
{
    double a = 1.0 + threadIdx.x * 1e-9, b = 1.0 - threadIdx.x * 1e-9;
    double c[16][2];
    double f[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
        c[i][0] = c[i][1] = 0.0;
        f[i] = i;
    }
    for (int it = 0; it < iters; ++it) {
        if (mode == 0 || mode == 2) {
#pragma unroll
            for (int i = 0; i < 16; ++i) dmma(c[i][0], c[i][1], a, b);
        }
        if (mode == 1 || mode == 2) {
#pragma unroll
            for (int i = 0; i < 16; ++i) f[i] = fma(f[i], a, b);
        }
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += c[i][0] + c[i][1] + f[i];
    if (s == 123.456) sink[0] = s;
}

double probe_fp64_peak(int mode, int iters)
{
    int dev = 0, sms = 0;
    TATRG_CUDA_CHECK(cudaGetDevice(&dev));
    TATRG_CUDA_CHECK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double *sink = ws_doubles(1);
    const int blocks = sms * 4, threads = 256;
    cudaEvent_t e0, e1;
    TATRG_CUDA_CHECK(cudaEventCreate(&e0));
    TATRG_CUDA_CHECK(cudaEventCreate(&e1));
    probe_kernel<<<blocks, threads, 0, stream()>>>(mode, iters / 4 + 1, sink);  // warm-up
    TATRG_CUDA_CHECK(cudaEventRecord(e0, stream()));
    probe_kernel<<<blocks, threads, 0, stream()>>>(mode, iters, sink);
    TATRG_CUDA_CHECK(cudaEventRecord(e1, stream()));
    TATRG_CUDA_CHECK(cudaEventSynchronize(e1));
    TATRG_LAUNCH_CHECK();
    float ms = 0;
    TATRG_CUDA_CHECK(cudaEventElapsedTime(&ms, e0, e1));
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    double warps = (double)blocks * threads / 32;
    double flops = 0;
    if (mode == 0 || mode == 2) flops += warps * iters * 16.0 * (8 * 8 * 4 * 2);
    if (mode == 1 || mode == 2) flops += warps * iters * 16.0 * 32 * 2;
    return flops / (ms * 1e-3) / 1e12;
}

}  // namespace tatrg
