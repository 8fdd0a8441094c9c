// ts.cu -- the two tall-and-skinny shapes of the tensor-GEMM that are bound by HBM, not by the
// tensor pipe: at most 64 columns on both small sides, >= 16384 rows.  They are the passes over the
// chi^4 x chi factors of the canonical form (Q_Phi, Q_Psi, A = Q u, the gauge projection)
// and of the Cholesky-QR passes of the RSVD blocks:
//
//   ts_apply:  C[cm(r) + j]     (+)= alpha sum_c A[am(r) + c] B[bk(c) + bn(j)]     rows x K times K x N
//   ts_dot:    C[cm(i) + cn(j)] (+)= alpha sum_r A[ak(r) + i] B[bk(r) + j]         (M x rows)(rows x N)
//
// Each row is read once from HBM in coalesced 8-byte runs into shared memory; the small operand /
// the accumulators stay on chip.  ts_dot writes one partial per CTA and a second kernel adds them
// in a fixed order (deterministic, like the split-K of gemm.cu).
#include <algorithm>

#include "common.h"

namespace tatrg {

namespace {

constexpr int TS_NT = 256;
constexpr int TS_ROWS = 128;   // rows per tile of ts_apply
constexpr int TD_ROWS = 64;    // rows per tile of ts_dot

// ---------------------------------------------------------------------------------------
template <int NH>   // the N <= 2 NH columns are split over four threads; each thread owns two rows
__global__ void __launch_bounds__(TS_NT) ts_apply_kernel(const __grid_constant__ GemmParams p)
{
    extern __shared__ double sm[];
    __shared__ long long offA[TS_ROWS], offC[TS_ROWS];
    const int K = p.K, N = p.N;
    const int ldx = K | 1;
    double *Xs = sm;                         // [TS_ROWS][ldx]
    double *Ws = sm + TS_ROWS * max(ldx, (2 * NH) | 1);   // [K][2 * NH]
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    for (int i = t; i < K * 2 * NH; i += TS_NT) {
        const int c = i / (2 * NH), j = i - c * 2 * NH;
        Ws[i] = (j < N) ? p.B[map_off(p.bk, c) + map_off(p.bn, j)] : 0.0;
    }
    const int tiles = (p.M + TS_ROWS - 1) / TS_ROWS;
    for (int tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
        const int r0 = tile * TS_ROWS;
        __syncthreads();
        // rows of this tile, coalesced along the contiguous column index
        // row offsets of the tile: one mixed-radix decomposition per thread instead of one per lane and row
        if (t < TS_ROWS)
            offA[t] = (r0 + t < p.M) ? map_off(p.am, r0 + t) : -1;
        else
            offC[t - TS_ROWS] = (r0 + t - TS_ROWS < p.M) ? map_off(p.cm, r0 + t - TS_ROWS) : -1;
        __syncthreads();
        {   // K <= 32: one element per lane and row; all loads of the tile are issued before the first use
            constexpr int RPW = TS_ROWS / (TS_NT / 32);
            double v[RPW];
#pragma unroll
            for (int i = 0; i < RPW; ++i) {
                const long long o = offA[warp + (TS_NT / 32) * i];
                v[i] = (o >= 0 && lane < K) ? p.A[o + lane] : 0.0;
            }
#pragma unroll
            for (int i = 0; i < RPW; ++i)
                if (lane < K) Xs[(warp + (TS_NT / 32) * i) * ldx + lane] = v[i];
        }
        __syncthreads();
        // thread = (row pair rp, rp + 64; quarter of the columns): every small-operand read feeds two rows
        constexpr int NQ = NH / 2;
        const int rp = t & 63, quarter = t >> 6;
        double acc0[NQ], acc1[NQ];
#pragma unroll
        for (int j = 0; j < NQ; ++j) acc0[j] = acc1[j] = 0.0;
        const double *x0r = Xs + rp * ldx, *x1r = Xs + (rp + 64) * ldx;
        const double *wq = Ws + quarter * NQ;
        for (int c = 0; c < K; ++c) {
            const double x0 = x0r[c], x1 = x1r[c];
            const double2 *w2 = reinterpret_cast<const double2 *>(wq + c * 2 * NH);
#pragma unroll
            for (int j = 0; j < NQ / 2; ++j) {
                const double2 w = w2[j];
                acc0[2 * j] = fma(x0, w.x, acc0[2 * j]);
                acc0[2 * j + 1] = fma(x0, w.y, acc0[2 * j + 1]);
                acc1[2 * j] = fma(x1, w.x, acc1[2 * j]);
                acc1[2 * j + 1] = fma(x1, w.y, acc1[2 * j + 1]);
            }
        }
        // results through shared memory (the X tile is dead), then whole rows per warp: coalesced stores
        __syncthreads();
        double *Ys = Xs;                     // [TS_ROWS][ldy]
        const int ldy = (2 * NH) | 1;
#pragma unroll
        for (int j = 0; j < NQ; ++j) {
            Ys[rp * ldy + quarter * NQ + j] = acc0[j];
            Ys[(rp + 64) * ldy + quarter * NQ + j] = acc1[j];
        }
        __syncthreads();
        for (int rr = warp; rr < TS_ROWS; rr += TS_NT / 32) {
            if (offC[rr] >= 0) {
                double *dst = p.C + offC[rr];
                for (int n = lane; n < N; n += 32) {
                    double v = p.alpha * Ys[rr * ldy + n];
                    if (p.accumulate) v += dst[n];
                    dst[n] = v;
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------
// Both small sides padded to W = 8 F <= 32.  The 256 threads form 4 row groups of 8 x 8 threads: group g
// takes the rows rr = g (mod 4) of a tile, thread (ti, tj) of a group owns the F x F outputs
// (ti + 8 a, tj + 8 b): 2 F shared-memory loads feed F^2 FMAs.  The groups are added at the end.
template <int F>
__global__ void __launch_bounds__(TS_NT) ts_dot_kernel(const __grid_constant__ GemmParams p, double *__restrict__ partial)
{
    extern __shared__ double sm[];
    __shared__ long long offA[TD_ROWS], offB[TD_ROWS];
    const int M = p.M, N = p.N;
    constexpr int W = 8 * F;
    constexpr int LD = W + 1;
    double *Xs = sm;                         // [TD_ROWS][LD]
    double *Zs = sm + TD_ROWS * LD;
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const int grp = t >> 6, ti = (t >> 3) & 7, tj = t & 7;
    double acc[F][F];
#pragma unroll
    for (int a = 0; a < F; ++a)
#pragma unroll
        for (int b = 0; b < F; ++b) acc[a][b] = 0.0;
    const int tiles = (p.K + TD_ROWS - 1) / TD_ROWS;
    for (int tile = blockIdx.x; tile < tiles; tile += gridDim.x) {
        const int r0 = tile * TD_ROWS;
        __syncthreads();
        if (t < TD_ROWS)
            offA[t] = (r0 + t < p.K) ? map_off(p.ak, r0 + t) : -1;
        else if (t < 2 * TD_ROWS)
            offB[t - TD_ROWS] = (r0 + t - TD_ROWS < p.K) ? map_off(p.bk, r0 + t - TD_ROWS) : -1;
        __syncthreads();
        {   // W <= 32: one element per lane, row and operand; loads first, then the shared-memory stores
            constexpr int RPW = TD_ROWS / (TS_NT / 32);
            double vx[RPW], vz[RPW];
#pragma unroll
            for (int i = 0; i < RPW; ++i) {
                const long long oa = offA[warp + (TS_NT / 32) * i], ob = offB[warp + (TS_NT / 32) * i];
                vx[i] = (oa >= 0 && lane < M) ? p.A[oa + lane] : 0.0;
                vz[i] = (ob >= 0 && lane < N) ? p.B[ob + lane] : 0.0;
            }
#pragma unroll
            for (int i = 0; i < RPW; ++i)
                if (lane < W) {
                    Xs[(warp + (TS_NT / 32) * i) * LD + lane] = vx[i];
                    Zs[(warp + (TS_NT / 32) * i) * LD + lane] = vz[i];
                }
        }
        __syncthreads();
#pragma unroll 4
        for (int rr = grp; rr < TD_ROWS; rr += 4) {
            double x[F], z[F];
#pragma unroll
            for (int a = 0; a < F; ++a) x[a] = Xs[rr * LD + ti + 8 * a];
#pragma unroll
            for (int b = 0; b < F; ++b) z[b] = Zs[rr * LD + tj + 8 * b];
#pragma unroll
            for (int a = 0; a < F; ++a)
#pragma unroll
                for (int b = 0; b < F; ++b) acc[a][b] = fma(x[a], z[b], acc[a][b]);
        }
    }
    // add the four row groups (through shared memory), write this CTA's partial
    __syncthreads();
    double *red = sm;                        // [4][W][W] <= 2 TD_ROWS LD doubles
#pragma unroll
    for (int a = 0; a < F; ++a)
#pragma unroll
        for (int b = 0; b < F; ++b) red[(grp * W + ti + 8 * a) * W + tj + 8 * b] = acc[a][b];
    __syncthreads();
    double *P = partial + (long long)blockIdx.x * M * N;
    for (int idx = t; idx < W * W; idx += TS_NT) {
        const int i = idx / W, j = idx - i * W;
        if (i < M && j < N) P[i * N + j] = (red[idx] + red[W * W + idx]) + (red[2 * W * W + idx] + red[3 * W * W + idx]);
    }
}

// C = alpha * sum_b partial[b] (+ C), through the output maps.  A CTA of 32 x 32 threads owns 32 outputs;
// thread (o, g) adds the partials b = g (mod 32) of output o, then the 32 groups are added in a fixed order.
__global__ void __launch_bounds__(1024) ts_dot_reduce_kernel(const __grid_constant__ GemmParams p, const double *__restrict__ partial,
                                                             int nparts)
{
    __shared__ double red[32][33];
    const int o = threadIdx.x & 31, g = threadIdx.x >> 5;
    const int idx = blockIdx.x * 32 + o, total = p.M * p.N;
    double s = 0.0;
    if (idx < total)
        for (int b = g; b < nparts; b += 32) s += partial[(long long)b * total + idx];
    red[g][o] = s;
    __syncthreads();
    if (g == 0 && idx < total) {
        double v = 0.0;
#pragma unroll
        for (int k = 0; k < 32; ++k) v += red[k][o];
        const int i = idx / p.N, j = idx - i * p.N;
        double *c = p.C + map_off(p.cm, i) + map_off(p.cn, j);
        v *= p.alpha;
        if (p.accumulate) v += *c;
        *c = v;
    }
}

// ---------------------------------------------------------------------------------------
// DMMA versions (the default when the 16-byte alignment conditions hold).  At 4 flop per byte (ts_apply) and
// 8 flop per byte (ts_dot) these passes need 26 - 52 TFLOP/s to run at HBM speed: out of reach of scalar FMAs
// fed from shared memory (the kernels above reach 0.25 - 0.48 of the copy bandwidth), within reach of the FP64
// tensor pipe with the small operand / the accumulators in registers and the rows read straight from global
// memory with 16-byte loads -- no shared-memory staging at all.
__device__ __forceinline__ void ts_dmma(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

// Y[r, n] (+)= alpha sum_c X[r, c] W[c, n], K, N <= 32 (even).  A warp takes 8 rows at a time: lane (lr, lk)
// loads X[row lr][8 g + 2 lk, +1] (the DMMA k order is free: step (g, e) sums k = 8 g + 2 lk + e), W lives in
// registers as B fragments, the D fragments are rows of Y stored with 16-byte stores.
constexpr int TSD_NT = 128;   // threads per CTA of the DMMA streaming kernels (several CTAs per SM)

__global__ void __launch_bounds__(TSD_NT, 4) ts_apply_dmma_kernel(const __grid_constant__ GemmParams p)
{
    // W as B fragments in fragment order: ws[g][j][lane] = (W[8 g + 2 lk][8 j + lr], W[8 g + 2 lk + 1][8 j + lr]):
    // one conflict-free 16-byte load per two DMMAs (64 registers of W per thread would leave one CTA per SM)
    __shared__ double2 ws[4][4][32];
    const int lane = threadIdx.x & 31, lr = lane >> 2, lk = lane & 3;
    const int K = p.K, N = p.N;
    for (int i = threadIdx.x; i < 4 * 4 * 32; i += TSD_NT) {
        const int l = i & 31, j = (i >> 5) & 3, g = i >> 7;
        const int k = 8 * g + 2 * (l & 3), n = 8 * j + (l >> 2);
        double2 v;
        v.x = (k < K && n < N) ? p.B[map_off(p.bk, k) + map_off(p.bn, n)] : 0.0;
        v.y = (k + 1 < K && n < N) ? p.B[map_off(p.bk, k + 1) + map_off(p.bn, n)] : 0.0;
        ws[g][j][l] = v;
    }
    __syncthreads();
    const long long nblk = ((long long)p.M + 7) / 8;
    const long long nwarp = (long long)gridDim.x * (TSD_NT / 32);
    constexpr int U = 2;   // blocks of 8 rows in flight per warp: all loads are issued before the first DMMA
    for (long long blk0 = (long long)blockIdx.x * (TSD_NT / 32) + (threadIdx.x >> 5); blk0 < nblk; blk0 += U * nwarp) {
        double2 a[U][4];
        long long row[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            row[u] = (blk0 + u * nwarp) * 8 + lr;
            const bool valid = row[u] < p.M;
            const double *xr = p.A + (valid ? map_off(p.am, (unsigned)row[u]) : 0);
#pragma unroll
            for (int g = 0; g < 4; ++g)
                a[u][g] = (valid && 8 * g + 2 * lk < K) ? *reinterpret_cast<const double2 *>(xr + 8 * g + 2 * lk) : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            double acc[4][2];
#pragma unroll
            for (int j = 0; j < 4; ++j) acc[j][0] = acc[j][1] = 0.0;
#pragma unroll
            for (int g = 0; g < 4; ++g) {
                double2 wv[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) wv[j] = ws[g][j][lane];
#pragma unroll
                for (int j = 0; j < 4; ++j) ts_dmma(acc[j][0], acc[j][1], a[u][g].x, wv[j].x);
#pragma unroll
                for (int j = 0; j < 4; ++j) ts_dmma(acc[j][0], acc[j][1], a[u][g].y, wv[j].y);
            }
            if (row[u] < p.M) {
                double *yr = p.C + map_off(p.cm, (unsigned)row[u]);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const int n = 8 * j + 2 * lk;
                    if (n < N) {
                        double2 *c = reinterpret_cast<double2 *>(yr + n);
                        double2 v = make_double2(p.alpha * acc[j][0], p.alpha * acc[j][1]);
                        if (p.accumulate) {
                            const double2 o = *c;
                            v.x += o.x;
                            v.y += o.y;
                        }
                        *c = v;
                    }
                }
            }
        }
    }
}

// C[i, j] = sum_r A[r, i] B[r, j], M, N <= 32 (even).  A warp takes 4 rows at a time: lane (lr, lk) loads
// A[row lk][4 lr .. 4 lr + 3] and B likewise; fragment i of the A operand stands for the columns 4 lr + i,
// fragment j of the B operand for the columns 4 lr + j (free choices), so one pair of 16-byte loads feeds 16
// DMMAs.  SYM (A and B are the same matrix: the Gram of a Cholesky-QR pass): the fragment pairs i < j are the
// transposes of the pairs j < i and are left out (10 DMMAs per 4 rows).
template <bool SYM>
__global__ void __launch_bounds__(TSD_NT, 4) ts_dot_dmma_kernel(const __grid_constant__ GemmParams p, double *__restrict__ partial)
{
    __shared__ double red[32][33];
    const int t = threadIdx.x, lane = t & 31, lr = lane >> 2, lk = lane & 3;
    const int M = p.M, N = p.N;
    double acc[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;
    const long long ngrp = ((long long)p.K + 3) / 4;
    const long long nwarp = (long long)gridDim.x * (TSD_NT / 32);
    constexpr int U = SYM ? 4 : 2;   // groups of 4 rows in flight per warp
    for (long long grp0 = (long long)blockIdx.x * (TSD_NT / 32) + (t >> 5); grp0 < ngrp; grp0 += U * nwarp) {
        double2 a0[U], a1[U], b0[U], b1[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const long long row = (grp0 + u * nwarp) * 4 + lk;
            a0[u] = a1[u] = b0[u] = b1[u] = make_double2(0.0, 0.0);
            if (row < p.K) {
                const double *ar = p.A + map_off(p.ak, (unsigned)row) + 4 * lr;
                if (4 * lr < M) a0[u] = *reinterpret_cast<const double2 *>(ar);
                if (4 * lr + 2 < M) a1[u] = *reinterpret_cast<const double2 *>(ar + 2);
                if (!SYM) {
                    const double *br = p.B + map_off(p.bk, (unsigned)row) + 4 * lr;
                    if (4 * lr < N) b0[u] = *reinterpret_cast<const double2 *>(br);
                    if (4 * lr + 2 < N) b1[u] = *reinterpret_cast<const double2 *>(br + 2);
                }
            }
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const double a[4] = {a0[u].x, a0[u].y, a1[u].x, a1[u].y};
            const double b[4] = {SYM ? a0[u].x : b0[u].x, SYM ? a0[u].y : b0[u].y, SYM ? a1[u].x : b1[u].x, SYM ? a1[u].y : b1[u].y};
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (!SYM || i >= j) ts_dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
    }
    // acc[i][j][e] = C[4 lr + i][4 (2 lk + e) + j]; the warps of the CTA are added one after the other
    for (int i = t; i < 32 * 33; i += TSD_NT) (&red[0][0])[i] = 0.0;
    __syncthreads();
    for (int w = 0; w < TSD_NT / 32; ++w) {
        if ((t >> 5) == w) {
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j)
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                        if (SYM && i < j) continue;
                        const int ca = 4 * lr + i, cb = 4 * (2 * lk + e) + j;
                        red[ca][cb] += acc[i][j][e];
                        if (SYM && i > j) red[cb][ca] += acc[i][j][e];
                    }
        }
        __syncthreads();
    }
    double *P = partial + (long long)blockIdx.x * M * N;
    for (int idx = t; idx < M * N; idx += TSD_NT) P[idx] = red[idx / N][idx % N];
}

bool even4(const Map4 &m) { return !(m.s0 & 1) && !(m.s1 & 1) && !(m.s2 & 1) && !(m.s3 & 1); }

bool single_unit(const Map4 &m) { return m.n0 == TATRG_RADIX_INF && m.s0 == 1; }

int g_sms = 0;
int sms()
{
    if (!g_sms) {
        int dev = 0;
        TATRG_CUDA_CHECK(cudaGetDevice(&dev));
        TATRG_CUDA_CHECK(cudaDeviceGetAttribute(&g_sms, cudaDevAttrMultiProcessorCount, dev));
    }
    return g_sms;
}

template <int NH>
void launch_apply(const GemmParams &p)
{
    const size_t tile = (size_t)TS_ROWS * std::max(p.K | 1, (2 * NH) | 1);   // X tile, reused for the results
    const size_t smem = (tile + (size_t)p.K * 2 * NH) * sizeof(double);
    static size_t attr = 0;
    if (smem > attr) {
        TATRG_CUDA_CHECK(cudaFuncSetAttribute(ts_apply_kernel<NH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr = smem;
    }
    const int tiles = (p.M + TS_ROWS - 1) / TS_ROWS;
    const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(8, (200u << 10) / smem));   // resident CTAs by shared memory
    const int grid = tiles < per_sm * sms() ? tiles : per_sm * sms();
    ts_apply_kernel<NH><<<grid, TS_NT, smem, stream()>>>(p);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

template <int F>
void launch_dot(const GemmParams &p)
{
    constexpr size_t smem = (size_t)2 * TD_ROWS * (8 * F + 1) * sizeof(double);
    static_assert(4 * 8 * F * 8 * F <= 2 * TD_ROWS * (8 * F + 1), "reduction scratch fits the tiles");
    static bool attr = false;
    if (!attr) {
        TATRG_CUDA_CHECK(cudaFuncSetAttribute(ts_dot_kernel<F>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr = true;
    }
    const int tiles = (p.K + TD_ROWS - 1) / TD_ROWS;
    const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(8, (200u << 10) / smem));
    const int grid = tiles < per_sm * sms() ? tiles : per_sm * sms();
    size_t mark = ws_mark();
    double *partial = ws_doubles((long long)grid * p.M * p.N);
    ts_dot_kernel<F><<<grid, TS_NT, smem, stream()>>>(p, partial);
    TATRG_LAUNCH_CHECK();
    ts_dot_reduce_kernel<<<(p.M * p.N + 31) / 32, 1024, 0, stream()>>>(p, partial, grid);
    TATRG_LAUNCH_CHECK();
    count_launch(2);
    ws_release(mark);
}

}  // namespace

// true if the launch was taken by one of the streaming kernels
bool tensor_gemm_ts(const GemmParams &p)
{
    if (p.batch != 1 || p.lower_only) return false;
    // rows x K times K x N: A rows contiguous along k, C rows contiguous along n
    // (up to 32 columns: above that the DFMA pipe, not HBM, bounds these kernels and the DMMA tiles win)
    if (p.M >= 16384 && p.K <= 32 && p.N <= 32 && p.K >= 1 && single_unit(p.ak) && single_unit(p.cn)) {
        if (!(p.K & 1) && !(p.N & 1) && !((uintptr_t)p.A & 15) && !((uintptr_t)p.C & 15) && even4(p.am) && even4(p.cm)) {
            const long long nblk = ((long long)p.M + 7) / 8;
            const int grid = (int)std::min<long long>((nblk + 7) / 8, 16LL * sms());
            ts_apply_dmma_kernel<<<grid, TSD_NT, 0, stream()>>>(p);
            TATRG_LAUNCH_CHECK();
            count_launch();
            return true;
        }
        if (p.N <= 32)
            launch_apply<16>(p);
        else
            launch_apply<32>(p);
        return true;
    }
    // (M x rows)(rows x N): both operands contiguous along their small index
    if (p.K >= 16384 && p.M <= 32 && p.N <= 32 && single_unit(p.am) && single_unit(p.bn)) {
        if (!(p.M & 1) && !(p.N & 1) && !((uintptr_t)p.A & 15) && !((uintptr_t)p.B & 15) && even4(p.ak) && even4(p.bk)) {
            const bool sym = p.A == p.B && p.M == p.N && p.ak.n0 == p.bk.n0 && p.ak.n1 == p.bk.n1 && p.ak.n2 == p.bk.n2 &&
                             p.ak.s0 == p.bk.s0 && p.ak.s1 == p.bk.s1 && p.ak.s2 == p.bk.s2 && p.ak.s3 == p.bk.s3;
            const long long ngrp = ((long long)p.K + 3) / 4;
            const int grid = (int)std::min<long long>((ngrp + 63) / 64, 8LL * sms());
            size_t mark = ws_mark();
            double *partial = ws_doubles((long long)grid * p.M * p.N);
            if (sym)
                ts_dot_dmma_kernel<true><<<grid, TSD_NT, 0, stream()>>>(p, partial);
            else
                ts_dot_dmma_kernel<false><<<grid, TSD_NT, 0, stream()>>>(p, partial);
            TATRG_LAUNCH_CHECK();
            ts_dot_reduce_kernel<<<(p.M * p.N + 31) / 32, 1024, 0, stream()>>>(p, partial, grid);
            TATRG_LAUNCH_CHECK();
            count_launch(2);
            ws_release(mark);
            return true;
        }
        const int w = p.M > p.N ? p.M : p.N;
        if (w <= 8)
            launch_dot<1>(p);
        else if (w <= 16)
            launch_dot<2>(p);
        else if (w <= 24)
            launch_dot<3>(p);
        else
            launch_dot<4>(p);
        return true;
    }
    return false;
}

}  // namespace tatrg
