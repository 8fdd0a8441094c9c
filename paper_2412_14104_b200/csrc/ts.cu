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
        if (p.N <= 32)
            launch_apply<16>(p);
        else
            launch_apply<32>(p);
        return true;
    }
    // (M x rows)(rows x N): both operands contiguous along their small index
    if (p.K >= 16384 && p.M <= 32 && p.N <= 32 && single_unit(p.am) && single_unit(p.bn)) {
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
