// cholqr_fused.cu -- Cholesky-QR of a tall block with at most 64 columns as ONE launch ("iterations
// of the QR decomposition": the orthonormalisation inside the subspace iterations of the bond swap, and
// of the isometries, Eqs. 2-3; DESIGN.md section 2 item 1).
//
// As separate launches one pass is {Gram by a split-K GEMM, reduction of the partial sums, 64 x 64 Cholesky,
// Y <- Y L^-T}: four to five dependent launches, 125 - 190 us for a 32768 x 64 block whose bytes pass through HBM
// in 5 us.  Here a resident grid does `passes` rounds with two grid barriers each (the scheme of sq_iter.cu):
//   every CTA owns the 64-row chunks c = blockIdx.x, blockIdx.x + gridDim.x, ... of Y (always the same ones, so no
//   chunk is ever read by another CTA); partial Gram of its chunks by DMMA from shared memory -> barrier -> every
//   CTA sums its share of the 64 x 64 entries over the partial Grams in a fixed order (deterministic) -> barrier ->
//   EVERY CTA factors the same Gram (chol64.cuh) and applies L^-T to its chunks, accumulating the partial Gram of
//   the RESULT on the way, so the second pass needs no extra sweep over Y.  A CTA with a single chunk keeps it in
//   shared memory from the first load to the last store.
#include <algorithm>
#include <stdint.h>
#include "ctx.h"
#include "chol64.cuh"

namespace tatrg {

namespace {

constexpr int CQ_B = 64;         // padded column count
constexpr int CQ_NT = CH64_NT;   // 8 warps
constexpr int CQ_LD = 68;        // row stride of the shared-memory tiles
constexpr int CQ_ROWS = 64;      // rows per chunk

struct CqParams {
    double *Y;          // m x n row-major (ld = n), in place
    long long m;
    int n, passes;      // n <= 64, passes 1 or 2
    double shift;       // relative diagonal shift of the first pass
    int *flag;          // raised (sticky) by a non-positive pivot
    double *ratio;      // optional: min / max of diag(L) of the first pass
    double *Rout;       // optional: n x n row-major, R = L_p^T ... L_1^T
    double *part, *gram, *Lkeep;
    unsigned *bar;
};

struct CqSmem {
    double Ys[CQ_ROWS][CQ_LD];   // the chunk in flight
    union {
        Chol64Work wk;           // scratch of the factorisation, then ...
        double Ls[CQ_B][CQ_LD];  // ... L^-1 of the current pass
    };
    double diag[CH64];
    int bad;
};

__device__ __forceinline__ void cq_dmma(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

// all CTAs of the grid; `target` counts the arrivals expected so far
__device__ __forceinline__ void cq_grid_barrier(unsigned *bar, unsigned &target)
{
    target += gridDim.x;
    __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;\n" ::"l"(bar) : "memory");
        unsigned v;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(bar) : "memory");
        } while (v < target);
    }
    __syncthreads();
}

__global__ void __launch_bounds__(CQ_NT, 2) cholqr64_kernel(const __grid_constant__ CqParams p)
{
    extern __shared__ __align__(16) unsigned char cq_raw[];
    CqSmem &sm = *reinterpret_cast<CqSmem *>(cq_raw);
    const int t = threadIdx.x, warp = t >> 5, lane = t & 31, g = lane >> 2, q = lane & 3;
    const int n = p.n;
    const long long m = p.m, nchunks = (m + CQ_ROWS - 1) / CQ_ROWS;
    const bool vec = n == CQ_B && (reinterpret_cast<uintptr_t>(p.Y) & 15) == 0;
    unsigned target = 0;
    long long resident = -1;   // chunk held by Ys (uniform over the CTA)

    auto load_chunk = [&](long long c) {
        if (resident == c) return;
        __syncthreads();       // everybody is done with the previous contents
        const long long r0 = c * CQ_ROWS;
        if (vec) {
#pragma unroll
            for (int i = 0; i < CQ_ROWS * CQ_B / 2 / CQ_NT; ++i) {
                const int idx = t + i * CQ_NT, row = idx >> 5, c2 = (idx & 31) * 2;
                double2 v = make_double2(0.0, 0.0);
                if (r0 + row < m) v = __ldcg(reinterpret_cast<const double2 *>(p.Y + (r0 + row) * CQ_B + c2));
                *reinterpret_cast<double2 *>(&sm.Ys[row][c2]) = v;
            }
        } else {
            for (int idx = t; idx < CQ_ROWS * CQ_B; idx += CQ_NT) {
                const int row = idx >> 6, col = idx & 63;
                sm.Ys[row][col] = (r0 + row < m && col < n) ? __ldcg(p.Y + (r0 + row) * n + col) : 0.0;
            }
        }
        __syncthreads();
        resident = c;
    };
    // partial Gram of the chunk in Ys: warp w -> Gram rows 8 w .. 8 w + 7, all 64 columns
    double gacc[8][2];
    auto gram_zero = [&]() {
#pragma unroll
        for (int cb = 0; cb < 8; ++cb) gacc[cb][0] = gacc[cb][1] = 0.0;
    };
    auto gram_add = [&]() {
#pragma unroll 4
        for (int k0 = 0; k0 < CQ_ROWS; k0 += 4) {
            const double a = sm.Ys[k0 + q][warp * 8 + g];
#pragma unroll
            for (int cb = 0; cb < 8; ++cb) cq_dmma(gacc[cb][0], gacc[cb][1], a, sm.Ys[k0 + q][cb * 8 + g]);
        }
    };

    gram_zero();
    for (long long c = blockIdx.x; c < nchunks; c += gridDim.x) {
        load_chunk(c);
        gram_add();
    }

    for (int pass = 0; pass < p.passes; ++pass) {
        {
            double *pp = p.part + (long long)blockIdx.x * (CQ_B * CQ_B) + (warp * 8 + g) * CQ_B + 2 * q;
#pragma unroll
            for (int cb = 0; cb < 8; ++cb) *reinterpret_cast<double2 *>(pp + cb * 8) = make_double2(gacc[cb][0], gacc[cb][1]);
        }
        cq_grid_barrier(p.bar, target);
        // this CTA's share of the Gram entries, summed over the partial Grams in a fixed order
        for (int e = blockIdx.x * CQ_NT + t; e < CQ_B * CQ_B; e += gridDim.x * CQ_NT) {
            const double *pe = p.part + e;
            const int G = (int)gridDim.x;
            double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
            int c = 0;
            for (; c + 4 <= G; c += 4) {
                s0 += __ldcg(pe + (long long)c * (CQ_B * CQ_B));
                s1 += __ldcg(pe + (long long)(c + 1) * (CQ_B * CQ_B));
                s2 += __ldcg(pe + (long long)(c + 2) * (CQ_B * CQ_B));
                s3 += __ldcg(pe + (long long)(c + 3) * (CQ_B * CQ_B));
            }
            for (; c < G; ++c) s0 += __ldcg(pe + (long long)c * (CQ_B * CQ_B));
            p.gram[e] = (s0 + s1) + (s2 + s3);
        }
        cq_grid_barrier(p.bar, target);
        // every CTA: G (+ shift) = L L^T, L^-1 (columns n .. 63 padded with the identity)
        {
            const int ty = t >> 4, tx = t & 15;
            double s[4][4], w[4][4];
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const int i = 4 * ty + a, c = 4 * tx + b;
                    const int r = i > c ? i : c, cc = i > c ? c : i;   // lower-triangle source
                    s[a][b] = (r < n) ? __ldcg(p.gram + r * CQ_B + cc) : (i == c ? 1.0 : 0.0);
                    if (i == c) sm.diag[i] = (i < n) ? s[a][b] : 0.0;
                }
            __syncthreads();
            chol64_factor(s, w, sm.wk, sm.diag, &sm.bad, n, pass == 0 ? p.shift : 0.0);
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const int i = 4 * ty + a, c = 4 * tx + b;
                    sm.Ls[i][c] = (c <= i) ? w[a][b] : 0.0;   // (the factorisation's scratch is dead: it ended with a barrier)
                    if (blockIdx.x == 0) p.Lkeep[pass * (CQ_B * CQ_B) + i * CQ_B + c] = (c <= i) ? s[a][b] : 0.0;
                }
            if (blockIdx.x == 0 && t == 0) {
                if (sm.bad) *p.flag = 1;
                if (pass == 0 && p.ratio) {
                    double lo = sm.diag[0], hi = sm.diag[0];
                    for (int j = 1; j < n; ++j) {
                        lo = fmin(lo, sm.diag[j]);
                        hi = fmax(hi, sm.diag[j]);
                    }
                    p.ratio[0] = lo;
                    p.ratio[1] = hi;
                }
            }
            __syncthreads();
        }
        // Y <- Y L^-T on the CTA's chunks: out[r, d] = sum_c Y[r, c] Linv[d, c]; warp w -> columns d = 8 w .. 8 w + 7
        {
            double bf[16];
#pragma unroll
            for (int ks = 0; ks < 16; ++ks) bf[ks] = sm.Ls[warp * 8 + g][ks * 4 + q];
            const bool more = pass + 1 < p.passes;
            gram_zero();
            for (long long c = blockIdx.x; c < nchunks; c += gridDim.x) {
                load_chunk(c);
                double o[8][2];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    o[u][0] = o[u][1] = 0.0;
#pragma unroll
                    for (int ks = 0; ks < 16; ++ks) cq_dmma(o[u][0], o[u][1], sm.Ys[u * 8 + g][ks * 4 + q], bf[ks]);
                }
                __syncthreads();   // every warp has read the old rows
                const long long r0 = c * CQ_ROWS;
                const int col = warp * 8 + 2 * q;
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int row = u * 8 + g;
                    *reinterpret_cast<double2 *>(&sm.Ys[row][col]) = make_double2(o[u][0], o[u][1]);
                    if (r0 + row < m) {
                        if (vec) {
                            *reinterpret_cast<double2 *>(p.Y + (r0 + row) * CQ_B + col) = make_double2(o[u][0], o[u][1]);
                        } else {
                            if (col < n) p.Y[(r0 + row) * n + col] = o[u][0];
                            if (col + 1 < n) p.Y[(r0 + row) * n + col + 1] = o[u][1];
                        }
                    }
                }
                __syncthreads();
                if (more) gram_add();   // (rows >= m and columns >= n of the result are exact zeros)
            }
        }
    }
    // R = L2^T L1^T of two passes (R[i][j] = sum_k L2[k][i] L1[j][k]); one pass: R = L1^T.  The factors are staged in
    // shared memory first (from global memory this short loop of dependent loads took 100 us)
    if (blockIdx.x == 0 && p.Rout) {
        __syncthreads();
        for (int e = t; e < CQ_B * CQ_B; e += CQ_NT) {
            sm.Ys[e >> 6][e & 63] = __ldcg(p.Lkeep + e);
            sm.Ls[e >> 6][e & 63] = p.passes == 2 ? __ldcg(p.Lkeep + CQ_B * CQ_B + e) : 0.0;
        }
        __syncthreads();
        for (int e = t; e < n * n; e += CQ_NT) {
            const int i = e / n, j = e - i * n;
            double sum = 0.0;
            if (p.passes == 2) {
#pragma unroll 4
                for (int k = i; k < n; ++k) sum = fma(sm.Ls[k][i], sm.Ys[j][k], sum);
            } else {
                sum = sm.Ys[j][i];
            }
            p.Rout[e] = sum;
        }
    }
}

}  // namespace

// false: not taken (the caller runs the pass as separate launches)
bool cholqr_fused(double *Y, long long m, int n, int passes, double shift_rel, int *flag_dev, double *ratio_dev,
                  double *Rout)
{
    Ctx &c = ctx();
    if (c.routes & ROUTE_UNFUSED_SQUEEZER) return false;
    if (n < 1 || n > CQ_B || passes < 1 || passes > 2 || m < CQ_ROWS) return false;
    if (n <= 32 && m >= 16384) return false;   // HBM-sized blocks of <= 32 columns: the streaming kernels of ts.cu (no padding)
    if (m >= (1LL << 20)) return false;        // HBM-sized blocks of 33..64 columns (canonical form at chi > 32): compute-bound, the GEMM tiles
                                               // on every SM are 1.2-1.6x faster than this grid of <= 128 CTAs (chi = 36..64: 4.1 -> 2.7 ... 32.2 -> 26.2 ms)
    const long long nchunks = (m + CQ_ROWS - 1) / CQ_ROWS;
    const int cap = c.sm_reserve > 0 ? c.sm_reserve : 128;   // resident: every CTA must find an SM
    const int grid = (int)std::min<long long>(nchunks, cap);
    static bool attr_done = false;
    if (!attr_done) {
        TATRG_CUDA_CHECK(cudaFuncSetAttribute(cholqr64_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(CqSmem)));
        attr_done = true;
    }
    size_t mark = ws_mark();
    CqParams p{};
    p.Y = Y;
    p.m = m;
    p.n = n;
    p.passes = passes;
    p.shift = shift_rel;
    p.flag = flag_dev;
    p.ratio = ratio_dev;
    p.Rout = Rout;
    p.part = ws_doubles((long long)(grid + 3) * CQ_B * CQ_B + 2);
    p.gram = p.part + (size_t)grid * CQ_B * CQ_B;
    p.Lkeep = p.gram + CQ_B * CQ_B;
    p.bar = reinterpret_cast<unsigned *>(p.Lkeep + 2 * CQ_B * CQ_B);
    TATRG_CUDA_CHECK(cudaMemsetAsync(p.bar, 0, sizeof(unsigned), stream()));
    cholqr64_kernel<<<grid, CQ_NT, sizeof(CqSmem), stream()>>>(p);
    TATRG_LAUNCH_CHECK();
    count_launch();
    count_flops(passes * 4.0 * (double)m * n * n);
    ws_release(mark);
    return true;
}

}  // namespace tatrg
