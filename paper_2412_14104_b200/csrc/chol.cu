// chol.cu -- Cholesky factorisation G = L L^T of the symmetric positive (semi)definite Gram
// matrices of the squeezer step (Eq. 12; DESIGN.md "Squeezers without a dense
// eigensolver") and of the tall-skinny Cholesky-QR.  Right-looking blocked algorithm: the
// NB x NB diagonal block is factored and inverted by one CTA in shared memory, the panel and the
// trailing update are tensor-GEMM launches (gemm.cu), so all O(n^3) work runs on the FP64 tensor
// pipe.
#include <algorithm>
#include "ctx.h"
#include "chol64.cuh"

namespace tatrg {

namespace {

constexpr int NB = CH64;      // diagonal block
constexpr int CH_NT = CH64_NT;

// One CTA: A (nb x nb, row-major, leading dimension lda, lower triangle used) -> L in place
// (lower; strict upper part of the block zeroed), Linv (nb x nb row-major, ld ldinv, lower) = L^-1.
// A pivot <= 0 (or NaN) raises *flag.  The factorisation itself: chol64.cuh.
__global__ void __launch_bounds__(CH_NT) chol_block_kernel(double *__restrict__ A, long long lda, int nb,
                                                          double *__restrict__ Linv, int *__restrict__ flag,
                                                          double *__restrict__ dminmax, double shift_rel,
                                                          long long ldinv)
{
    __shared__ Chol64Smem sm;
    const int t = threadIdx.x, ty = t >> 4, tx = t & 15;
    double s[4][4], w[4][4];
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int i = 4 * ty + a, c = 4 * tx + b;
            const int r = i > c ? i : c, cc = i > c ? c : i;   // lower-triangle source
            s[a][b] = (r < nb) ? A[r * lda + cc] : (i == c ? 1.0 : 0.0);
            if (i == c) sm.diag[i] = (i < nb) ? s[a][b] : 0.0;
        }
    __syncthreads();
    chol64_factor(s, w, sm.wk, sm.diag, &sm.bad, nb, shift_rel);
#pragma unroll
    for (int a = 0; a < 4; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            const int i = 4 * ty + a, c = 4 * tx + b;
            if (i < nb && c < nb) {
                A[i * lda + c] = (c <= i) ? s[a][b] : 0.0;
                Linv[i * ldinv + c] = (c <= i) ? w[a][b] : 0.0;
            }
        }
    if (t == 0 && sm.bad) *flag = 1;
    if (t == 0 && dminmax) {
        double lo = sm.diag[0], hi = sm.diag[0];
        for (int j = 1; j < nb; ++j) {
            lo = fmin(lo, sm.diag[j]);
            hi = fmax(hi, sm.diag[j]);
        }
        dminmax[0] = lo;
        dminmax[1] = hi;
    }
}

// ---------------------------------------------------------------------------------------------------------
// The blocked factorisation as ONE resident grid (n > 64).  Launched panel by panel it is 3 dependent launches per
// 64 columns (diagonal block, panel, trailing update): 48 launches and 1.2 - 1.5 ms for n = 1024, nearly all of it
// launch and dependency latency -- and a squeezer chain starts with two of them.  Here G CTAs stay resident and
// meet at two grid-wide barriers per panel:
//   every CTA factors the diagonal block itself (chol64.cuh: identical code on identical bytes; no barrier and no
//   broadcast of L_jj^-1 needed), the warps of all CTAs share out the rows of the panel L21 = A21 L_jj^-T (DMMA,
//   B fragments from L_jj^-1 in shared memory)  -> barrier ->  the CTAs share out the 64 x 64 tiles of the lower
//   triangle of the trailing block, A22[I][K] -= L21[I] L21[K]^T, both operands staged in shared memory -> barrier.
constexpr int CR_LD = 68;

struct CholResSmem {
    union {
        Chol64Work wk;
        struct {
            double LI[NB][CR_LD];
            double LK[NB][CR_LD];
        } t;
    };
    double Ls[NB][CR_LD];   // L_jj^-1
    double diag[NB];
    int bad;
};

__device__ __forceinline__ void cr_dmma(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

__device__ __forceinline__ void cr_grid_barrier(unsigned *bar, unsigned &target)
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

__global__ void __launch_bounds__(CH_NT, 1) chol_resident_kernel(double *__restrict__ A, int n, double *__restrict__ Linv,
                                                                 long long ldinv, long long inv_step,
                                                                 int *__restrict__ flag, unsigned *__restrict__ bar)
{
    extern __shared__ __align__(16) unsigned char cr_smem[];
    CholResSmem &sm = *reinterpret_cast<CholResSmem *>(cr_smem);
    const int t = threadIdx.x, warp = t >> 5, lane = t & 31, g = lane >> 2, q = lane & 3;
    const int ty = t >> 4, tx = t & 15;
    unsigned target = 0;
    for (int j0 = 0; j0 < n; j0 += NB) {
        const int nb = n - j0 < NB ? n - j0 : NB;
        // ---- diagonal block, by every CTA
        double s[4][4], w[4][4];
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const int i = 4 * ty + a, c = 4 * tx + b;
                const int r = i > c ? i : c, cc = i > c ? c : i;   // lower-triangle source
                s[a][b] = (r < nb) ? __ldcg(A + (long long)(j0 + r) * n + j0 + cc) : (i == c ? 1.0 : 0.0);
                if (i == c) sm.diag[i] = (i < nb) ? s[a][b] : 0.0;
            }
        __syncthreads();
        chol64_factor(s, w, sm.wk, sm.diag, &sm.bad, nb, 0.0);
#pragma unroll
        for (int a = 0; a < 4; ++a)
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const int i = 4 * ty + a, c = 4 * tx + b;
                sm.Ls[i][c] = (c <= i) ? w[a][b] : 0.0;
                if (blockIdx.x == 0 && i < nb && c < nb)
                    Linv[(j0 / NB) * inv_step + i * ldinv + c] = (c <= i) ? w[a][b] : 0.0;
            }
        if (blockIdx.x == 0 && t == 0 && sm.bad) *flag = 1;
        __syncthreads();
        const int below = n - j0 - NB;   // rows under the diagonal block
        if (below > 0) {
            // ---- panel: 8-row units shared out over all warps of the grid; in place (a unit's rows are its own)
            const int nu = (below + 7) / 8;
            for (int u = blockIdx.x * (CH_NT / 32) + warp; u < nu; u += gridDim.x * (CH_NT / 32)) {
                const int r = j0 + NB + 8 * u + g;
                double *row = A + (long long)(r < n ? r : 0) * n + j0;
                double af[16];
#pragma unroll
                for (int ks = 0; ks < 16; ++ks) af[ks] = (r < n) ? __ldcg(row + 4 * ks + q) : 0.0;
#pragma unroll
                for (int cb = 0; cb < 8; ++cb) {
                    double d0 = 0.0, d1 = 0.0;
#pragma unroll
                    for (int ks = 0; ks < 16; ++ks) cr_dmma(d0, d1, af[ks], sm.Ls[cb * 8 + g][ks * 4 + q]);
                    if (r < n) {
                        row[cb * 8 + 2 * q] = d0;
                        row[cb * 8 + 2 * q + 1] = d1;
                    }
                }
            }
        }
        cr_grid_barrier(bar, target);   // the panel is complete; nobody reads the old diagonal block any more
        if (blockIdx.x == 0) {
#pragma unroll
            for (int a = 0; a < 4; ++a)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const int i = 4 * ty + a, c = 4 * tx + b;
                    if (i < nb && c < nb) A[(long long)(j0 + i) * n + j0 + c] = (c <= i) ? s[a][b] : 0.0;
                }
        }
        if (below <= 0) break;
        // ---- trailing update: tiles (I, K), K <= I, of the blocks under / right of the panel
        const int nbk = (below + NB - 1) / NB, ntile = nbk * (nbk + 1) / 2;
        for (int tile = blockIdx.x; tile < ntile; tile += gridDim.x) {
            int I = (int)((sqrtf(8.0f * tile + 1.0f) - 1.0f) * 0.5f);
            while (I * (I + 1) / 2 > tile) --I;
            while ((I + 1) * (I + 2) / 2 <= tile) ++I;
            const int K = tile - I * (I + 1) / 2;
            const int ri = j0 + NB + I * NB, rk = j0 + NB + K * NB;
            __syncthreads();   // the previous tile's fragments have been read
            {   // all loads in flight before the first store (thread t: column t & 63 of rows (t >> 6) + 4 i)
                const int cc = t & 63, rr0 = t >> 6;
                double vi[16], vk[16];
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const int rr = rr0 + 4 * i;
                    vi[i] = (ri + rr < n) ? __ldcg(A + (long long)(ri + rr) * n + j0 + cc) : 0.0;
                    vk[i] = (K != I && rk + rr < n) ? __ldcg(A + (long long)(rk + rr) * n + j0 + cc) : 0.0;
                }
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    sm.t.LI[rr0 + 4 * i][cc] = vi[i];
                    sm.t.LK[rr0 + 4 * i][cc] = vk[i];
                }
            }
            __syncthreads();
            const double(*LK)[CR_LD] = (K != I) ? sm.t.LK : sm.t.LI;
            double acc[8][2];
#pragma unroll
            for (int cb = 0; cb < 8; ++cb) acc[cb][0] = acc[cb][1] = 0.0;
#pragma unroll
            for (int ks = 0; ks < 16; ++ks) {
                const double a = sm.t.LI[warp * 8 + g][ks * 4 + q];
#pragma unroll
                for (int cb = 0; cb < 8; ++cb) cr_dmma(acc[cb][0], acc[cb][1], a, LK[cb * 8 + g][ks * 4 + q]);
            }
            const int r = ri + warp * 8 + g;
            if (r < n) {
                double *row = A + (long long)r * n + rk;
                double old[8][2];
#pragma unroll
                for (int cb = 0; cb < 8; ++cb) {
                    const int c = cb * 8 + 2 * q;
                    old[cb][0] = (rk + c < n) ? __ldcg(row + c) : 0.0;
                    old[cb][1] = (rk + c + 1 < n) ? __ldcg(row + c + 1) : 0.0;
                }
#pragma unroll
                for (int cb = 0; cb < 8; ++cb) {
                    const int c = cb * 8 + 2 * q;
                    if (rk + c < n) row[c] = old[cb][0] - acc[cb][0];
                    if (rk + c + 1 < n) row[c + 1] = old[cb][1] - acc[cb][1];
                }
            }
        }
        cr_grid_barrier(bar, target);
    }
    // ---- strict upper triangle of the result: zero
    const long long total = (long long)n * n;
    for (long long i = (long long)blockIdx.x * CH_NT + t; i < total; i += (long long)gridDim.x * CH_NT) {
        const int r = (int)(i / n), c = (int)(i - (long long)r * n);
        if (c > r && (c / NB) > (r / NB)) A[i] = 0.0;   // (inside the diagonal blocks CTA 0 has written the zeros)
    }
}

// x[i][i] += shift_rel * max_diag ; one CTA
__global__ void add_shift_kernel(double *__restrict__ A, int n, double shift_rel)
{
    __shared__ double red[32];
    double m = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) m = fmax(m, A[(long long)i * n + i]);
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
    __syncthreads();
    m = 0.0;
    for (int i = 0; i < (int)(blockDim.x >> 5); ++i) m = fmax(m, red[i]);
    const double d = shift_rel * m;
    for (int i = threadIdx.x; i < n; i += blockDim.x) A[(long long)i * n + i] += d;
}

__global__ void zero_upper_kernel(double *__restrict__ A, int n)
{
    long long total = (long long)n * n;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x) {
        int r = (int)(i / n), c = (int)(i - (long long)r * n);
        if (c > r) A[i] = 0.0;
    }
}

// G = I + E with |E| tiny: L = I + strict_lower(E) + diag(E)/2 and L^-1 = 2I - L, both to O(|E|^2)
__global__ void near_identity_chol_kernel(double *__restrict__ G, double *__restrict__ Linv, int n)
{
    long long total = (long long)n * n;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x) {
        int r = (int)(i / n), c = (int)(i - (long long)r * n);
        double e = G[i] - (r == c ? 1.0 : 0.0);
        double l = (c < r) ? e : (c == r ? 0.5 * e : 0.0);
        G[i] = (r == c ? 1.0 : 0.0) + l;
        Linv[i] = (r == c ? 1.0 : 0.0) - l;
    }
}

Ten view2(double *p, char a, long long na, long long sa, char b, long long nb_, long long sb)
{
    Ten t;
    t.p = p;
    t.legs = {Leg{a, na, sa}, Leg{b, nb_, sb}};
    return t;
}

constexpr size_t CHOL_SMEM = 0;

void chol_attr()
{
    static bool attr_done = false;
    if (!attr_done) {
        TATRG_CUDA_CHECK(cudaFuncSetAttribute(chol_block_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CHOL_SMEM));
        attr_done = true;
    }
}

}  // namespace

// Asynchronous: the n x n (n <= 64) block A (row-major, leading dimension lda) -> its lower Cholesky
// factor in place, Linv (row-major, leading dimension 64) = L^-1, *flag raised on a non-positive
// pivot, dminmax[0..1] = smallest / largest diagonal entry of L (a cheap condition estimate);
// shift_rel > 0 adds shift_rel * max_i A_ii to the diagonal first.
void chol_block(double *A, long long lda, int n, double *Linv, int *flag, double *dminmax, double shift_rel)
{
    if (n > NB) fail(-22, "chol_block: n = %d > %d", n, NB);
    chol_attr();
    chol_block_kernel<<<1, CH_NT, CHOL_SMEM, stream()>>>(A, lda, n, Linv, flag, dminmax, shift_rel, NB);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

// In place: the n x n symmetric matrix A (row-major, lower triangle read) becomes its lower
// Cholesky factor (upper triangle zeroed) after adding shift_rel * max_i A_ii to the diagonal.
// Linv_full (optional, n x n row-major) receives L^-1.
// Returns false when a pivot was not positive (A then holds garbage).
void cholesky_lower_async(double *A, int n, double shift_rel, double *Linv_full, int *flag)
{
    size_t mark = ws_mark();
    double *Linv = ws_doubles(NB * NB);
    if (shift_rel > 0.0) {
        add_shift_kernel<<<1, 256, 0, stream()>>>(A, n, shift_rel);
        count_launch();
    }
    if (Linv_full) fill_zero(Linv_full, (long long)n * n);
    chol_attr();
    const int want_ctas = ctx().chol_ctas;
    if (n > NB && want_ctas > 0) {
        // one resident grid (chol_resident_kernel); the inverted diagonal blocks go to Linv_full's diagonal blocks or
        // (not wanted) to one scratch block
        static bool res_attr = false;
        if (!res_attr) {
            TATRG_CUDA_CHECK(cudaFuncSetAttribute(chol_resident_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(CholResSmem)));
            res_attr = true;
        }
        unsigned *bar = reinterpret_cast<unsigned *>(ws_alloc(sizeof(unsigned)));
        TATRG_CUDA_CHECK(cudaMemsetAsync(bar, 0, sizeof(unsigned), stream()));
        const int grid = std::max(1, std::min(want_ctas, (n + NB - 1) / NB * 2));
        chol_resident_kernel<<<grid, CH_NT, sizeof(CholResSmem), stream()>>>(A, n, Linv_full ? Linv_full : Linv, Linv_full ? n : NB,
                                                                         Linv_full ? (long long)NB * n + NB : 0, flag, bar);
        TATRG_LAUNCH_CHECK();
        count_launch();
        count_flops((double)n * n * n / 3.0);
    } else {
    for (int j0 = 0; j0 < n; j0 += NB) {
        const int nb = n - j0 < NB ? n - j0 : NB;
        double *Ajj = A + (long long)j0 * n + j0;
        double *Lij = Linv_full ? Linv_full + (long long)j0 * n + j0 : Linv;   // inverse of the diagonal block
        const long long ldi = Linv_full ? n : NB;
        chol_block_kernel<<<1, CH_NT, CHOL_SMEM, stream()>>>(Ajj, n, nb, Lij, flag, nullptr, 0.0, ldi);
        TATRG_LAUNCH_CHECK();
        count_launch();
        const int rest = n - j0 - nb;
        if (rest <= 0) break;
        double *A21 = A + (long long)(j0 + nb) * n + j0;
        double *A22 = A + (long long)(j0 + nb) * n + j0 + nb;
        // L21 = A21 Linv^T, in place: the output is one column tile wide and K = nb is never split, so
        // every CTA reads exactly the rows it later writes
        contract(view2(A21, 'i', rest, n, 'k', nb, 1), view2(Lij, 'j', nb, ldi, 'k', nb, 1),
                 view2(A21, 'i', rest, n, 'j', nb, 1));
        // A22 -= L21 L21^T
        contract(view2(A21, 'i', rest, n, 'k', nb, 1), view2(A21, 'j', rest, n, 'k', nb, 1),
                 view2(A22, 'i', rest, n, 'j', rest, 1), -1.0, true, true);
    }
    int blocks = (int)(((long long)n * n + 255) / 256 < 1184 ? ((long long)n * n + 255) / 256 : 1184);
    zero_upper_kernel<<<blocks, 256, 0, stream()>>>(A, n);
    TATRG_LAUNCH_CHECK();
    count_launch();
    }
    if (Linv_full) {
        // L^-1 from the inverted diagonal blocks, doubling the block size:
        // inv([L11 0; L21 L22]) = [inv11 0; -inv22 L21 inv11, inv22]; equal pairs of one level are one batched GEMM
        double *tt = ws_doubles((long long)n * n / 2 + NB * NB);
        for (long long sz = NB; sz < n; sz *= 2) {
            const long long full = n / (2 * sz);                       // pairs with two complete halves
            auto pair = [&](long long j0, long long s2, long long nbat) {
                const long long bs = 2 * sz * ((long long)n + 1);      // batch stride along the diagonal
                auto v3 = [&](double *p, char a, long long na, long long sa, char b, long long nb_, long long sb) {
                    Ten t;
                    t.p = p;
                    t.legs = {Leg{'B', nbat, bs}, Leg{a, na, sa}, Leg{b, nb_, sb}};
                    return t;
                };
                const double *L21 = A + (j0 + sz) * n + j0;
                double *I11 = Linv_full + j0 * n + j0, *I22 = Linv_full + (j0 + sz) * n + j0 + sz;
                double *I21 = Linv_full + (j0 + sz) * n + j0;
                Ten T;
                T.p = tt;
                T.legs = {Leg{'B', nbat, s2 * sz}, Leg{'i', s2, sz}, Leg{'j', sz, 1}};
                contract(v3(const_cast<double *>(L21), 'i', s2, n, 'k', sz, 1), v3(I11, 'k', sz, n, 'j', sz, 1), T);
                contract(v3(I22, 'l', s2, n, 'i', s2, 1), T, v3(I21, 'l', s2, n, 'j', sz, 1), -1.0, false);
            };
            if (full > 0) pair(0, sz, full);
            const long long j0 = full * 2 * sz;
            if (n - j0 > sz) pair(j0, n - j0 - sz, 1);                 // ragged last pair
        }
    }
    ws_release(mark);
}

bool cholesky_lower(double *A, int n, double shift_rel, double *Linv_full)
{
    size_t mark = ws_mark();
    int *flag = (int *)ws_alloc(sizeof(int));
    TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(int), stream()));
    cholesky_lower_async(A, n, shift_rel, Linv_full, flag);
    int h = 0;
    TATRG_CUDA_CHECK(cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
    TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
    ws_release(mark);
    return h == 0;
}

// out[0], out[1] = min, max of the diagonal of the n x n row-major matrix L (one CTA)
__global__ void diag_minmax_kernel(const double *__restrict__ L, int n, double *__restrict__ out)
{
    __shared__ double lo_s[32], hi_s[32];
    double lo = INFINITY, hi = -INFINITY;
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
        const double d = L[(long long)i * n + i];
        lo = fmin(lo, d);
        hi = fmax(hi, d);
    }
    for (int o = 16; o > 0; o >>= 1) {
        lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
    }
    if ((threadIdx.x & 31) == 0) {
        lo_s[threadIdx.x >> 5] = lo;
        hi_s[threadIdx.x >> 5] = hi;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < (int)(blockDim.x >> 5); ++i) {
            lo = fmin(lo, lo_s[i]);
            hi = fmax(hi, hi_s[i]);
        }
        out[0] = lo;
        out[1] = hi;
    }
}

void diag_minmax(const double *L, int n, double *out)
{
    diag_minmax_kernel<<<1, 256, 0, stream()>>>(L, n, out);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

void near_identity_chol(double *G, int n, double *Linv)
{
    int blocks = (int)(((long long)n * n + 255) / 256 < 1184 ? ((long long)n * n + 255) / 256 : 1184);
    near_identity_chol_kernel<<<blocks, 256, 0, stream()>>>(G, Linv, n);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

}  // namespace tatrg
