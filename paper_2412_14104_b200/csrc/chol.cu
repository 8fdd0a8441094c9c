// chol.cu -- Cholesky factorisation G = L L^T of the symmetric positive (semi)definite Gram
// matrices of the squeezer step (Eq. 12; DESIGN.md "Squeezers without a dense
// eigensolver") and of the tall-skinny Cholesky-QR.  Right-looking blocked algorithm: the
// NB x NB diagonal block is factored and inverted by one CTA in shared memory, the panel and the
// trailing update are tensor-GEMM launches (gemm.cu), so all O(n^3) work runs on the FP64 tensor
// pipe.
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
