// chol.cu -- Cholesky factorisation G = L L^T of the symmetric positive (semi)definite Gram
// matrices of the squeezer step (Eq. 12; DESIGN.md "Squeezers without a dense
// eigensolver") and of the tall-skinny Cholesky-QR.  Right-looking blocked algorithm: the
// NB x NB diagonal block is factored and inverted by one CTA in shared memory, the panel and the
// trailing update are tensor-GEMM launches (gemm.cu), so all O(n^3) work runs on the FP64 tensor
// pipe.
#include "ctx.h"

namespace tatrg {

namespace {

constexpr int NB = 64;       // diagonal block
constexpr int CH_NT = 256;

// One CTA: A (nb x nb, row-major, leading dimension lda, lower triangle used) -> L in place
// (lower; strict upper part of the block zeroed), Linv (nb x nb row-major, ld NB, lower) = L^-1.
// A pivot <= 0 (or NaN) raises *flag.
__global__ void __launch_bounds__(CH_NT) chol_block_kernel(double *__restrict__ A, long long lda, int nb,
                                                          double *__restrict__ Linv, int *__restrict__ flag,
                                                          double *__restrict__ dminmax)
{
    extern __shared__ double chol_sm[];
    double (*S)[NB + 1] = reinterpret_cast<double (*)[NB + 1]>(chol_sm);
    double (*W)[NB + 1] = reinterpret_cast<double (*)[NB + 1]>(chol_sm + NB * (NB + 1));
    __shared__ int bad;
    const int t = threadIdx.x;
    if (t == 0) bad = 0;
    for (int i = t; i < nb * nb; i += CH_NT) {
        int r = i / nb, c = i - r * nb;
        S[r][c] = (c <= r) ? A[r * lda + c] : 0.0;
    }
    __syncthreads();
    for (int j = 0; j < nb; ++j) {
        // column j: S[j][j] = sqrt(pivot), S[i][j] /= S[j][j]
        double piv = S[j][j];
        __syncthreads();
        if (!(piv > 0.0)) {
            if (t == 0) bad = 1;
            piv = 1.0;
        }
        const double d = sqrt(piv);
        if (t == 0) S[j][j] = d;
        for (int i = j + 1 + t; i < nb; i += CH_NT) S[i][j] /= d;
        __syncthreads();
        // trailing update of the lower triangle: S[i][c] -= S[i][j] S[c][j], j < c <= i
        const int rem = nb - j - 1;
        for (int e = t; e < rem * rem; e += CH_NT) {
            int i = j + 1 + e / rem, c = j + 1 + e % rem;
            if (c <= i) S[i][c] = fma(-S[i][j], S[c][j], S[i][c]);
        }
        __syncthreads();
    }
    // inverse of the lower-triangular L: column c of W solved by forward substitution, one
    // thread per column (nb <= 64 columns; tiny)
    if (t < nb) {
        const int c = t;
        for (int i = 0; i < nb; ++i) {
            double s = (i == c) ? 1.0 : 0.0;
            for (int k = c; k < i; ++k) s = fma(-S[i][k], W[k][c], s);
            W[i][c] = (i >= c) ? s / S[i][i] : 0.0;
        }
    }
    __syncthreads();
    for (int i = t; i < nb * nb; i += CH_NT) {
        int r = i / nb, c = i - r * nb;
        A[r * lda + c] = S[r][c];
        Linv[r * NB + c] = W[r][c];
    }
    if (t == 0 && bad) *flag = 1;
    if (t == 0 && dminmax) {
        double lo = S[0][0], hi = S[0][0];
        for (int j = 1; j < nb; ++j) {
            lo = fmin(lo, S[j][j]);
            hi = fmax(hi, S[j][j]);
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

Ten view2(double *p, char a, long long na, long long sa, char b, long long nb_, long long sb)
{
    Ten t;
    t.p = p;
    t.legs = {Leg{a, na, sa}, Leg{b, nb_, sb}};
    return t;
}

constexpr size_t CHOL_SMEM = 2 * NB * (NB + 1) * sizeof(double);

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
// pivot, dminmax[0..1] = smallest / largest diagonal entry of L (a cheap condition estimate).
void chol_block(double *A, long long lda, int n, double *Linv, int *flag, double *dminmax)
{
    if (n > NB) fail(-22, "chol_block: n = %d > %d", n, NB);
    chol_attr();
    chol_block_kernel<<<1, CH_NT, CHOL_SMEM, stream()>>>(A, lda, n, Linv, flag, dminmax);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

// In place: the n x n symmetric matrix A (row-major, lower triangle read) becomes its lower
// Cholesky factor (upper triangle zeroed) after adding shift_rel * max_i A_ii to the diagonal.
// Returns false when a pivot was not positive (A then holds garbage).
bool cholesky_lower(double *A, int n, double shift_rel)
{
    size_t mark = ws_mark();
    int *flag = (int *)ws_alloc(sizeof(int));
    TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(int), stream()));
    double *Linv = ws_doubles(NB * NB);
    if (shift_rel > 0.0) {
        add_shift_kernel<<<1, 256, 0, stream()>>>(A, n, shift_rel);
        count_launch();
    }
    double *tmp = ws_doubles((long long)n * NB);
    chol_attr();
    for (int j0 = 0; j0 < n; j0 += NB) {
        const int nb = n - j0 < NB ? n - j0 : NB;
        double *Ajj = A + (long long)j0 * n + j0;
        chol_block_kernel<<<1, CH_NT, CHOL_SMEM, stream()>>>(Ajj, n, nb, Linv, flag, nullptr);
        TATRG_LAUNCH_CHECK();
        count_launch();
        const int rest = n - j0 - nb;
        if (rest <= 0) break;
        double *A21 = A + (long long)(j0 + nb) * n + j0;
        double *A22 = A + (long long)(j0 + nb) * n + j0 + nb;
        // L21 = A21 Linv^T
        Ten T = view2(tmp, 'i', rest, nb, 'j', nb, 1);
        contract(view2(A21, 'i', rest, n, 'k', nb, 1), view2(Linv, 'j', nb, NB, 'k', nb, 1), T);
        // A22 -= L21 L21^T ; then store L21
        contract(T.as("ik"), T.as("jk"), view2(A22, 'i', rest, n, 'j', rest, 1), -1.0, true);
        TATRG_CUDA_CHECK(cudaMemcpy2DAsync(A21, sizeof(double) * n, tmp, sizeof(double) * nb, sizeof(double) * nb,
                                           rest, cudaMemcpyDeviceToDevice, stream()));
    }
    int blocks = (int)(((long long)n * n + 255) / 256 < 1184 ? ((long long)n * n + 255) / 256 : 1184);
    zero_upper_kernel<<<blocks, 256, 0, stream()>>>(A, n);
    TATRG_LAUNCH_CHECK();
    count_launch();
    int h = 0;
    TATRG_CUDA_CHECK(cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
    TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
    ws_release(mark);
    return h == 0;
}

}  // namespace tatrg
