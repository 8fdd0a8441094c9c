// jacobi.cu -- one-sided (Hestenes) Jacobi SVD, batched, for every dense SVD / symmetric
// eigenproblem of the path: the small core of the RSVD (reading O9), the
// canonical-form SVD, the Ritz step of the isometries (Eq. 3) and the
// eigendecompositions / SVD of the squeezers (Eq. 12, reading O6).
//
// G (column-major m x n) is rotated from the right until its columns are mutually orthogonal:
// G_in V = U diag(s).  A symmetric PSD matrix S is handled by the same routine: S V = V diag(lambda).
// Parallel round-robin ordering: n/2 disjoint column pairs per round, one CTA per pair; the
// matrices stay L2-resident.  Columns are finally sorted by decreasing norm.
#include "common.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

namespace tatrg {

namespace {

constexpr int JT = 128;

__device__ __forceinline__ void block_sum3(double &a, double &b, double &c)
{
    __shared__ double sh[3][JT / 32];
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
        c += __shfl_xor_sync(0xffffffffu, c, o);
    }
    int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) {
        sh[0][w] = a;
        sh[1][w] = b;
        sh[2][w] = c;
    }
    __syncthreads();
    a = b = c = 0.0;
#pragma unroll
    for (int i = 0; i < JT / 32; ++i) {
        a += sh[0][i];
        b += sh[1][i];
        c += sh[2][i];
    }
}

__global__ void __launch_bounds__(JT) jacobi_round_kernel(double *__restrict__ G, int m, int n,
                                                         double *__restrict__ V, int round, int npad,
                                                         long long strideG, long long strideV, double tol,
                                                         const double *__restrict__ fro2,
                                                         unsigned long long *__restrict__ maxcos)
{
    const int pi = blockIdx.x;
    const int nm1 = npad - 1;
    int p, q;
    if (pi == 0) {
        p = nm1;
        q = round;
    } else {
        p = (round + pi) % nm1;
        q = (round - pi + nm1) % nm1;
    }
    if (p > q) {
        int tmp = p;
        p = q;
        q = tmp;
    }
    if (q >= n) return;  // dummy column of the odd-n padding
    double *gp = G + blockIdx.y * strideG + (long long)p * m;
    double *gq = G + blockIdx.y * strideG + (long long)q * m;
    double aa = 0.0, bb = 0.0, ab = 0.0;
    for (int i = threadIdx.x; i < m; i += JT) {
        double a = gp[i], b = gq[i];
        aa = fma(a, a, aa);
        bb = fma(b, b, bb);
        ab = fma(a, b, ab);
    }
    block_sum3(aa, bb, ab);
    if (aa == 0.0 && bb == 0.0) return;
    const bool swap = aa < bb;      // keep the larger column at the lower index
    double c = 1.0, s = 0.0;
    bool rot = false;
    // A column that has collapsed to (numerically) nothing -- the surplus columns of a matrix with
    // fewer rows than columns, exact null vectors -- carries no direction (and its products
    // underflow): it is left alone.  1e-20 |G|_F is far below anything the path keeps (RANK_TOL).
    const double dead = 1e-40 * fro2[blockIdx.y];
    if (aa > dead && bb > dead) {
        double cosv = fabs(ab) / sqrt(aa * bb);
        // one threshold for "rotate" and "not converged" (as LAPACK's dgesvj): a converged pair is
        // never touched again, so rounding in the rotations cannot keep the sweep count alive
        if (cosv > tol) {
            if (threadIdx.x == 0) atomicMax(maxcos, (unsigned long long)__double_as_longlong(cosv));
            double zeta = (bb - aa) / (2.0 * ab);
            double tt = copysign(1.0, zeta) / (fabs(zeta) + sqrt(1.0 + zeta * zeta));
            c = 1.0 / sqrt(1.0 + tt * tt);
            s = c * tt;
            rot = true;
        }
    }
    if (!rot && !swap) return;
    for (int i = threadIdx.x; i < m; i += JT) {
        double a = gp[i], b = gq[i];
        double na = c * a - s * b, nb = s * a + c * b;
        gp[i] = swap ? nb : na;
        gq[i] = swap ? na : nb;
    }
    double *vp = V + blockIdx.y * strideV + (long long)p * n;
    double *vq = V + blockIdx.y * strideV + (long long)q * n;
    for (int i = threadIdx.x; i < n; i += JT) {
        double a = vp[i], b = vq[i];
        double na = c * a - s * b, nb = s * a + c * b;
        vp[i] = swap ? nb : na;
        vq[i] = swap ? na : nb;
    }
}

__global__ void __launch_bounds__(JT) colnorm_kernel(const double *__restrict__ G, int m, int n,
                                                    long long strideG, double *__restrict__ s,
                                                    long long strideS)
{
    const double *g = G + blockIdx.y * strideG + (long long)blockIdx.x * m;
    double a = 0.0, b = 0.0, c = 0.0;
    for (int i = threadIdx.x; i < m; i += JT) a = fma(g[i], g[i], a);
    block_sum3(a, b, c);
    if (threadIdx.x == 0) s[blockIdx.y * strideS + blockIdx.x] = sqrt(a);
}

// perm[rank] = original column; sorted norms written to s_out
__global__ void rank_kernel(const double *__restrict__ s_in, int n, int *__restrict__ perm,
                            double *__restrict__ s_out, long long strideS)
{
    const double *si = s_in + (long long)blockIdx.x * n;
    for (int j = threadIdx.x; j < n; j += blockDim.x) {
        double v = si[j];
        int r = 0;
        for (int i = 0; i < n; ++i) {
            double u = si[i];
            r += (u > v) || (u == v && i < j);
        }
        perm[(long long)blockIdx.x * n + r] = j;
        s_out[blockIdx.x * strideS + r] = v;
    }
}

__global__ void permute_cols_kernel(const double *__restrict__ in, double *__restrict__ out, int rows,
                                    int n, const int *__restrict__ perm, long long stride)
{
    const int j = blockIdx.x;
    const int src = perm[(long long)blockIdx.y * n + j];
    const double *a = in + blockIdx.y * stride + (long long)src * rows;
    double *b = out + blockIdx.y * stride + (long long)j * rows;
    for (int i = threadIdx.x; i < rows; i += blockDim.x) b[i] = a[i];
}

}  // namespace

void jacobi_svd(double *G, int m, int n, double *V, double *s, int batch, long long strideG,
                long long strideV, long long strideS)
{
    if (n < 1 || m < 1 || batch < 1) return;
    if (batch == 1 && m <= 64 && n <= 64) {
        svd_small(G, m, n, V, s);
        return;
    }
    size_t mark = ws_mark();
    for (int b = 0; b < batch; ++b) fill_identity(V + b * strideV, n);
    const int npad = n + (n & 1);
    const int mn = m > n ? m : n;
    const double tol = 8.0 * sqrt((double)(mn > 16 ? mn : 16)) * 1.1102230246251565e-16;
    unsigned long long *flag = (unsigned long long *)ws_alloc(sizeof(unsigned long long));
    double *fro2 = ws_doubles(batch);
    for (int b = 0; b < batch; ++b) sumsq(G + b * strideG, (long long)m * n, fro2 + b);
    const int max_sweeps = 300;
    int sweep = 0;
    if (n > 1) {
        for (; sweep < max_sweeps; ++sweep) {
            TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(unsigned long long), stream()));
            dim3 grid(npad / 2, batch);
            for (int r = 0; r < npad - 1; ++r)
                jacobi_round_kernel<<<grid, JT, 0, stream()>>>(G, m, n, V, r, npad, strideG, strideV, tol, fro2, flag);
            TATRG_LAUNCH_CHECK();
            count_launch(npad - 1);
            unsigned long long h = 0;
            TATRG_CUDA_CHECK(cudaMemcpyAsync(&h, flag, sizeof(h), cudaMemcpyDeviceToHost, stream()));
            TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
            if (h == 0) break;
        }
        if (sweep == max_sweeps) fail(-34, "jacobi_svd: no convergence after %d sweeps (m=%d n=%d)", max_sweeps, m, n);
    }
    // sort by decreasing norm
    double *s_un = ws_doubles((long long)batch * n);
    int *perm = (int *)ws_alloc(sizeof(int) * (size_t)batch * n);
    colnorm_kernel<<<dim3(n, batch), JT, 0, stream()>>>(G, m, n, strideG, s_un, n);
    rank_kernel<<<batch, 256, 0, stream()>>>(s_un, n, perm, s, strideS);
    double *tmp = ws_doubles((long long)m * n > (long long)n * n ? (long long)m * n : (long long)n * n);
    for (int b = 0; b < batch; ++b) {
        permute_cols_kernel<<<dim3(n, 1), JT, 0, stream()>>>(G + b * strideG, tmp, m, n, perm + (long long)b * n, 0);
        TATRG_CUDA_CHECK(cudaMemcpyAsync(G + b * strideG, tmp, sizeof(double) * m * n, cudaMemcpyDeviceToDevice, stream()));
        permute_cols_kernel<<<dim3(n, 1), JT, 0, stream()>>>(V + b * strideV, tmp, n, n, perm + (long long)b * n, 0);
        TATRG_CUDA_CHECK(cudaMemcpyAsync(V + b * strideV, tmp, sizeof(double) * n * n, cudaMemcpyDeviceToDevice, stream()));
    }
    TATRG_LAUNCH_CHECK();
    count_launch(2 + 2 * batch);
    ws_release(mark);
}

}  // namespace tatrg
