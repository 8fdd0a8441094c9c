// gauge.cu -- gauge fixing of SVD / eigen bases against a seeded reference (DESIGN.md reading
// G12): for every cluster [c0, c1) of (near-)degenerate singular values, the basis block is
// rotated by the orthogonal factor of qr+(P[c0:c1, c0:c1]), P = basis^T * G_ref.  A cluster of
// size 1 is the sign convention <u, g_ref> > 0.  One CTA per cluster; clusters are tiny.
#include "common.h"

namespace tatrg {

namespace {

constexpr int CL_MAX = 32;

// W (n x n row-major) = blockdiag(Q_c), Q_c R_c = P[c0:c1, c0:c1], diag(R_c) >= 0.
__global__ void cluster_qr_kernel(const double *__restrict__ P, int ldp, double *__restrict__ W, int n,
                                  const int *__restrict__ bounds)
{
    __shared__ double a[CL_MAX][CL_MAX + 1];   // working copy -> R
    __shared__ double qm[CL_MAX][CL_MAX + 1];  // accumulates Q
    __shared__ double v[CL_MAX];
    const int c0 = bounds[blockIdx.x], c1 = bounds[blockIdx.x + 1];
    const int c = c1 - c0;
    const int t = threadIdx.x;   // blockDim.x == CL_MAX; thread t owns column t
    for (int i = 0; i < c; ++i)
        if (t < c) {
            a[i][t] = P[(long long)(c0 + i) * ldp + c0 + t];
            qm[i][t] = (i == t) ? 1.0 : 0.0;
        }
    __syncthreads();
    for (int j = 0; j < c; ++j) {
        // Householder vector from column j (every thread computes it redundantly)
        double xn2 = 0.0;
        for (int i = j + 1; i < c; ++i) xn2 += a[i][j] * a[i][j];
        double alpha = a[j][j];
        double beta = alpha, tau = 0.0, scal = 0.0;
        if (xn2 != 0.0) {
            beta = -copysign(sqrt(alpha * alpha + xn2), alpha);
            tau = (beta - alpha) / beta;
            scal = 1.0 / (alpha - beta);
        }
        __syncthreads();
        if (t < c) v[t] = (t < j) ? 0.0 : (t == j ? 1.0 : a[t][j] * scal);
        __syncthreads();
        if (t < c && tau != 0.0) {
            // A <- H A (column t), Q <- Q H (row t)
            double w = 0.0;
            for (int i = j; i < c; ++i) w += v[i] * a[i][t];
            w *= tau;
            for (int i = j; i < c; ++i) a[i][t] -= v[i] * w;
            double u = 0.0;
            for (int i = j; i < c; ++i) u += qm[t][i] * v[i];
            u *= tau;
            for (int i = j; i < c; ++i) qm[t][i] -= u * v[i];
        }
        __syncthreads();
    }
    // sign fix: Q <- Q diag(sign R_jj); write the block, zero the rest of the block rows
    if (t < c) {
        double sg = (a[t][t] < 0.0) ? -1.0 : 1.0;
        for (int i = 0; i < c; ++i) qm[i][t] *= sg;
    }
    __syncthreads();
    for (int i = 0; i < c; ++i)
        for (int col = t; col < n; col += blockDim.x) {
            double val = (col >= c0 && col < c1) ? qm[i][col - c0] : 0.0;
            W[(long long)(c0 + i) * n + col] = val;
        }
}

}  // namespace

void cluster_qr(const double *P, int ldp, double *W, int n, const int *bounds_dev, int nclusters)
{
    if (nclusters < 1) return;
    cluster_qr_kernel<<<nclusters, CL_MAX, 0, stream()>>>(P, ldp, W, n, bounds_dev);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

}  // namespace tatrg
