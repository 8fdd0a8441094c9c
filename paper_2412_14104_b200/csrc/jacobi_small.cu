// jacobi_small.cu -- the small dense SVD / symmetric eigenproblems of the path solved by ONE CTA in
// shared memory (no launch per rotation round): the l x l core of the RSVD (
// reading O9), the canonical-form SVD, the Ritz step of the isometries (Eq. 3) and
// the b x b cores of the squeezer's subspace iteration (Eq. 12).  n <= 64.
//
//   svd mode: one-sided (Hestenes) Jacobi on the columns of [G; V] stacked (V starts as identity),
//             G_in V = U diag(s); round-robin ordering, warps own pairs, lanes own rows.
//   sym mode: two-sided Jacobi on the symmetric S: S <- J^T S J, V <- V J; converges in a handful of
//             sweeps whatever the grading of the spectrum and returns a complete orthonormal basis
//             also when S is rank deficient (the one-sided iteration on a graded PSD matrix needs
//             30+ sweeps: its columns start almost parallel).
// Results are sorted by decreasing singular value / eigenvalue.
#include "common.h"

namespace tatrg {

namespace {

constexpr int SJ_NT = 1024;   // eig_small_kernel
constexpr int SV_NT = 256;    // svd_small_kernel: 8 warps x 4 pairs, 8 lanes per pair
constexpr int SV_LPP = 8;     // lanes per pair
constexpr int SJ_MAX = 64;

__device__ __forceinline__ double warp_sum(double v)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__device__ __forceinline__ void rr_pair(int round, int pi, int npad, int &p, int &q)
{
    const int nm1 = npad - 1;
    if (pi == 0) {
        p = nm1;
        q = round;
    } else {
        p = (round + pi) % nm1;
        q = (round - pi + nm1) % nm1;
    }
    if (p > q) {
        int t = p;
        p = q;
        q = t;
    }
}

// column stride of the working array: rows of G, rows of V, and a pad that spreads the four pairs of a warp
// over the shared-memory banks
__host__ __device__ inline int svd_small_ld(int m, int n) { return m + n + (((m + n) & 15) == 0 ? 8 : 0); }

// G: m x n column-major (ld = m) in global; on exit G = U diag(s) sorted, V (n x n column-major), s[n].
// A round of the round-robin ordering rotates n/2 disjoint column pairs.  A pair is latency, not work (one dot
// product, ~40 dependent FP64 operations for the rotation, 2 (m + n) updated entries), and the FP64 pipe issues
// one warp instruction whatever the number of lanes that need it: so a warp takes FOUR pairs, eight lanes each
// (the rotation is computed once per warp instruction for four pairs), and 8 warps cover the 32 pairs of n = 64.
__global__ void __launch_bounds__(SV_NT) svd_small_kernel(double *__restrict__ Gg, int m, int n,
                                                         double *__restrict__ Vg, double *__restrict__ sg,
                                                         double tol, int max_sweeps, int *__restrict__ fail_flag)
{
    extern __shared__ double sm[];
    const int ld = svd_small_ld(m, n);   // column j = sm[j*ld .. j*ld+m) (G part) then n entries of V
    double *W = sm;
    __shared__ int nrot;
    __shared__ double fro2_s;
    __shared__ double nrm[SJ_MAX];
    __shared__ int perm[SJ_MAX];
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    constexpr int NW = SV_NT / 32;
    constexpr unsigned FULL = 0xffffffffu;

    for (int i = t; i < n * ld; i += SV_NT) {
        int j = i / ld, r = i - j * ld;
        W[i] = (r < m) ? Gg[(long long)j * m + r] : ((r - m == j) ? 1.0 : 0.0);
    }
    __syncthreads();
    {   // Frobenius norm (for the dead-column rule)
        double a = 0.0;
        for (int i = t; i < n * ld; i += SV_NT) {
            int r = i % ld;
            if (r < m) a = fma(W[i], W[i], a);
        }
        a = warp_sum(a);
        if (t == 0) fro2_s = 0.0;
        __syncthreads();
        if (lane == 0) atomicAdd(&fro2_s, a);
        __syncthreads();
    }
    const double dead = 1e-40 * fro2_s;
    const double tol2 = tol * tol;
    const int npad = n + (n & 1);
    const int sub = lane & (SV_LPP - 1), grp = lane / SV_LPP;
    int sweep = 0;
    for (; n > 1 && sweep < max_sweeps; ++sweep) {
        if (t == 0) nrot = 0;
        // squared column norms: recomputed once per sweep, then carried through the rotations
        // (a_pp' = a_pp - t a_pq, a_qq' = a_qq + t a_pq), so that a pair costs one dot product
        for (int j = warp; j < n; j += NW) {
            double a = 0.0;
            for (int i = lane; i < m; i += 32) a = fma(W[j * ld + i], W[j * ld + i], a);
            a = warp_sum(a);
            if (lane == 0) nrm[j] = a;
        }
        __syncthreads();
        for (int round = 0; round < npad - 1; ++round) {
            // every lane of the warp runs through the same instructions (no branch of its own before the shuffles)
            for (int pi0 = warp * (32 / SV_LPP); pi0 < npad / 2; pi0 += NW * (32 / SV_LPP)) {
                const int pi = pi0 + grp;
                int p = 0, q = 0;
                if (pi < npad / 2) rr_pair(round, pi, npad, p, q);
                const bool valid = pi < npad / 2 && q < n;
                if (!valid) p = q = 0;
                double *cp = W + p * ld, *cq = W + q * ld;
                const double aa = nrm[p], bb = nrm[q];
                double ab0 = 0.0, ab1 = 0.0;
                for (int i = sub; i < m; i += 2 * SV_LPP) {
                    ab0 = fma(cp[i], cq[i], ab0);
                    if (i + SV_LPP < m) ab1 = fma(cp[i + SV_LPP], cq[i + SV_LPP], ab1);
                }
                double ab = ab0 + ab1;
                for (int o = SV_LPP / 2; o > 0; o >>= 1) ab += __shfl_xor_sync(FULL, ab, o);
                const bool live = valid && !(aa == 0.0 && bb == 0.0);
                const bool swap = live && aa < bb;
                double c = 1.0, s = 0.0, na2 = aa, nb2 = bb;
                bool rot = false;
                if (live && aa > dead && bb > dead && ab * ab > tol2 * aa * bb) {
                    // tan of the rotation angle: the smaller root of t^2 + 2 zeta t - 1 = 0, zeta = (bb - aa) / (2 ab)
                    const double dlt = bb - aa;
                    const double tt = copysign(2.0 * fabs(ab), dlt * ab) / (fabs(dlt) + sqrt(fma(dlt, dlt, 4.0 * ab * ab)));
                    c = rsqrt(fma(tt, tt, 1.0));
                    s = c * tt;
                    na2 = aa - tt * ab;
                    nb2 = bb + tt * ab;
                    rot = true;
                }
                if (rot || swap) {
                    for (int i = sub; i < m + n; i += SV_LPP) {
                        double a = cp[i], b = cq[i];
                        double na = c * a - s * b, nb = s * a + c * b;
                        cp[i] = swap ? nb : na;
                        cq[i] = swap ? na : nb;
                    }
                    if (sub == 0) {
                        nrm[p] = swap ? nb2 : na2;
                        nrm[q] = swap ? na2 : nb2;
                        if (rot) atomicAdd(&nrot, 1);
                    }
                }
                __syncwarp();
            }
            __syncthreads();
        }
        if (nrot == 0) break;
        __syncthreads();
    }
    if (t == 0 && sweep >= max_sweeps && n > 1) *fail_flag = 1;
    // norms, ranks, permuted write-back
    for (int j = warp; j < n; j += NW) {
        double a = 0.0;
        for (int i = lane; i < m; i += 32) a = fma(W[j * ld + i], W[j * ld + i], a);
        a = warp_sum(a);
        if (lane == 0) nrm[j] = sqrt(a);
    }
    __syncthreads();
    if (t < n) {
        double v = nrm[t];
        int r = 0;
        for (int i = 0; i < n; ++i) r += (nrm[i] > v) || (nrm[i] == v && i < t);
        perm[r] = t;
    }
    __syncthreads();
    for (int i = t; i < n * ld; i += SV_NT) {
        int j = i / ld, r = i - j * ld;
        double v = W[perm[j] * ld + r];
        if (r < m)
            Gg[(long long)j * m + r] = v;
        else if (r < m + n)
            Vg[(long long)j * n + (r - m)] = v;
    }
    if (t < n) sg[t] = nrm[perm[t]];
}

// S: n x n symmetric (row- or column-major alike); on exit V (n x n, column j = eigenvector j,
// stored column-major) and lam[n] descending.
__global__ void __launch_bounds__(SJ_NT) eig_small_kernel(const double *__restrict__ Sg, int n,
                                                         double *__restrict__ Vg, double *__restrict__ lg,
                                                         int max_sweeps, int *__restrict__ fail_flag)
{
    extern __shared__ double sm[];
    const int ld = n + 1;
    double *S = sm;                 // S[r*ld + c]
    double *V = sm + n * ld;        // V[c*ld + r] : column c contiguous
    __shared__ double cs[SJ_MAX / 2][2];
    __shared__ int pq[SJ_MAX / 2][2];
    __shared__ double dmax;
    __shared__ int nrot;
    __shared__ double dg[SJ_MAX];
    __shared__ int perm[SJ_MAX];
    const int t = threadIdx.x;

    for (int i = t; i < n * n; i += SJ_NT) {
        int r = i / n, c = i - r * n;
        S[r * ld + c] = 0.5 * (Sg[i] + Sg[(long long)c * n + r]);
        V[c * ld + r] = (r == c) ? 1.0 : 0.0;
    }
    __syncthreads();
    const int npad = n + (n & 1), half = npad / 2;
    // entries below 1e-20 of the largest diagonal entry are dead (far below anything the path keeps)
    if (t == 0) {
        double d = 0.0;
        for (int i = 0; i < n; ++i) d = fmax(d, fabs(S[i * ld + i]));
        dmax = d;
    }
    __syncthreads();
    const double floor_abs = 1e-20 * dmax;
    int sweep = 0;
    for (; n > 1 && sweep < max_sweeps; ++sweep) {
        if (t == 0) nrot = 0;
        __syncthreads();
        for (int round = 0; round < npad - 1; ++round) {
            if (t < half) {
                int p, q;
                rr_pair(round, t, npad, p, q);
                double c = 1.0, s = 0.0;
                if (q < n) {
                    double apq = S[p * ld + q], app = S[p * ld + p], aqq = S[q * ld + q];
                    // the classical relative criterion: a pair is converged when |a_pq| <= eps sqrt(|a_pp a_qq|)
                    if (fabs(apq) > floor_abs && fabs(apq) > 2.2e-16 * sqrt(fabs(app * aqq))) {
                        atomicAdd(&nrot, 1);
                        const double dlt = aqq - app;
                        const double tt = copysign(2.0 * fabs(apq), dlt * apq) / (fabs(dlt) + sqrt(fma(dlt, dlt, 4.0 * apq * apq)));
                        c = rsqrt(fma(tt, tt, 1.0));
                        s = c * tt;
                    }
                } else {
                    q = -1;
                }
                pq[t][0] = p;
                pq[t][1] = q;
                cs[t][0] = c;
                cs[t][1] = s;
            }
            __syncthreads();
            // columns: S <- S J, V <- V J   (pair index = i / n, row = i % n)
            for (int i = t; i < half * n; i += SJ_NT) {
                int k = i / n, r = i - k * n;
                int p = pq[k][0], q = pq[k][1];
                if (q < 0) continue;
                double c = cs[k][0], s = cs[k][1];
                double a = S[r * ld + p], b = S[r * ld + q];
                S[r * ld + p] = c * a - s * b;
                S[r * ld + q] = s * a + c * b;
                double va = V[p * ld + r], vb = V[q * ld + r];
                V[p * ld + r] = c * va - s * vb;
                V[q * ld + r] = s * va + c * vb;
            }
            __syncthreads();
            // rows: S <- J^T S
            for (int i = t; i < half * n; i += SJ_NT) {
                int k = i / n, cc = i - k * n;
                int p = pq[k][0], q = pq[k][1];
                if (q < 0) continue;
                double c = cs[k][0], s = cs[k][1];
                double a = S[p * ld + cc], b = S[q * ld + cc];
                S[p * ld + cc] = c * a - s * b;
                S[q * ld + cc] = s * a + c * b;
            }
            __syncthreads();
        }
        if (nrot == 0) break;
        __syncthreads();
    }
    if (t == 0 && sweep >= max_sweeps && n > 1) *fail_flag = 1;
    if (t < n) dg[t] = S[t * ld + t];
    __syncthreads();
    if (t < n) {
        double v = dg[t];
        int r = 0;
        for (int i = 0; i < n; ++i) r += (dg[i] > v) || (dg[i] == v && i < t);
        perm[r] = t;
    }
    __syncthreads();
    for (int i = t; i < n * n; i += SJ_NT) {
        int j = i / n, r = i - j * n;
        Vg[i] = V[perm[j] * ld + r];
    }
    if (t < n) lg[t] = dg[perm[t]];
}

bool attr_done = false;
void set_attr()
{
    if (attr_done) return;
    TATRG_CUDA_CHECK(cudaFuncSetAttribute(svd_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)(SJ_MAX * svd_small_ld(SJ_MAX, SJ_MAX) * sizeof(double))));
    TATRG_CUDA_CHECK(cudaFuncSetAttribute(eig_small_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)(2 * SJ_MAX * (SJ_MAX + 1) * sizeof(double))));
    attr_done = true;
}

}  // namespace

void svd_small_async(double *G, int m, int n, double *V, double *s, int *flag_dev, double tol_override)
{
    if (m > SJ_MAX || n > SJ_MAX || m < 1 || n < 1) fail(-22, "svd_small: size %d x %d not supported", m, n);
    set_attr();
    const int mn = m > n ? m : n;
    const double tol = tol_override > 0.0 ? tol_override : 8.0 * sqrt((double)(mn > 16 ? mn : 16)) * 1.1102230246251565e-16;
    const size_t smem = (size_t)n * svd_small_ld(m, n) * sizeof(double);
    svd_small_kernel<<<1, SV_NT, smem, stream()>>>(G, m, n, V, s, tol, 100, flag_dev);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

// One-CTA SVD; requires m, n <= 64.  Same contract as jacobi_svd (batch 1).
void svd_small(double *G, int m, int n, double *V, double *s)
{
    size_t mark = ws_mark();
    int *flag = (int *)ws_alloc(sizeof(int));
    TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(int), stream()));
    svd_small_async(G, m, n, V, s, flag);
    int h = 0;
    TATRG_CUDA_CHECK(cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
    TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
    ws_release(mark);
    if (h) fail(-34, "svd_small: no convergence (m=%d n=%d)", m, n);
}

void eig_small_async(const double *S, int n, double *V, double *lam, int *flag_dev)
{
    if (n > SJ_MAX || n < 1) fail(-22, "eig_small: n = %d not supported", n);
    set_attr();
    const size_t smem = (size_t)2 * n * (n + 1) * sizeof(double);
    eig_small_kernel<<<1, SJ_NT, smem, stream()>>>(S, n, V, lam, 60, flag_dev);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

// One-CTA symmetric eigensolver; n <= 64.  V column-major (column j = eigenvector j), lam descending.
void eig_small(const double *S, int n, double *V, double *lam)
{
    size_t mark = ws_mark();
    int *flag = (int *)ws_alloc(sizeof(int));
    TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(int), stream()));
    eig_small_async(S, n, V, lam, flag);
    int h = 0;
    TATRG_CUDA_CHECK(cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
    TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
    ws_release(mark);
    if (h) fail(-34, "eig_small: no convergence (n=%d)", n);
}

}  // namespace tatrg
