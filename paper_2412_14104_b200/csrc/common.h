// common.h -- shared declarations of libtatrg (CUDA product path; no code shared with oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string>
#include <vector>

namespace tatrg {

// Mixed-radix index map: idx = d0 + n0*(d1 + n1*(d2 + n2*d3)) -> d0*s0 + d1*s1 + d2*s2 + d3*s3
// (element offsets).  Every leg permutation / leg grouping of the path's contractions is
// expressed with these, so no transpose kernel ever runs.
// An unused level has radix RADIX_INF (its quotient is always 0).
#define TATRG_RADIX_INF 0x7fffffffu
struct Map4 {
    unsigned n0, n1, n2, pad;
    long long s0, s1, s2, s3;
};

__host__ __device__ __forceinline__ long long map_off(const Map4 &m, unsigned i)
{
    unsigned q0 = i / m.n0;
    long long off = (long long)(i - q0 * m.n0) * m.s0;
    if (q0) {
        unsigned q1 = q0 / m.n1;
        off += (long long)(q0 - q1 * m.n1) * m.s1;
        if (q1) {
            unsigned q2 = q1 / m.n2;
            off += (long long)(q1 - q2 * m.n2) * m.s2 + (long long)q2 * m.s3;
        }
    }
    return off;
}

// the same for the summed index in front of a k tile's copies: no integer division when it is one leg, or two
// legs with a power-of-two faster one (the common cases; the divisions cost 2 % of the persistent GEMM's time on
// the contraction shapes and more in the small tiles, whose threads evaluate the map up to 32 times per k tile)
__host__ __device__ __forceinline__ long long map_off_k(const Map4 &m, unsigned i)
{
    if (m.n0 == TATRG_RADIX_INF) return (long long)i * m.s0;
    if (m.n1 == TATRG_RADIX_INF && (m.n0 & (m.n0 - 1u)) == 0u) {
#ifdef __CUDA_ARCH__
        const int sh = __ffs((int)m.n0) - 1;
#else
        int sh = 0;
        while ((1u << sh) < m.n0) ++sh;
#endif
        return (long long)(i & (m.n0 - 1u)) * m.s0 + (long long)(i >> sh) * m.s1;
    }
    return map_off(m, i);
}

inline Map4 map1(long long s) { return Map4{TATRG_RADIX_INF, TATRG_RADIX_INF, TATRG_RADIX_INF, 0, s, 0, 0, 0}; }

// C[b][cm(m)+cn(n)] (+)= alpha * sum_k A[b][am(m)+ak(k)] * B[b][bk(k)+bn(n)]
struct GemmParams {
    const double *A;
    const double *B;
    double *C;
    int M, N, K, batch;
    Map4 am, ak, bk, bn, cm, cn;
    Map4 ab, bb, cb;       // batch index maps of A, B, C
    double alpha;
    int accumulate;        // C += instead of C =
    int lower_only;        // symmetric output (A^T A): tiles strictly above the diagonal are skipped, the
                           // upper triangle of C is then undefined
    int a_kfast, b_kfast;  // loader thread order: 1 = consecutive threads walk k (k is the contiguous index)
    int ksplit;            // >1: partial sums go to `partial`, reduced by a second kernel
    int ktiles_per_split;  // in units of BK
    double *partial;       // [ksplit][batch][M][N]
    int tiles_n;           // set by the launcher: column tiles of the chosen CTA tile
    int tri_b;             // the caller promises B[k][n] = 0 for k > n (a triangular factor applied from the right):
                           // the persistent tile skips the k tiles that hold only those zeros (same result bit for bit)
};

// algorithmic flops of one launch (a symmetric lower-only output counts its lower triangle, a triangular
// B its non-zero part)
inline double gemm_flops(const GemmParams &p)
{
    if (p.tri_b) {   // sum over n of min(K, n + 1)
        const double full = p.N > p.K ? (double)(p.N - p.K) * p.K : 0.0;
        const double t = (double)(p.N < p.K ? p.N : p.K);
        return 2.0 * (double)p.M * (0.5 * t * (t + 1.0) + full) * p.batch;
    }
    const double mn = p.lower_only ? 0.5 * p.M * ((double)p.N + 1.0) : (double)p.M * p.N;
    return 2.0 * mn * (double)p.K * p.batch;
}

// ---- context -------------------------------------------------------------------------
cudaStream_t stream();
void count_launch(int n = 1);
void count_flops(double f);
void trace_mark(const char *label);   // TATRG_TRACE: labelled timestamp on the main stream
int prof_begin(double flops, int big);
void prof_end(int slot);
void prof_shape(int M, int N, int K, int batch, int ksplit);   // shape of the next profiled launch (trace)
int set_error(int code, const char *fmt, ...);
void *ws_alloc(size_t bytes);          // bump allocation from the caller's workspace (throws Err)
double *ws_doubles(long long n);
size_t ws_mark();
void ws_release(size_t mark);

struct Err {
    int code;
};

#define TATRG_CUDA_CHECK(expr)                                                         \
    do {                                                                               \
        cudaError_t _e = (expr);                                                       \
        if (_e != cudaSuccess) {                                                       \
            ::tatrg::set_error(-5, "CUDA error %s at %s:%d", cudaGetErrorString(_e),   \
                               __FILE__, __LINE__);                                    \
            throw ::tatrg::Err{-5};                                                    \
        }                                                                              \
    } while (0)
#define TATRG_LAUNCH_CHECK() TATRG_CUDA_CHECK(cudaGetLastError())

[[noreturn]] void fail(int code, const char *fmt, ...);

// ---- kernels (host launchers) ----------------------------------------------------------
// gemm.cu
void tensor_gemm(GemmParams p);
void tensor_gemm_big(const GemmParams &p, int bn);   // gemm_big.cu: the 128 x bn CTA tile, bn = 128 or 64
bool tensor_gemm_persistent(const GemmParams &p, int num_sms);   // gemm_p.cu: persistent 128 x 128 tile; false = not taken
bool tensor_gemm_tma(const GemmParams &p, int num_sms);          // gemm_tma.cu: TMA-fed producer (plain 2D operands); false = not taken
bool tensor_gemm_ts(const GemmParams &p);   // ts.cu: HBM-bound tall-and-skinny shapes; false = not taken
double probe_fp64_peak(int mode, int iters);
// qr.cu : thin QR with R_ii >= 0 of the row-major m x n matrix Y (ld = n), m >= 1, n <= 256.
// Q overwrites Y; R (n x n, row-major, upper triangular) to Rout (device).
void tsqr(double *Y, long long m, int n, double *Rout);
// Asynchronous Cholesky-QR of a tall block (n <= 256): `passes` rounds of {C = Y^T Y (+ shift_rel * max diag),
// C = L L^T, Y <- Y L^-T}; no host synchronisation.  A failed factorisation raises *flag_dev (sticky);
// ratio_dev (optional) receives min / max of the first pass's diag(L); Rout (optional, n x n row-major)
// receives the accumulated triangular factor.  The caller checks the flag when it next synchronises.
// src (optional): the block is read from there and Q written to Y (src itself is left alone).
// last_Linv (optional, n x n row-major; passes >= 2): the last pass's factor is not applied but returned, Y then
// holds Q' with Q = Q' last_Linv^T (the identity when the block took a route that applies every pass).
void cholqr_async(double *Y, long long m, int n, int passes, double shift_rel, int *flag_dev, double *ratio_dev,
                  double *Rout, const double *src = nullptr, double *last_Linv = nullptr);
// cholqr_fused.cu : the same for blocks of <= 64 columns (1 or 2 passes) as one resident grid; false = not taken
bool cholqr_fused(double *Y, long long m, int n, int passes, double shift_rel, int *flag_dev, double *ratio_dev,
                  double *Rout);
// jacobi.cu : one-sided Jacobi SVD of `batch` column-major m x n matrices (ld = m), m >= n.
// On exit G = U*diag(s) (columns orthogonal, sorted by decreasing norm), V (n x n, column
// major) accumulates the rotations (G_in * V = G_out), s[n] = column norms (descending).
void jacobi_svd(double *G, int m, int n, double *V, double *s, int batch, long long strideG,
                long long strideV, long long strideS);
// jacobi_small.cu : one-CTA versions for m, n <= 64 (same output conventions)
void svd_small(double *G, int m, int n, double *V, double *s);
// without host synchronisation: no convergence within the sweep limit raises *flag_dev (sticky, device)
// tol_override > 0: convergence threshold on the column cosines (default: a few eps), for estimates
void svd_small_async(double *G, int m, int n, double *V, double *s, int *flag_dev, double tol_override = 0.0);
void eig_small_async(const double *S, int n, double *V, double *lam, int *flag_dev);
void eig_small(const double *S, int n, double *V, double *lam);   // symmetric S; V column j = eigenvector j
// reduce.cu
void sumsq(const double *x, long long n, double *out);                       // out[0] = sum x^2
void dot(const double *x, const double *y, long long n, double *out);        // out[0] = sum x y
void sumsq_static(const double *x, long long n, double *out);                // sumsq with static scratch: no workspace, no allocation
void scale_by_rsqrt(double *x, long long n, const double *sumsq_dev);        // x *= 1/sqrt(*sumsq)
// x[i, c] *= f(v[c]) for a row-major (rows x cols) array; mode 0: v, 1: 1/v, 2: sqrt(v), 3: 1/sqrt(v), 4: v^2
void scale_cols(double *x, long long rows, int cols, const double *v, int mode);
// x[r, c] *= f(v[r])
void scale_rows(double *x, long long rows, long long cols, const double *v, int mode);
// x[i] *= f(v[(i / inner) % n]) : scales a tensor along one leg (inner = its stride, n = its size);
// mode 5: v^-3/2
void scale_leg(double *x, long long total, long long inner, long long n, const double *v, int mode);
void scale_inner_copy(const double *src, double *dst, long long total, long long n, const double *v);   // dst[.., c] = src[.., c] * v[c]
void symmetrize(double *x, int n);                                            // x = (x + x^T)/2
void fill_identity(double *x, int n);
void fill_zero(double *x, long long n);
void transpose_small(const double *in, double *out, int rows, int cols);      // out[c,r] = in[r,c]
void max_dev_identity(const double *G, int n, double *out);                   // out[0] = max |G - I| over the lower triangle
// chol.cu : in place lower Cholesky factor of the symmetric n x n matrix A (+ shift_rel * max diag on the
// diagonal); false if a pivot was not positive
bool cholesky_lower(double *A, int n, double shift_rel, double *Linv_full = nullptr);
// the same without host synchronisation: a non-positive pivot raises *flag_dev (sticky, device)
void cholesky_lower_async(double *A, int n, double shift_rel, double *Linv_full, int *flag_dev);
// G = I + E, |E| <~ 1e-8: in place lower Cholesky factor and its inverse by the first-order formulas (error O(|E|^2))
void near_identity_chol(double *G, int n, double *Linv);
void diag_minmax(const double *L, int n, double *out);   // out[0..1] = min, max of diag(L), L n x n row-major
void chol_block(double *A, long long lda, int n, double *Linv, int *flag, double *dminmax, double shift_rel = 0.0);
// rng.cu : out[0..n) = the seeded N(0,1) stream `subseed` (the recipe of seeded_inputs/), generated on the device
void device_fill_gauss(double *out, unsigned long long n, unsigned long long subseed);
// gauge.cu
void cluster_qr(const double *P, int ldp, double *W, int n, const int *bounds_dev, int nclusters);

}  // namespace tatrg
