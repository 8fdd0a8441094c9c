// common.h -- shared declarations of libtatrg (CUDA product path; no code shared with oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string>
#include <vector>

namespace tatrg {

// Two-level index map: idx -> (idx % n0) * s0 + (idx / n0) * s1   (element offsets).
// Every leg permutation / leg grouping of the path's contractions is expressed with these,
// so no transpose kernel ever runs.
struct Map2 {
    long long n0, s0, s1;
};
__host__ __device__ inline long long map2(const Map2 &m, long long i)
{
    return (i % m.n0) * m.s0 + (i / m.n0) * m.s1;
}
// one-level map (stride s)
inline Map2 M1(long long s) { return Map2{1LL << 40, s, 0}; }
// two-level map: hi index (size irrelevant) stride s_hi, lo index of size n_lo stride s_lo
inline Map2 M2(long long s_hi, long long n_lo, long long s_lo) { return Map2{n_lo, s_lo, s_hi}; }

struct GemmParams {
    const double *A;
    const double *B;
    double *C;
    int M, N, K, batch;
    Map2 am, ak, bk, bn, cm, cn;
    long long a_bs, b_bs, c_bs;
    double alpha;
    int ksplit;            // >1: partial sums go to `partial`, reduced by a second kernel
    int ktiles_per_split;  // in units of BK
    double *partial;       // [ksplit][batch][M][N]
};

// ---- context -------------------------------------------------------------------------
struct Ctx;
Ctx &ctx();
cudaStream_t stream();
void count_launch(int n = 1);
void count_flops(double f);
int set_error(int code, const char *fmt, ...);
void *ws_alloc(size_t bytes);          // bump allocation from the caller's workspace (throws)
size_t ws_mark();
void ws_release(size_t mark);

struct WsError {
    int code;
};

#define TATRG_CUDA_CHECK(expr)                                                         \
    do {                                                                               \
        cudaError_t _e = (expr);                                                       \
        if (_e != cudaSuccess) {                                                       \
            ::tatrg::set_error(-5, "CUDA error %s at %s:%d", cudaGetErrorString(_e),   \
                               __FILE__, __LINE__);                                    \
            throw ::tatrg::WsError{-5};                                                \
        }                                                                              \
    } while (0)

// ---- kernels (host launchers) ----------------------------------------------------------
// gemm.cu
void tensor_gemm(GemmParams p);
double probe_fp64_peak(int mode, int iters);
// small.cu
void jacobi_svd(double *G, int ldg, int m, int n, double *V, int ldv, double *s, int *sweeps_out);
// reduce.cu
void sumsq(const double *x, long long n, double *out);                       // out[0] = sum x^2
void dot(const double *x, const double *y, long long n, double *out);        // out[0] = sum x y
void scale_by_rsqrt(double *x, long long n, const double *sumsq_dev);        // x *= 1/sqrt(*sumsq)
void scale_cols(double *x, long long rows, int cols, const double *v, int inv); // x[r,c] *= v[c]

}  // namespace tatrg
