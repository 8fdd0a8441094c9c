// reduce.cu -- HBM-bound norm / trace / scaling kernels of the path:
//   per-step tensor normalisation c_m = |Phi|_F |Psi|_F and the trace tTr T = <Phi, Psi>
//   (Eq. 15 closed periodically; reading O8), plus the diagonal
//   scalings by sigma (Eq. 1, Eq. 5).  Vectorised 16-byte loads, grid = 8 CTAs per SM,
//   deterministic two-pass reductions (no atomics).
#include "common.h"

// Scratch of sumsq_static (below): the per-CTA partial sums of the two-pass reduction, one slot per CTA of the
// largest grid (148 x 8 = 1184 doubles = 9472 bytes).  A file-scope device array: every GPU that loads the library
// holds it until the process exits; no call allocates it.  In HOST code this name is a host-side stand-in, not a
// device address -- the launcher below asks the runtime for the address (cudaGetSymbolAddress) once per device.
#define TATRG_SUMSQ_STATIC_SLOTS (148 * 8)
static __device__ __align__(256) double g_sumsq_static_partials[TATRG_SUMSQ_STATIC_SLOTS];

namespace tatrg {

namespace {

constexpr int RED_THREADS = 256;
constexpr int RED_MAX_BLOCKS = 148 * 8;

__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double sh[32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sh[w] = v;
    __syncthreads();
    int nw = (blockDim.x + 31) >> 5;
    v = (threadIdx.x < nw) ? sh[threadIdx.x] : 0.0;
    if (w == 0)
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;  // valid in thread 0
}

// mode 0: sum x^2 ; mode 1: sum x*y
template <int MODE>
__global__ void __launch_bounds__(RED_THREADS) reduce_pass1(const double *__restrict__ x,
                                                           const double *__restrict__ y, long long n,
                                                           double *__restrict__ partial)
{
    double acc0 = 0.0, acc1 = 0.0;
    long long tid = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long stride = (long long)gridDim.x * blockDim.x;
    bool al = ((reinterpret_cast<uintptr_t>(x) & 15) == 0) &&
              (MODE == 0 || (reinterpret_cast<uintptr_t>(y) & 15) == 0);
    if (al) {
        long long n2 = n >> 1;
        const double2 *x2 = reinterpret_cast<const double2 *>(x);
        const double2 *y2 = reinterpret_cast<const double2 *>(y);
        for (long long i = tid; i < n2; i += stride) {
            double2 a = __ldg(x2 + i);
            if (MODE == 0) {
                acc0 = fma(a.x, a.x, acc0);
                acc1 = fma(a.y, a.y, acc1);
            } else {
                double2 b = __ldg(y2 + i);
                acc0 = fma(a.x, b.x, acc0);
                acc1 = fma(a.y, b.y, acc1);
            }
        }
        if ((n & 1) && tid == 0) {
            double a = x[n - 1];
            acc0 = fma(a, MODE == 0 ? a : y[n - 1], acc0);
        }
    } else {
        for (long long i = tid; i < n; i += stride) {
            double a = x[i];
            acc0 = fma(a, MODE == 0 ? a : y[i], acc0);
        }
    }
    double s = block_sum(acc0 + acc1);
    if (threadIdx.x == 0) partial[blockIdx.x] = s;
}

__global__ void __launch_bounds__(RED_THREADS) reduce_pass2(const double *__restrict__ partial, int n,
                                                           double *__restrict__ out)
{
    double a = 0.0;
    for (int i = threadIdx.x; i < n; i += blockDim.x) a += partial[i];
    a = block_sum(a);
    if (threadIdx.x == 0) out[0] = a;
}

__global__ void scale_rsqrt_kernel(double *__restrict__ x, long long n, const double *__restrict__ ss)
{
    const double f = 1.0 / sqrt(ss[0]);
    long long tid = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long stride = (long long)gridDim.x * blockDim.x;
    if ((reinterpret_cast<uintptr_t>(x) & 15) == 0) {
        long long n2 = n >> 1;
        double2 *x2 = reinterpret_cast<double2 *>(x);
        for (long long i = tid; i < n2; i += stride) {
            double2 a = x2[i];
            a.x *= f;
            a.y *= f;
            x2[i] = a;
        }
        if ((n & 1) && tid == 0) x[n - 1] *= f;
    } else {
        for (long long i = tid; i < n; i += stride) x[i] *= f;
    }
}

__device__ __forceinline__ double scale_fn(double v, int mode)
{
    switch (mode) {
        case 0: return v;
        case 1: return 1.0 / v;
        case 2: return sqrt(v > 0.0 ? v : 0.0);
        case 3: return 1.0 / sqrt(v);
        case 4: return v * v;
        default: return 1.0 / (v * sqrt(v));
    }
}

__global__ void scale_cols_kernel(double *__restrict__ x, long long total, int cols,
                                  const double *__restrict__ v, int mode)
{
    long long tid = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = tid; i < total; i += stride) x[i] *= scale_fn(v[i % cols], mode);
}

__global__ void scale_rows_kernel(double *__restrict__ x, long long total, long long cols,
                                  const double *__restrict__ v, int mode)
{
    long long tid = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = tid; i < total; i += stride) x[i] *= scale_fn(v[i / cols], mode);
}

// x[i] *= f(v[(i / inner) % n])
__global__ void scale_leg_kernel(double *__restrict__ x, long long total, long long inner, long long n,
                                 const double *__restrict__ v, int mode)
{
    long long tid = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = tid; i < total; i += stride) x[i] *= scale_fn(v[(i / inner) % n], mode);
}

// dst[i] = src[i] * v[i % n] for the innermost leg (n even, 16-byte aligned buffers): two elements per thread
__global__ void scale_inner_copy_kernel(const double2 *__restrict__ src, double2 *__restrict__ dst, long long pairs, int n,
                                        const double *__restrict__ v)
{
    long long tid = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = tid; i < pairs; i += stride) {
        const int c = (int)((2 * i) % n);
        double2 a = src[i];
        a.x *= v[c];
        a.y *= v[c + 1];
        dst[i] = a;
    }
}

// x = (x + x^T)/2, n x n
__global__ void symmetrize_kernel(double *x, int n)
{
    long long total = (long long)n * n;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x) {
        int r = (int)(i / n), c = (int)(i % n);
        if (r < c) {
            double a = 0.5 * (x[i] + x[(long long)c * n + r]);
            x[i] = a;
            x[(long long)c * n + r] = a;
        }
    }
}

__global__ void identity_kernel(double *x, int n)
{
    long long total = (long long)n * n;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x)
        x[i] = (i / n == i % n) ? 1.0 : 0.0;
}

__global__ void transpose_kernel(const double *__restrict__ in, double *__restrict__ out, int rows, int cols)
{
    long long total = (long long)rows * cols;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total;
         i += (long long)gridDim.x * blockDim.x) {
        int r = (int)(i / cols), c = (int)(i % cols);
        out[(long long)c * rows + r] = in[i];
    }
}

int grid_for(long long n, int per_thread = 4)
{
    long long b = (n + (long long)RED_THREADS * per_thread - 1) / ((long long)RED_THREADS * per_thread);
    if (b < 1) b = 1;
    if (b > RED_MAX_BLOCKS) b = RED_MAX_BLOCKS;
    return (int)b;
}

}  // namespace

void sumsq(const double *x, long long n, double *out)
{
    size_t mark = ws_mark();
    int g = grid_for(n, 8);
    double *partial = ws_doubles(g);
    reduce_pass1<0><<<g, RED_THREADS, 0, stream()>>>(x, nullptr, n, partial);
    reduce_pass2<<<1, RED_THREADS, 0, stream()>>>(partial, g, out);
    TATRG_LAUNCH_CHECK();
    count_launch(2);
    ws_release(mark);
}

void dot(const double *x, const double *y, long long n, double *out)
{
    size_t mark = ws_mark();
    int g = grid_for(n, 8);
    double *partial = ws_doubles(g);
    reduce_pass1<1><<<g, RED_THREADS, 0, stream()>>>(x, y, n, partial);
    reduce_pass2<<<1, RED_THREADS, 0, stream()>>>(partial, g, out);
    TATRG_LAUNCH_CHECK();
    count_launch(2);
    ws_release(mark);
}

// sumsq without any allocation and without the caller's workspace (tatrg_sumsq_static): the same two kernels on the
// same grid as sumsq -- the result is the same to the last bit -- with the partial sums in the file-scope array
// g_sumsq_static_partials.  Its device address is looked up once per device, with that device current.  Nothing in
// the array has to start at zero: pass 1 writes every slot that pass 2 reads.  All calls share the array, so two
// calls whose kernels overlap on the GPU (different streams, no dependency between them) race.
void sumsq_static(const double *x, long long n, double *out)
{
    constexpr int MAX_DEVICES = 64;
    static double *scratch_of_device[MAX_DEVICES] = {};
    int dev = -1;
    TATRG_CUDA_CHECK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) fail(-22, "sumsq_static: device ordinal %d not supported", dev);
    if (!scratch_of_device[dev]) {
        void *p = nullptr;
        TATRG_CUDA_CHECK(cudaGetSymbolAddress(&p, g_sumsq_static_partials));
        scratch_of_device[dev] = static_cast<double *>(p);
    }
    double *partial = scratch_of_device[dev];
    const int g = grid_for(n, 8);
    if (g > TATRG_SUMSQ_STATIC_SLOTS) fail(-22, "sumsq_static: %d partial sums exceed the %d static slots", g, TATRG_SUMSQ_STATIC_SLOTS);
    reduce_pass1<0><<<g, RED_THREADS, 0, stream()>>>(x, nullptr, n, partial);
    reduce_pass2<<<1, RED_THREADS, 0, stream()>>>(partial, g, out);
    TATRG_LAUNCH_CHECK();
    count_launch(2);
}

void scale_by_rsqrt(double *x, long long n, const double *sumsq_dev)
{
    scale_rsqrt_kernel<<<grid_for(n, 8), RED_THREADS, 0, stream()>>>(x, n, sumsq_dev);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

void scale_cols(double *x, long long rows, int cols, const double *v, int mode)
{
    long long total = rows * cols;
    if (total <= 0) return;
    scale_cols_kernel<<<grid_for(total), RED_THREADS, 0, stream()>>>(x, total, cols, v, mode);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

void scale_rows(double *x, long long rows, long long cols, const double *v, int mode)
{
    long long total = rows * cols;
    if (total <= 0) return;
    scale_rows_kernel<<<grid_for(total), RED_THREADS, 0, stream()>>>(x, total, cols, v, mode);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

void scale_leg(double *x, long long total, long long inner, long long n, const double *v, int mode)
{
    if (total <= 0) return;
    scale_leg_kernel<<<grid_for(total), RED_THREADS, 0, stream()>>>(x, total, inner, n, v, mode);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

// dst = src scaled along its innermost leg of size n (one pass instead of a copy and an in-place scaling)
void scale_inner_copy(const double *src, double *dst, long long total, long long n, const double *v)
{
    if (total <= 0) return;
    if ((n & 1) || (total & 1) || (((uintptr_t)src | (uintptr_t)dst) & 15)) {
        TATRG_CUDA_CHECK(cudaMemcpyAsync(dst, src, sizeof(double) * total, cudaMemcpyDeviceToDevice, stream()));
        scale_leg(dst, total, 1, n, v, 0);
        return;
    }
    scale_inner_copy_kernel<<<grid_for(total / 2), RED_THREADS, 0, stream()>>>(reinterpret_cast<const double2 *>(src),
                                                                              reinterpret_cast<double2 *>(dst), total / 2, (int)n, v);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

void symmetrize(double *x, int n)
{
    symmetrize_kernel<<<grid_for((long long)n * n), RED_THREADS, 0, stream()>>>(x, n);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

void fill_identity(double *x, int n)
{
    identity_kernel<<<grid_for((long long)n * n), RED_THREADS, 0, stream()>>>(x, n);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

void fill_zero(double *x, long long n)
{
    TATRG_CUDA_CHECK(cudaMemsetAsync(x, 0, n * sizeof(double), stream()));
}

// out[0] = max_{i >= j} |G_ij - delta_ij| (non-negative doubles order like their bit patterns)
__global__ void max_dev_identity_kernel(const double *__restrict__ G, int n, unsigned long long *__restrict__ out)
{
    const long long total = (long long)n * n;
    double m = 0.0;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const int r = (int)(i / n), c = (int)(i - (long long)r * n);
        if (c > r) continue;
        const double v = fabs(G[i] - (r == c ? 1.0 : 0.0));
        m = (v > m || v != v) ? v : m;
    }
    for (int o = 16; o > 0; o >>= 1) {
        const double w = __shfl_xor_sync(0xffffffffu, m, o);
        m = (w > m || w != w) ? w : m;
    }
    if ((threadIdx.x & 31) == 0) {
        if (m != m) m = INFINITY;
        atomicMax(out, (unsigned long long)__double_as_longlong(m));
    }
}

void max_dev_identity(const double *G, int n, double *out)
{
    TATRG_CUDA_CHECK(cudaMemsetAsync(out, 0, sizeof(double), stream()));
    max_dev_identity_kernel<<<grid_for((long long)n * n), RED_THREADS, 0, stream()>>>(G, n, (unsigned long long *)out);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

void transpose_small(const double *in, double *out, int rows, int cols)
{
    transpose_kernel<<<grid_for((long long)rows * cols), RED_THREADS, 0, stream()>>>(in, out, rows, cols);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

}  // namespace tatrg
