// rng.cu -- the device implementation of the seeded Gaussian input recipe (DESIGN.md
// "Input recipe"), used when the caller does not hand the sketches / gauge references over with
// tatrg_set_sketch.  Same counter-based generator as the host module seeded_inputs/ (which the oracle
// draws from; the rules allow each side its own implementation of the same generator):
//   h(k) = mix(subseed + (k + 1) * golden),  u = ((h >> 11) + 0.5) / 2^53,
//   pair p: r = sqrt(-2 ln u(2p)), element 2p = r cos(2 pi u(2p+1)), element 2p+1 = r sin(2 pi u(2p+1)).
// The values equal the host generator's up to the last-bit differences of the libm functions; a caller
// who needs the host-generated bits supplies them (bench.py's end-to-end arm does).
#include "common.h"

namespace tatrg {

namespace {

__device__ __forceinline__ unsigned long long mix64(unsigned long long z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

__device__ __forceinline__ double u01(unsigned long long subseed, unsigned long long k)
{
    const unsigned long long h = mix64(subseed + (k + 1ULL) * 0x9E3779B97F4A7C15ULL);
    return ((double)(h >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

__global__ void fill_gauss_kernel(double *__restrict__ out, unsigned long long n, unsigned long long subseed)
{
    const unsigned long long pairs = (n + 1) >> 1;
    for (unsigned long long p = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; p < pairs;
         p += (unsigned long long)gridDim.x * blockDim.x) {
        const double u1 = u01(subseed, 2ULL * p), u2 = u01(subseed, 2ULL * p + 1ULL);
        const double r = sqrt(-2.0 * log(u1));
        double s, c;
        sincos(6.283185307179586476925286766559 * u2, &s, &c);
        out[2ULL * p] = r * c;
        if (2ULL * p + 1ULL < n) out[2ULL * p + 1ULL] = r * s;
    }
}

}  // namespace

void device_fill_gauss(double *out, unsigned long long n, unsigned long long subseed)
{
    if (n == 0) return;
    const unsigned long long pairs = (n + 1) >> 1;
    const int blocks = (int)(pairs / 256 + 1 < 148ULL * 16 ? pairs / 256 + 1 : 148ULL * 16);
    fill_gauss_kernel<<<blocks, 256, 0, stream()>>>(out, n, subseed);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

}  // namespace tatrg
