/*
 * seeded_inputs/gauss.c -- counter-based seeded Gaussian INPUT generator.
 *
 * This file is the one piece of code that both the CPU oracle (oracle/) and the
 * CUDA product path (paper_2412_14104_b200/) are allowed to share: it produces
 * the seeded N(0,1) matrices the method *consumes* (RSVD sketches Omega,
 * PAPER.md:25, :106; gauge reference matrices) and holds none
 * of the method's arithmetic.
 *
 * Recipe:
 *   subseed = splitmix64(seed ^ (step << 8) ^ which)
 *   h(k)    = k-th output of the splitmix64 stream started at `subseed`
 *   pair p  : u1 = ((h(2p)   >> 11) + 0.5) / 2^53
 *             u2 = ((h(2p+1) >> 11) + 0.5) / 2^53
 *             r  = sqrt(-2 ln u1)
 *             element 2p = r cos(2 pi u2), element 2p+1 = r sin(2 pi u2)
 * Counter based, so any sub-range can be filled independently (threads).
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

#define SI_GOLDEN 0x9E3779B97F4A7C15ULL

static inline uint64_t si_mix(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

/* one splitmix64 step applied to x (the "hash" used to derive sub-seeds) */
uint64_t si_splitmix64(uint64_t x) { return si_mix(x + SI_GOLDEN); }

uint64_t si_subseed(uint64_t seed, uint64_t step, uint64_t which)
{
    return si_splitmix64(seed ^ (step << 8) ^ which);
}

static inline double si_u01(uint64_t subseed, uint64_t k)
{
    uint64_t h = si_mix(subseed + (k + 1ULL) * SI_GOLDEN);
    return ((double)(h >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

/* out[i] = element (offset + i) of the stream `subseed`, i in [0, n) */
void si_fill_gauss(double *out, uint64_t n, uint64_t subseed, uint64_t offset)
{
    const double two_pi = 6.283185307179586476925286766559;
    uint64_t first = offset, last = offset + n; /* element range [first,last) */
    uint64_t p0 = first >> 1, p1 = (last + 1) >> 1;
    long long p;
#pragma omp parallel for schedule(static)
    for (p = (long long)p0; p < (long long)p1; ++p) {
        double u1 = si_u01(subseed, 2ULL * (uint64_t)p);
        double u2 = si_u01(subseed, 2ULL * (uint64_t)p + 1ULL);
        double r = sqrt(-2.0 * log(u1));
        double a = two_pi * u2;
        uint64_t e0 = 2ULL * (uint64_t)p, e1 = e0 + 1ULL;
        if (e0 >= first && e0 < last) out[e0 - first] = r * cos(a);
        if (e1 >= first && e1 < last) out[e1 - first] = r * sin(a);
    }
}
