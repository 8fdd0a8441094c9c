// sq_iter.cu -- the subspace iteration of one squeezer (Eq. 12; reading G10; DESIGN.md
// "Squeezers") as ONE launch.
//
// The top chi singular triplets of F = L_L^T L_R (N2 x N2, N2 = n^2) are found by the block iteration
// Q <- orth(F orth(F^T Q)) with a block of 64 columns (step.cpp: SqChain).  Written as separate launches,
// one half step (a product with F or F^T, then one or two Cholesky-QR passes) is eight dependent launches of
// a few microseconds of work each, and a squeezer takes 25 - 40 half steps: the chain is pure launch and
// dependency latency (0.35 ms per iteration measured at chi = 32, against 10 us of arithmetic).  Here a small
// resident grid runs the whole list of half steps, separated by grid-wide barriers:
//
//   product      CTA c owns UT blocks of 8 rows of the output (UT = 1, 2, 4, 8, 16: a template parameter).  Its
//                rows of F (or of the transposed copy F^T: both products read rows) go straight from global
//                memory into DMMA.8x8x4 A fragments, each element once per CTA, one group of 8 summed indices
//                ahead; the 64-column iterate is staged by all threads with cp.async.cg (L2: other CTAs wrote it
//                before the last barrier) into a four-stage ring of shared-memory tiles of 32 rows that every warp
//                reads as B fragments.  Warps: min(UT, 8) row groups x 8 / min(UT, 8) column groups.
//   Cholesky-QR  partial Gram of the CTA's own rows (kept in shared memory) -> barrier -> every CTA sums its
//                share of the 64 x 64 entries over the partial Grams in a fixed order (deterministic) ->
//                barrier -> EVERY CTA factors the same 64 x 64 Gram (chol64.cuh: identical code on identical
//                bytes, so all CTAs hold the same L^-1) and applies it to its own rows -> barrier.
//
// The grid is sized by the caller to fit into the SMs that the persistent GEMM leaves free (step.cpp:
// CHAIN_SM_RESERVE), one CTA per SM; a CTA that finds no SM yet simply arrives late at the first barrier
// (every kernel it could be waiting behind ends on its own).
#include <algorithm>
#include "ctx.h"
#include "chol64.cuh"
#include "sq_iter.h"

namespace tatrg {

namespace {

constexpr int SQ_B = 64;        // block width of the iteration
constexpr int SQ_NT = CH64_NT;  // 8 warps
constexpr int SQ_LD = 68;       // row stride of the Y / L^-1 tiles: conflict-free fragment reads
constexpr int SQ_BK = 32;       // rows of the iterate per staged tile
constexpr int SQ_NST = 4;       // staged tiles in flight
constexpr int SQ_LDB = 66;      // row stride of the staged tile: rows 2q + e of a B fragment fall into distinct banks

template <int UT>
struct SqSmem {
    double Ys[UT * 8][SQ_LD];            // the CTA's rows of the current block
    union {
        double Bs[SQ_NST][SQ_BK][SQ_LDB];   // product: staged rows of the iterate
        Chol64Work wk;                      // Cholesky-QR: scratch of the factorisation, then ...
        double Ls[SQ_B][SQ_LD];             // ... L^-1 of the current pass
    };
    double diag[CH64];
    int bad;
};

__device__ __forceinline__ void dmma(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

__device__ __forceinline__ unsigned ld_acquire(const unsigned *p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc, bool valid)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    const int bytes = valid ? 16 : 0;   // 0: the 16 bytes are zero-filled
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(gsrc), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

// all CTAs of the grid; `target` counts the arrivals expected so far
__device__ __forceinline__ void grid_barrier(unsigned *bar, unsigned &target)
{
    target += gridDim.x;
    __syncthreads();
    if (threadIdx.x == 0) {
        // release: the CTA's writes (ordered before this by the barrier above) are visible to whoever acquires the count
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;\n" ::"l"(bar) : "memory");
        while (ld_acquire(bar) < target) {
        }
    }
    __syncthreads();
}

template <int UT>
__global__ void __launch_bounds__(SQ_NT, 1) sq_iter_kernel(const __grid_constant__ SqIterParams p)
{
    constexpr int RW = UT >= 8 ? 8 : UT;     // row groups of warps
    constexpr int RBW = UT >= 8 ? UT / 8 : 1;   // 8-row blocks per warp
    constexpr int NCB = 8 / (8 / RW);        // 8-column blocks per warp  (8 / RW column groups)
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SqSmem<UT> &sm = *reinterpret_cast<SqSmem<UT> *>(smem_raw);
    const int t = threadIdx.x, warp = t >> 5, lane = t & 31, g = lane >> 2, q = lane & 3;
    const int N2 = p.N2;
    const int row0 = blockIdx.x * UT * 8;    // first row of this CTA
    const bool vecF = (N2 & 1) == 0;
    const int wr = warp % RW, wc = warp / RW;   // this warp's row group / column group in the product
    const int ntiles = (N2 + SQ_BK - 1) / SQ_BK;
    unsigned target = 0;

    for (int st = 0; st < p.nsteps; ++st) {
        const int code = p.steps[st];
        const bool trans = code & SQ_TRANS;
        const double *__restrict__ src = (code & SQ_FROM_START) ? p.start : p.buf[trans ? 0 : 1];
        double *__restrict__ dst = p.buf[trans ? 1 : 0];
        const double *__restrict__ F = trans ? p.Ft : p.F;
        const int passes = (code & SQ_TWO_PASSES) ? 2 : 1;
        const int slot = (code >> SQ_RATIO_SHIFT) & 3;

        // ---- product: out[r, z] = sum_k F[r, k] in[k, z]
        {
            double acc[RBW][NCB][2];
#pragma unroll
            for (int rb = 0; rb < RBW; ++rb)
#pragma unroll
                for (int cb = 0; cb < NCB; ++cb) acc[rb][cb][0] = acc[rb][cb][1] = 0.0;
            // the order of the summed index inside a group of 8 is free: DMMA step e sums k = k8 + 2 q + e
            const double *frow[RBW];
            bool rok[RBW];
#pragma unroll
            for (int rb = 0; rb < RBW; ++rb) {
                const int r = row0 + (wr * RBW + rb) * 8 + g;
                rok[rb] = r < N2;
                frow[rb] = F + (long long)(rok[rb] ? r : 0) * N2 + 2 * q;
            }
            auto load_a = [&](int k8, double (&a)[RBW][2]) {
#pragma unroll
                for (int rb = 0; rb < RBW; ++rb) {
                    a[rb][0] = a[rb][1] = 0.0;
                    const int ka = k8 + 2 * q;
                    if (rok[rb]) {
                        if (vecF && ka + 1 < N2) {
                            const double2 v = __ldg(reinterpret_cast<const double2 *>(frow[rb] + k8));
                            a[rb][0] = v.x;
                            a[rb][1] = v.y;
                        } else {
                            if (ka < N2) a[rb][0] = __ldg(frow[rb] + k8);
                            if (ka + 1 < N2) a[rb][1] = __ldg(frow[rb] + k8 + 1);
                        }
                    }
                }
            };
            auto stage_b = [&](int tile, int buf) {   // rows tile*BK .. of the iterate: BK x 64 doubles = 1024 chunks
#pragma unroll
                for (int i = 0; i < (SQ_BK * SQ_B / 2) / SQ_NT; ++i) {
                    const int ch = t + i * SQ_NT, kr = ch >> 5, c2 = (ch & 31) * 2;
                    const int k = tile * SQ_BK + kr;
                    cp_async16(&sm.Bs[buf][kr][c2], src + (long long)(k < N2 ? k : 0) * SQ_B + c2, k < N2);
                }
                cp_async_commit();
            };
            double a_cur[RBW][2], a_nxt[RBW][2];
#pragma unroll
            for (int i = 0; i < SQ_NST - 1; ++i) {
                if (i < ntiles)
                    stage_b(i, i);
                else
                    cp_async_commit();
            }
            load_a(0, a_cur);
#pragma unroll 1
            for (int tile = 0; tile < ntiles; ++tile) {
                const int buf = tile % SQ_NST;
                cp_async_wait<SQ_NST - 2>();   // tile `tile` has landed (one group per tile, empty ones past the end)
                __syncthreads();               // ... for every thread, and everybody is done with tile - 1
                if (tile + SQ_NST - 1 < ntiles)
                    stage_b(tile + SQ_NST - 1, (tile + SQ_NST - 1) % SQ_NST);
                else
                    cp_async_commit();
#pragma unroll
                for (int kk = 0; kk < SQ_BK; kk += 8) {
                    load_a(tile * SQ_BK + kk + 8, a_nxt);   // beyond N2: zeros, no loads
#pragma unroll
                    for (int cb = 0; cb < NCB; ++cb) {
                        const int col = (wc * NCB + cb) * 8 + g;
                        const double b0 = sm.Bs[buf][kk + 2 * q][col], b1 = sm.Bs[buf][kk + 2 * q + 1][col];
#pragma unroll
                        for (int rb = 0; rb < RBW; ++rb) {
                            dmma(acc[rb][cb][0], acc[rb][cb][1], a_cur[rb][0], b0);
                            dmma(acc[rb][cb][0], acc[rb][cb][1], a_cur[rb][1], b1);
                        }
                    }
#pragma unroll
                    for (int rb = 0; rb < RBW; ++rb) {
                        a_cur[rb][0] = a_nxt[rb][0];
                        a_cur[rb][1] = a_nxt[rb][1];
                    }
                }
            }
            cp_async_wait<0>();
            __syncthreads();
#pragma unroll
            for (int rb = 0; rb < RBW; ++rb)
#pragma unroll
                for (int cb = 0; cb < NCB; ++cb)
                    *reinterpret_cast<double2 *>(&sm.Ys[(wr * RBW + rb) * 8 + g][(wc * NCB + cb) * 8 + 2 * q]) =
                        make_double2(acc[rb][cb][0], acc[rb][cb][1]);
            __syncthreads();
        }

        for (int pass = 0; pass < passes; ++pass) {
            // ---- partial Gram of the CTA's rows: warp w -> Gram rows 8w .. 8w+7, all 64 columns
            {
                double gacc[8][2];
#pragma unroll
                for (int cb = 0; cb < 8; ++cb) gacc[cb][0] = gacc[cb][1] = 0.0;
#pragma unroll 2
                for (int k0 = 0; k0 < UT * 8; k0 += 4) {
                    const double a = sm.Ys[k0 + q][warp * 8 + g];
#pragma unroll
                    for (int cb = 0; cb < 8; ++cb) dmma(gacc[cb][0], gacc[cb][1], a, sm.Ys[k0 + q][cb * 8 + g]);
                }
                double *pp = p.part + (long long)blockIdx.x * (SQ_B * SQ_B) + (warp * 8 + g) * SQ_B + 2 * q;
#pragma unroll
                for (int cb = 0; cb < 8; ++cb) *reinterpret_cast<double2 *>(pp + cb * 8) = make_double2(gacc[cb][0], gacc[cb][1]);
            }
            grid_barrier(p.bar, target);
            // ---- this CTA's share of the Gram entries, summed over the partial Grams in a fixed order
            for (int e = blockIdx.x * SQ_NT + t; e < SQ_B * SQ_B; e += gridDim.x * SQ_NT) {
                const double *pe = p.part + e;
                const int G = (int)gridDim.x;
                double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
                int c = 0;
                for (; c + 4 <= G; c += 4) {
                    s0 += __ldcg(pe + (long long)c * (SQ_B * SQ_B));
                    s1 += __ldcg(pe + (long long)(c + 1) * (SQ_B * SQ_B));
                    s2 += __ldcg(pe + (long long)(c + 2) * (SQ_B * SQ_B));
                    s3 += __ldcg(pe + (long long)(c + 3) * (SQ_B * SQ_B));
                }
                for (; c < G; ++c) s0 += __ldcg(pe + (long long)c * (SQ_B * SQ_B));
                p.gram[e] = (s0 + s1) + (s2 + s3);
            }
            grid_barrier(p.bar, target);
            // ---- every CTA: G (+ shift) = L L^T, L^-1
            {
                const int ty = t >> 4, tx = t & 15;
                double s[4][4], w[4][4];
#pragma unroll
                for (int a = 0; a < 4; ++a)
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        const int i = 4 * ty + a, c = 4 * tx + b;
                        const int r = i > c ? i : c, cc = i > c ? c : i;   // lower-triangle source
                        s[a][b] = __ldcg(p.gram + r * SQ_B + cc);
                        if (i == c) sm.diag[i] = s[a][b];
                    }
                __syncthreads();
                chol64_factor(s, w, sm.wk, sm.diag, &sm.bad, SQ_B, (passes == 1) ? p.shift : 0.0);
#pragma unroll
                for (int a = 0; a < 4; ++a)
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        const int i = 4 * ty + a, c = 4 * tx + b;
                        sm.Ls[i][c] = (c <= i) ? w[a][b] : 0.0;   // (the factorisation's scratch is dead: it ended with a barrier)
                        if (blockIdx.x == 0 && (code & SQ_WANT_R)) p.Lkeep[pass * (SQ_B * SQ_B) + i * SQ_B + c] = (c <= i) ? s[a][b] : 0.0;
                    }
                if (blockIdx.x == 0 && t == 0) {
                    if (sm.bad) *p.flag = 1;
                    if (slot && pass == 0) {
                        double lo = sm.diag[0], hi = sm.diag[0];
                        for (int j = 1; j < SQ_B; ++j) {
                            lo = fmin(lo, sm.diag[j]);
                            hi = fmax(hi, sm.diag[j]);
                        }
                        p.ratio[2 * (slot - 1)] = lo;
                        p.ratio[2 * (slot - 1) + 1] = hi;
                    }
                }
                __syncthreads();
            }
            // ---- Y <- Y L^-T on the CTA's rows: out[r, d] = sum_c Y[r, c] Linv[d, c]; warp w -> columns d = 8w ..
            {
                double bf[16];
#pragma unroll
                for (int ks = 0; ks < 16; ++ks) bf[ks] = sm.Ls[warp * 8 + g][ks * 4 + q];
                const bool final_pass = pass == passes - 1;
                // 8 row blocks at a time: the results wait in registers until every warp has read the old rows
#pragma unroll 1
                for (int u0 = 0; u0 < UT; u0 += 8) {
                    constexpr int UB = UT < 8 ? UT : 8;
                    double o[UB][2];
#pragma unroll
                    for (int u = 0; u < UB; ++u) {
                        o[u][0] = o[u][1] = 0.0;
#pragma unroll
                        for (int ks = 0; ks < 16; ++ks) dmma(o[u][0], o[u][1], sm.Ys[(u0 + u) * 8 + g][ks * 4 + q], bf[ks]);
                    }
                    __syncthreads();
#pragma unroll
                    for (int u = 0; u < UB; ++u) {
                        const double2 v = make_double2(o[u][0], o[u][1]);
                        *reinterpret_cast<double2 *>(&sm.Ys[(u0 + u) * 8 + g][warp * 8 + 2 * q]) = v;
                        const int r = row0 + (u0 + u) * 8 + g;
                        if (final_pass && r < N2) *reinterpret_cast<double2 *>(dst + (long long)r * SQ_B + warp * 8 + 2 * q) = v;
                    }
                }
                __syncthreads();
            }
        }
        // ---- R = L2^T L1^T of a two-pass step (R[i][j] = sum_k L2[k][i] L1[j][k]); one pass: R = L1^T.  The factors
        // are staged in shared memory first (from global memory this short loop of dependent loads took 100 us)
        if (blockIdx.x == 0 && (code & SQ_WANT_R) && p.Rout) {
            constexpr int LDS_ = SQ_B + 1;
            double *L1s = &sm.Bs[0][0][0], *L2s = L1s + SQ_B * LDS_;   // 2 x 64 x 65 doubles fit into the staging ring
            static_assert(2 * SQ_B * LDS_ <= SQ_NST * SQ_BK * SQ_LDB, "staging ring too small for the two factors");
            __syncthreads();
            for (int e = t; e < SQ_B * SQ_B; e += SQ_NT) {
                L1s[(e >> 6) * LDS_ + (e & 63)] = __ldcg(p.Lkeep + e);
                L2s[(e >> 6) * LDS_ + (e & 63)] = passes == 2 ? __ldcg(p.Lkeep + SQ_B * SQ_B + e) : 0.0;
            }
            __syncthreads();
            for (int e = t; e < SQ_B * SQ_B; e += SQ_NT) {
                const int i = e / SQ_B, j = e % SQ_B;
                double sum = 0.0;
                if (passes == 2) {
#pragma unroll 4
                    for (int k = i; k < SQ_B; ++k) sum = fma(L2s[k * LDS_ + i], L1s[j * LDS_ + k], sum);
                } else {
                    sum = L1s[j * LDS_ + i];
                }
                p.Rout[e] = sum;
            }
            __syncthreads();
        }
        if (st + 1 < p.nsteps) grid_barrier(p.bar, target);
    }
}

template <int UT>
void launch_ut(const SqIterParams &p, int grid)
{
    static bool attr_done = false;
    if (!attr_done) {
        TATRG_CUDA_CHECK(cudaFuncSetAttribute(sq_iter_kernel<UT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(SqSmem<UT>)));
        TATRG_CUDA_CHECK(cudaFuncSetAttribute(sq_iter_kernel<UT>, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        attr_done = true;
    }
    sq_iter_kernel<UT><<<grid, SQ_NT, sizeof(SqSmem<UT>), stream()>>>(p);
}

int blocks_per_cta(int N2, int wanted)   // smallest power of two with ceil(nblk / UT) <= wanted
{
    const int nblk = (N2 + 7) / 8;
    int ut = 1;
    while (ut < SQ_UMAX && (nblk + ut - 1) / ut > std::max(1, wanted)) ut *= 2;
    return ut;
}

}  // namespace

size_t sq_iter_scratch_doubles(int grid) { return (size_t)(grid + 3) * SQ_B * SQ_B + 2; }

int sq_iter_grid(int N2, int wanted)
{
    const int nblk = (N2 + 7) / 8, ut = blocks_per_cta(N2, wanted);
    return (nblk + ut - 1) / ut;
}

void sq_iter_launch(SqIterParams p, int wanted, double *scratch)
{
    if (p.nsteps < 1 || p.nsteps > SQ_MAXSTEPS) fail(-22, "sq_iter: %d half steps", p.nsteps);
    const int nblk = (p.N2 + 7) / 8, ut = blocks_per_cta(p.N2, wanted), grid = (nblk + ut - 1) / ut;
    p.part = scratch;
    p.gram = scratch + (size_t)grid * SQ_B * SQ_B;
    p.Lkeep = p.gram + SQ_B * SQ_B;
    p.bar = reinterpret_cast<unsigned *>(p.Lkeep + 2 * SQ_B * SQ_B);
    TATRG_CUDA_CHECK(cudaMemsetAsync(p.bar, 0, sizeof(unsigned), stream()));
    switch (ut) {
    case 1: launch_ut<1>(p, grid); break;
    case 2: launch_ut<2>(p, grid); break;
    case 4: launch_ut<4>(p, grid); break;
    case 8: launch_ut<8>(p, grid); break;
    default: launch_ut<16>(p, grid); break;
    }
    TATRG_LAUNCH_CHECK();
    count_launch();
    double fl = 0.0;
    for (int i = 0; i < p.nsteps; ++i)
        fl += 2.0 * p.N2 * (double)p.N2 * SQ_B + ((p.steps[i] & SQ_TWO_PASSES) ? 2 : 1) * 4.0 * p.N2 * (double)SQ_B * SQ_B;
    count_flops(fl);
}

}  // namespace tatrg
