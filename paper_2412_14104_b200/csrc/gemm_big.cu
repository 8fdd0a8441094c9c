// gemm_big.cu -- the non-persistent 128x64 (outputs at most 64 columns wide, two CTAs per SM) and 128x128
// CTA tiles of the tensor-GEMM (see gemm.cu for the operation; the hot 128x128 shapes run on the persistent
// tile of gemm_p.cu):
//   C[b][cm(m)+cn(n)] (+)= alpha * sum_k A[b][am(m)+ak(k)] * B[b][bk(k)+bn(n)]
// on the FP64 tensor pipe (mma.sync m8n8k4 -> DMMA.8x8x4).  This is the kernel the O(q r chi^7) bond
// swap (Table 1) and the O(r^2 chi^7) triad contraction (Eqs. 13-14)
// run on.
//
// 128x128: 16 warps, warp tile 32 x 32 (32 FP64 accumulators per thread), BK = 32, 3-stage cp.async
// pipeline synchronised by per-stage mbarriers ("full": the copies of all threads have landed, "empty":
// all threads are done reading) instead of a CTA-wide barrier per k tile.  128x64: 8 warps, warp tile
// 32 x 32, BK = 16, 3 stages, the same mbarrier pipeline, two CTAs per SM.
// The shared-memory layout of an operand tile follows the operand's contiguous index in global
// memory, so that 16-byte cp.async copies land on 16 consecutive bytes of shared memory:
//   contiguous index = the free index (m or n):  tile stored [k][m], leading dimension 128 + 4
//   contiguous index = the summed index k:       tile stored [m][k], leading dimension  16 + 4
// Both leading dimensions are = 4 (mod 8) doubles, which makes the 8-byte DMMA fragment loads
// (lane -> (row = lane/4, k = lane%4)) conflict free.  Leg permutations stay folded into the gather
// addresses (Map4); the 16-byte path is taken when every pair of consecutive elements along the
// contiguous index is 16-byte aligned in global memory (checked on the host), else 8-byte copies.
#include "common.h"

namespace tatrg {

namespace {

constexpr int BM = 128;
constexpr int LD_F = BM + 4;   // [k][m] layout; the [m][k] layout has leading dimension BK + 4
constexpr int RASTER_W = 12;

__device__ __forceinline__ void cp_async(double *smem_dst, const double *gsrc, int bytes, int vec)
{
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    if (vec)
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(gsrc), "r"(bytes));
    else
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(d), "l"(gsrc), "r"(bytes));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}
// ---- mbarrier helpers (shared::cta): per-stage "full" / "empty" barriers of the decoupled pipeline
__device__ __forceinline__ void mbar_init(unsigned long long *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *bar)
{
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}\n" ::"r"((unsigned)__cvta_generic_to_shared(bar))
                 : "memory");
}
// arrives on `bar` once all cp.async copies issued so far by this thread have landed
__device__ __forceinline__ void mbar_arrive_on_cp_async(unsigned long long *bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        " .reg .pred p;\n"
        "WAIT_%=:\n"
        " mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        " @p bra DONE_%=;\n"
        " bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)),
        "r"(parity)
        : "memory");
}

__device__ __forceinline__ void dmma(double &d0, double &d1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(d0), "+d"(d1)
                 : "d"(a), "d"(b));
}

// Loader of one ROWS x BK operand tile by NT threads.  KF: k is the contiguous index in global
// memory.  VEC: 16-byte copies (pairs along the contiguous index), else 8-byte copies.
template <bool KF, bool VEC, int ROWS, int NT, int BK>
struct TileLoader {
    static constexpr int LD_K = BK + 4;
    static constexpr int W = VEC ? 2 : 1;             // elements per copy
    static constexpr int PER = ROWS * BK / (NT * W);  // copies per thread per tile
    static constexpr int TPR = NT / BK;               // !KF: threads along the free index per k row
    static constexpr int LDF = ROWS + 4;              // !KF: leading dimension of the [k][free] tile
    static_assert(PER >= 1 && PER * NT * W == ROWS * BK, "loader layout");
    long long fix[PER];                               // offsets of the free index (fixed over k tiles)
    int free_left[PER];                               // valid elements from this copy's free index on
    const double *base;
    int kl;                                           // this thread's k inside the tile
    int soff[PER];                                    // shared-memory offsets

    __device__ __forceinline__ void init(const double *b, const Map4 &mfree, int f0, int F, int t)
    {
        base = b;
        if (KF) {
            // k pairs (VEC) or singles along the 16-wide k; free index strided over threads
            constexpr int KT = BK / W;                // threads along k
            kl = (t % KT) * (VEC ? 2 : 1);
#pragma unroll
            for (int j = 0; j < PER; ++j) {
                int fl = t / KT + (NT / KT) * j;
                free_left[j] = F - (f0 + fl);
                fix[j] = free_left[j] > 0 ? map_off(mfree, f0 + fl) : 0;
                soff[j] = fl * LD_K + kl;
            }
        } else {
            // free-index pairs (VEC) or singles; TPR threads along the free index, k = t / TPR
            kl = t / TPR;
#pragma unroll
            for (int j = 0; j < PER; ++j) {
                int fl = ((t % TPR) + TPR * j) * W;
                free_left[j] = F - (f0 + fl);
                fix[j] = free_left[j] > 0 ? map_off(mfree, f0 + fl) : 0;
                soff[j] = kl * LDF + fl;
            }
        }
    }

    __device__ __forceinline__ void load(double *stage, const Map4 &mk, int k0, int K) const
    {
        const int k_left = K - (k0 + kl);
        const long long ko = k_left > 0 ? map_off_k(mk, (unsigned)(k0 + kl)) : 0;   // no integer division in the common cases
#pragma unroll
        for (int j = 0; j < PER; ++j) {
            int n;   // valid elements of this copy
            if (KF)
                n = free_left[j] > 0 ? min(k_left, VEC ? 2 : 1) : 0;
            else
                n = k_left > 0 ? min(free_left[j], VEC ? 2 : 1) : 0;
            n = max(n, 0);
            cp_async(stage + soff[j], n > 0 ? base + fix[j] + ko : base, n * 8, VEC);
        }
    }
};

template <bool A_KF, bool B_KF, bool VEC, int BN, int WN, int BK, int STAGES, bool MBAR>
__global__ void __launch_bounds__(128 * BN / WN, BN == 128 ? 1 : 2) tgemm_big_kernel(const __grid_constant__ GemmParams p)
{
    constexpr int LD_K = BK + 4;
    constexpr int NT = 128 * BN / WN;                 // (BM / 32) * (BN / WN) warps
    constexpr int LD_FB = BN + 4;                     // [k][n] layout of the B tile
    constexpr int A_STAGE = A_KF ? BM * LD_K : BK * LD_F;
    constexpr int B_STAGE = B_KF ? BN * LD_K : BK * LD_FB;
    constexpr int WM = 32, FM = WM / 8, FN = WN / 8;
    extern __shared__ __align__(16) double smem[];
    double *As = smem;
    double *Bs = smem + STAGES * A_STAGE;

    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    int tile_m, tile_n;
    {
        const int tiles_m = (p.M + BM - 1) / BM;
        const int band = blockIdx.x / (RASTER_W * p.tiles_n);
        const int in_band = blockIdx.x - band * (RASTER_W * p.tiles_n);
        const int w = min(RASTER_W, tiles_m - band * RASTER_W);
        tile_n = in_band / w;
        tile_m = band * RASTER_W + (in_band - tile_n * w);
    }
    const int m0 = tile_m * BM, n0 = tile_n * BN;
    if (p.lower_only && n0 >= m0 + BM) return;   // tile strictly above the diagonal of a symmetric output
    int bz = blockIdx.z;
    const int split = bz / p.batch;
    bz -= split * p.batch;

    // this CTA's range of the summed index (split-K ranges are given in units of 16)
    int k_begin = 0, k_end = p.K;
    if (p.ksplit > 1) {
        k_begin = min(p.K, split * p.ktiles_per_split * 16);
        k_end = min(p.K, k_begin + p.ktiles_per_split * 16);
    }
    const int nkt = (k_end - k_begin + BK - 1) / BK;

    TileLoader<A_KF, VEC, BM, NT, BK> la;
    TileLoader<B_KF, VEC, BN, NT, BK> lb;
    la.init(p.A + map_off(p.ab, bz), p.am, m0, p.M, t);
    lb.init(p.B + map_off(p.bb, bz), p.bn, n0, p.N, t);

    double acc[FM][FN][2];
#pragma unroll
    for (int i = 0; i < FM; ++i)
#pragma unroll
        for (int j = 0; j < FN; ++j) acc[i][j][0] = acc[i][j][1] = 0.0;

    const int wm0 = (warp & 3) * WM, wn0 = (warp >> 2) * WN;
    const int lr = lane >> 2, lk = lane & 3;
    // fragment base offsets inside a stage
    const int a_off = A_KF ? (wm0 + lr) * LD_K + lk : lk * LD_F + wm0 + lr;
    const int b_off = B_KF ? (wn0 + lr) * LD_K + lk : lk * LD_FB + wn0 + lr;
    constexpr int A_I = A_KF ? 8 * LD_K : 8;        // step between 8-row fragments
    constexpr int B_J = B_KF ? 8 * LD_K : 8;
    constexpr int A_KK = A_KF ? 4 : 4 * LD_F;       // step between k groups of 4
    constexpr int B_KK = B_KF ? 4 : 4 * LD_FB;

    // MBAR: every stage has a "full" barrier (all threads' copies of the tile have landed) and an
    // "empty" barrier (all threads are done reading it), so a warp only waits for data and for the
    // slot it refills -- never for the slowest warp of the current tile, as with the CTA-wide barrier.
    __shared__ unsigned long long full_bar[STAGES], empty_bar[STAGES];
    if (MBAR) {
        if (t == 0) {
#pragma unroll
            for (int s = 0; s < STAGES; ++s) {
                mbar_init(&full_bar[s], NT);
                mbar_init(&empty_bar[s], NT);
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if (s < nkt) {
            la.load(As + s * A_STAGE, p.ak, k_begin + s * BK, k_end);
            lb.load(Bs + s * B_STAGE, p.bk, k_begin + s * BK, k_end);
            if (MBAR) mbar_arrive_on_cp_async(&full_bar[s]);
        }
        cp_async_commit();
    }
    for (int it = 0; it < nkt; ++it) {
        const int slot = it % STAGES;
        if (MBAR) {
            mbar_wait(&full_bar[slot], (unsigned)(it / STAGES) & 1u);
        } else {
            cp_async_wait<STAGES - 2>();
            __syncthreads();
            const int nx = it + STAGES - 1;
            if (nx < nkt) {
                la.load(As + (nx % STAGES) * A_STAGE, p.ak, k_begin + nx * BK, k_end);
                lb.load(Bs + (nx % STAGES) * B_STAGE, p.bk, k_begin + nx * BK, k_end);
            }
            cp_async_commit();
        }
        const double *as = As + slot * A_STAGE + a_off;
        const double *bs = Bs + slot * B_STAGE + b_off;
#pragma unroll
        for (int kk = 0; kk < BK / 4; ++kk) {
            double a[FM], b[FN];
#pragma unroll
            for (int i = 0; i < FM; ++i) a[i] = as[kk * A_KK + i * A_I];
#pragma unroll
            for (int j = 0; j < FN; ++j) b[j] = bs[kk * B_KK + j * B_J];
#pragma unroll
            for (int i = 0; i < FM; ++i)
#pragma unroll
                for (int j = 0; j < FN; ++j) dmma(acc[i][j][0], acc[i][j][1], a[i], b[j]);
        }
        if (MBAR) {
            mbar_arrive(&empty_bar[slot]);             // this thread is done with the tile
            const int nx = it + STAGES - 1;            // refill the slot of tile it - 1
            if (nx < nkt) {
                const int ns = nx % STAGES;
                if (it >= 1) mbar_wait(&empty_bar[ns], (unsigned)((it - 1) / STAGES) & 1u);
                la.load(As + ns * A_STAGE, p.ak, k_begin + nx * BK, k_end);
                lb.load(Bs + ns * B_STAGE, p.bk, k_begin + nx * BK, k_end);
                mbar_arrive_on_cp_async(&full_bar[ns]);
            }
        }
    }
    cp_async_wait<0>();

    // ---- epilogue
    if (p.ksplit > 1) {
        double *P = p.partial + ((long long)split * p.batch + bz) * (long long)p.M * p.N;
#pragma unroll
        for (int i = 0; i < FM; ++i) {
            int m = m0 + wm0 + i * 8 + lr;
            if (m >= p.M) continue;
#pragma unroll
            for (int j = 0; j < FN; ++j) {
                int n = n0 + wn0 + j * 8 + lk * 2;
                if (n < p.N) P[(long long)m * p.N + n] = acc[i][j][0];
                if (n + 1 < p.N) P[(long long)m * p.N + n + 1] = acc[i][j][1];
            }
        }
        return;
    }
    double *Cb = p.C + map_off(p.cb, bz);
    long long cmo[FM];
    bool cmv[FM];
#pragma unroll
    for (int i = 0; i < FM; ++i) {
        int m = m0 + wm0 + i * 8 + lr;
        cmv[i] = m < p.M;
        cmo[i] = cmv[i] ? map_off(p.cm, m) : 0;
    }
#pragma unroll
    for (int j = 0; j < FN; ++j) {
        const int n = n0 + wn0 + j * 8 + lk * 2;
        const bool v0 = n < p.N, v1 = n + 1 < p.N;
        const long long c0 = v0 ? map_off(p.cn, n) : 0;
        const long long c1 = v1 ? map_off(p.cn, n + 1) : 0;
#pragma unroll
        for (int i = 0; i < FM; ++i) {
            if (!cmv[i]) continue;
            double *Cr = Cb + cmo[i];
            if (v0) {
                double v = p.alpha * acc[i][j][0];
                if (p.accumulate) v += Cr[c0];
                Cr[c0] = v;
            }
            if (v1) {
                double v = p.alpha * acc[i][j][1];
                if (p.accumulate) v += Cr[c1];
                Cr[c1] = v;
            }
        }
    }
}

template <bool A_KF, bool B_KF, bool VEC, int BN, int WN, int BK, int STAGES, bool MBAR>
void launch_big(const GemmParams &p_in)
{
    constexpr int NT = 128 * BN / WN;
    constexpr int LD_K = BK + 4;
    constexpr int A_STAGE = A_KF ? BM * LD_K : BK * LD_F;
    constexpr int B_STAGE = B_KF ? BN * LD_K : BK * (BN + 4);
    constexpr size_t smem = (size_t)STAGES * (A_STAGE + B_STAGE) * sizeof(double);
    static bool attr_done = false;
    auto kern = tgemm_big_kernel<A_KF, B_KF, VEC, BN, WN, BK, STAGES, MBAR>;
    if (!attr_done) {
        TATRG_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_done = true;
    }
    GemmParams p = p_in;
    p.tiles_n = (p.N + BN - 1) / BN;
    const long long tiles = (long long)((p.M + BM - 1) / BM) * p.tiles_n;
    if (tiles > 0x7fffffffLL) fail(-22, "tensor_gemm: too many tiles");
    dim3 grid((unsigned)tiles, 1, p.batch * (p.ksplit > 1 ? p.ksplit : 1));
    const int slot = prof_begin(gemm_flops(p), BN == 128);
    kern<<<grid, NT, smem, stream()>>>(p);
    prof_end(slot);
    TATRG_LAUNCH_CHECK();
    count_launch();
}

bool even_or_inf(unsigned n) { return n == TATRG_RADIX_INF || (n & 1u) == 0; }
bool even(long long s) { return (s & 1LL) == 0; }

// every level above the first has an even stride
bool upper_even(const Map4 &m) { return even(m.s1) && even(m.s2) && even(m.s3); }
bool all_even(const Map4 &m) { return even(m.s0) && upper_even(m); }

// 16-byte copies along the contiguous index `fast` of an operand (the other index is `slow`)
bool vec_ok(const double *base, const Map4 &fast, const Map4 &slow, const Map4 &batch)
{
    return ((uintptr_t)base & 15) == 0 && fast.s0 == 1 && even_or_inf(fast.n0) && upper_even(fast) && all_even(slow) &&
           all_even(batch);
}

template <int BN, int WN, int BK, int STAGES, bool MBAR>
void dispatch_big(const GemmParams &p)
{
    const bool akf = p.a_kfast != 0, bkf = p.b_kfast != 0;
    const bool va = akf ? vec_ok(p.A, p.ak, p.am, p.ab) : vec_ok(p.A, p.am, p.ak, p.ab);
    const bool vb = bkf ? vec_ok(p.B, p.bk, p.bn, p.bb) : vec_ok(p.B, p.bn, p.bk, p.bb);
    const bool vec = va && vb;
    if (akf) {
        if (bkf)
            vec ? launch_big<true, true, true, BN, WN, BK, STAGES, MBAR>(p) : launch_big<true, true, false, BN, WN, BK, STAGES, MBAR>(p);
        else
            vec ? launch_big<true, false, true, BN, WN, BK, STAGES, MBAR>(p) : launch_big<true, false, false, BN, WN, BK, STAGES, MBAR>(p);
    } else {
        if (bkf)
            vec ? launch_big<false, true, true, BN, WN, BK, STAGES, MBAR>(p) : launch_big<false, true, false, BN, WN, BK, STAGES, MBAR>(p);
        else
            vec ? launch_big<false, false, true, BN, WN, BK, STAGES, MBAR>(p) : launch_big<false, false, false, BN, WN, BK, STAGES, MBAR>(p);
    }
}

}  // namespace

// The 128 x 64 tile (two CTAs per SM) for outputs 17..64 columns wide and for short summed indices; the
// 128 x 128 instantiation is the fallback of the persistent tile (gemm_p.cu) for operands whose free-index
// offsets do not fit its 32-bit loader state.
void tensor_gemm_big(const GemmParams &p, int bn)
{
    if (bn == 64)
        dispatch_big<64, 32, 16, 3, true>(p);
    else
        dispatch_big<128, 32, 32, 3, true>(p);
}

}  // namespace tatrg
