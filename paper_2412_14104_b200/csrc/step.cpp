// step.cpp -- host orchestration of one Triad-ATRG coarse-graining step (arXiv:2412.14104,
// /root/reference/PAPER.md Sec. 2): which kernels run, on which strided views, in which order.
// All arithmetic on tensors runs in the CUDA kernels (gemm.cu, qr.cu, jacobi.cu, reduce.cu,
// gauge.cu); the host takes the rank / cluster decisions on downloaded spectra (O(chi) scalars)
// and keeps the ln Z bookkeeping.
//
// Rotated frame (reading G8): legs (0 | 1, 2 | 3) = (coarse-graining direction |
// grouped transverse pair | lone transverse leg).  Leg letters used in the contractions below:
//   x,c  direction-0 legs        p,q / P,Q  pair legs of the upper / lower site
//   t / T  lone leg upper / lower   a,b  canonical bonds alpha, beta   g,d  swap bond gamma
//   k,l  oversampled internal lines (r chi)   m,n,w  renormalised legs   z  sketch columns
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <chrono>
#include <functional>

#include "ctx.h"
#include "sq_iter.h"

extern "C" {
uint64_t si_subseed(uint64_t seed, uint64_t step, uint64_t which);
void si_fill_gauss(double *out, uint64_t n, uint64_t subseed, uint64_t offset);
}

namespace tatrg {

namespace {

constexpr double RANK_TOL = 1e-14;     // reading G9
// SMs the persistent GEMM leaves free while chains of small kernels run beside it (measured at c3: 4 -> 81.7 ms
// per step, 8 -> 79.7, 12 -> 80.3, 20 -> 81.2)
constexpr int CHAIN_SM_RESERVE = 8;
constexpr int LONE_SM_RESERVE = 16;   // ... to the lone-leg squeezer beside the grouped-leg Gram chains (its iteration is one resident grid)
constexpr double CLUSTER_TOL = 1e-8;   // reading G12

std::vector<double> d2h(const double *p, long long n)
{
    std::vector<double> v((size_t)n);
    if (n > 0) {
        TATRG_CUDA_CHECK(cudaMemcpyAsync(v.data(), p, sizeof(double) * n, cudaMemcpyDeviceToHost, stream()));
        TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
    }
    return v;
}

void h2d(double *dst, const double *src, long long n)
{
    TATRG_CUDA_CHECK(cudaMemcpyAsync(dst, src, sizeof(double) * n, cudaMemcpyHostToDevice, stream()));
}

void d2d(double *dst, const double *src, long long n)
{
    TATRG_CUDA_CHECK(cudaMemcpyAsync(dst, src, sizeof(double) * n, cudaMemcpyDeviceToDevice, stream()));
}

int num_rank(const std::vector<double> &s, int cap)
{
    if (s.empty() || !(s[0] > 0)) return 0;
    int k = 0;
    for (double v : s) k += (v > RANK_TOL * s[0]);
    return cap >= 0 ? std::min(cap, k) : k;
}

double rel_gap(const std::vector<double> &s, int cut)
{
    if (cut <= 0 || cut >= (int)s.size()) return INFINITY;
    return (s[cut - 1] - s[cut]) / s[0];
}

// cluster boundaries of the first k values of the descending s
std::vector<int> cluster_bounds(const std::vector<double> &s, int k)
{
    std::vector<int> b{0};
    for (int i = 1; i < k; ++i)
        if (s[i - 1] - s[i] > CLUSTER_TOL * s[0]) b.push_back(i);
    b.push_back(k);
    return b;
}

// W (k x k, row-major, device) = blockdiag of qr+ of the diagonal cluster blocks of P (k x k)
Ten gauge_rotation(const Ten &P, const std::vector<double> &s, int k)
{
    std::vector<int> b = cluster_bounds(s, k);
    for (size_t i = 0; i + 1 < b.size(); ++i)
        if (b[i + 1] - b[i] > 32) fail(-34, "gauge fixing: degenerate cluster of %d values (max 32)", b[i + 1] - b[i]);
    int *bd = (int *)ws_alloc(sizeof(int) * b.size());
    TATRG_CUDA_CHECK(cudaMemcpyAsync(bd, b.data(), sizeof(int) * b.size(), cudaMemcpyHostToDevice, stream()));
    TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));  // b is a local
    Ten W = ws_tensor("ab", {k, k});
    cluster_qr(P.p, k, W.p, k, bd, (int)b.size() - 1);
    return W;
}

// Fork / join of independent chains of small kernels (the three squeezers, the four isometries):
// chain i enqueues on side stream i, which waits for everything enqueued on the main stream so
// far, and bump-allocates from its own slice of the free workspace; join() makes the main stream
// wait for all chains and returns the slices.  Between enter(i) and leave() every launcher of the
// library (they all use stream() and the workspace allocator) works for chain i.  Buffers that must
// outlive the join are allocated on the main stream before the Fork is constructed.
class Fork {
public:
    // main_slice: the main stream keeps a slice of the workspace too and goes on enqueuing while forked
    // (ordering with the chains through side_after_main / main_after_side)
    // chain_bytes > 0 (with main_slice): every chain gets a slice of that size from the top of the free workspace
    // and the main stream keeps the rest
    explicit Fork(int n, bool main_slice = false, size_t chain_bytes = 0)
        : c_(ctx()), n_(n), main_(c_.stream), lo0_(c_.lo), hi0_(c_.hi)
    {
        if (n < 1 || n > Ctx::MAX_CHAINS) fail(-22, "Fork: %d chains", n);
        if (!c_.side_ok) {
            // the chains are latency-bound sequences of small kernels: their CTAs go first whenever an SM frees up
            int prio_lo = 0, prio_hi = 0;
            TATRG_CUDA_CHECK(cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi));
            for (auto &st : c_.side) TATRG_CUDA_CHECK(cudaStreamCreateWithPriority(&st, cudaStreamNonBlocking, prio_hi));
            for (auto &e : c_.join_ev) TATRG_CUDA_CHECK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            for (auto &e : c_.dep_ev) TATRG_CUDA_CHECK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
            TATRG_CUDA_CHECK(cudaEventCreateWithFlags(&c_.fork_ev, cudaEventDisableTiming));
            c_.side_ok = true;
        }
        if (!c_.pinned) TATRG_CUDA_CHECK(cudaMallocHost((void **)&c_.pinned, Ctx::PINNED_BYTES));
        TATRG_CUDA_CHECK(cudaEventRecord(c_.fork_ev, main_));
        size_t slice = ((hi0_ - lo0_) / (n + (main_slice ? 1 : 0))) & ~(size_t)255;
        size_t main_size = slice;
        if (main_slice && chain_bytes > 0) {
            chain_bytes = (chain_bytes + 255) & ~(size_t)255;
            if (chain_bytes * n + (1 << 20) > hi0_ - lo0_) fail(-12, "Fork: workspace too small for %d chains of %zu bytes", n, chain_bytes);
            slice = chain_bytes;
            main_size = (hi0_ - lo0_) - chain_bytes * n;
        }
        for (int i = 0; i < n; ++i) {
            TATRG_CUDA_CHECK(cudaStreamWaitEvent(c_.side[i], c_.fork_ev, 0));
            lo_[i] = lo0_ + (main_slice ? main_size : 0) + i * slice;
            hi_[i] = lo_[i] + slice;
        }
        main_lo_ = main_slice ? lo0_ : hi0_;   // without a slice nothing is allocated on the main stream while forked
        main_hi_ = main_slice ? lo0_ + main_size : hi0_;
        c_.lo = main_lo_;
        c_.hi = main_hi_;
    }
    // chain i continues only after everything enqueued on the main stream so far
    void side_after_main(int i)
    {
        TATRG_CUDA_CHECK(cudaEventRecord(c_.dep_ev[i], main_));
        TATRG_CUDA_CHECK(cudaStreamWaitEvent(c_.side[i], c_.dep_ev[i], 0));
    }
    // the main stream continues only after everything enqueued on chain i so far
    void main_after_side(int i)
    {
        TATRG_CUDA_CHECK(cudaEventRecord(c_.join_ev[i], c_.side[i]));
        TATRG_CUDA_CHECK(cudaStreamWaitEvent(main_, c_.join_ev[i], 0));
    }
    // chain i continues only after everything enqueued on chain j so far
    void side_after_side(int i, int j)
    {
        TATRG_CUDA_CHECK(cudaEventRecord(c_.dep_ev[j], c_.side[j]));
        TATRG_CUDA_CHECK(cudaStreamWaitEvent(c_.side[i], c_.dep_ev[j], 0));
    }
    void enter(int i)
    {
        if (cur_ < 0) main_lo_ = c_.lo;
        cur_ = i;
        c_.stream = c_.side[i];
        c_.lo = lo_[i];
        c_.hi = hi_[i];
    }
    void leave()
    {
        if (cur_ < 0) return;
        lo_[cur_] = c_.lo;
        c_.peak = std::max(c_.peak, c_.lo + (c_.ws_bytes - hi0_));
        cur_ = -1;
        c_.stream = main_;
        c_.lo = main_lo_;
        c_.hi = main_hi_;
    }
    void sync(int i) { TATRG_CUDA_CHECK(cudaStreamSynchronize(c_.side[i])); }
    // page-locked host scratch of chain i (PINNED_BYTES / MAX_CHAINS bytes)
    char *pinned(int i) { return c_.pinned + (size_t)i * (Ctx::PINNED_BYTES / Ctx::MAX_CHAINS); }
    void join()
    {
        leave();
        for (int i = 0; i < n_; ++i) {
            TATRG_CUDA_CHECK(cudaEventRecord(c_.join_ev[i], c_.side[i]));
            TATRG_CUDA_CHECK(cudaStreamWaitEvent(main_, c_.join_ev[i], 0));
        }
        c_.lo = lo0_;
        c_.hi = hi0_;
        joined_ = true;
    }
    ~Fork()
    {
        if (joined_) return;
        c_.stream = main_;   // unwinding after an error: the caller (guarded) drains the device
        c_.lo = lo0_;
        c_.hi = hi0_;
    }

private:
    Ctx &c_;
    int n_;
    cudaStream_t main_;
    size_t lo0_, hi0_;
    size_t lo_[Ctx::MAX_CHAINS], hi_[Ctx::MAX_CHAINS];
    size_t main_lo_ = 0, main_hi_ = 0;
    int cur_ = -1;
    bool joined_ = false;
};

struct StepCfg {
    uint64_t seed;
    int step;
};

// Seeded Gaussian input `which` (rows x cols, row-major): the caller's buffer if one of the right
// size was set, else generated here with the shared generator (sub-seed recipe of DESIGN.md).
// Starts the upload of every host-resident caller-supplied input of this step on the copy stream
// (after everything enqueued so far: the buffers may still be in use by the previous step).
void prefetch_inputs()
{
    Ctx &c = ctx();
    for (int w = 0; w < 9; ++w) c.pre[w] = nullptr;
    c.pre_timed = false;
    c.h2d_ms = 0;
    c.h2d_bytes = 0;
    bool any = false;
    for (int w = 0; w < 9; ++w) any = any || (c.in[w].ptr && !c.in[w].on_device && c.in[w].n > 0);
    if (!any) return;
    if (!c.copy_stream) {
        TATRG_CUDA_CHECK(cudaStreamCreateWithFlags(&c.copy_stream, cudaStreamNonBlocking));
        for (auto &e : c.pre_ev) TATRG_CUDA_CHECK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        TATRG_CUDA_CHECK(cudaEventCreate(&c.pre_t0));
        TATRG_CUDA_CHECK(cudaEventCreate(&c.pre_t1));
    }
    TATRG_CUDA_CHECK(cudaEventRecord(c.pre_ev[0], c.stream));
    TATRG_CUDA_CHECK(cudaStreamWaitEvent(c.copy_stream, c.pre_ev[0], 0));
    TATRG_CUDA_CHECK(cudaEventRecord(c.pre_t0, c.copy_stream));
    for (int w = 0; w < 9; ++w) {
        const Input &in = c.in[w];
        if (!in.ptr || in.on_device || in.n == 0) continue;
        c.pre[w] = ws_doubles((long long)in.n);
        c.pre_n[w] = in.n;
        TATRG_CUDA_CHECK(cudaMemcpyAsync(c.pre[w], in.ptr, sizeof(double) * in.n, cudaMemcpyHostToDevice, c.copy_stream));
        TATRG_CUDA_CHECK(cudaEventRecord(c.pre_ev[w], c.copy_stream));
        c.h2d_bytes += sizeof(double) * in.n;
    }
    TATRG_CUDA_CHECK(cudaEventRecord(c.pre_t1, c.copy_stream));
    c.pre_timed = true;
}

Ten get_input(int which, long long rows, long long cols, const StepCfg &cfg, const char *names2)
{
    Ctx &c = ctx();
    long long n = rows * cols;
    Ten t;
    Input &in = c.in[which];
    if (in.ptr && in.n != (size_t)n)
        fail(-22, "input %d set with tatrg_set_sketch has %zu doubles, this step needs %lld x %lld = %lld (tatrg_sketch_shape)",
             which, in.n, rows, cols, n);
    if (in.ptr) {
        if (!in.on_device && c.pre[which] && c.pre_n[which] == (size_t)n) {
            TATRG_CUDA_CHECK(cudaStreamWaitEvent(stream(), c.pre_ev[which], 0));
            return Ten::make(c.pre[which], names2, {rows, cols});
        }
        if (in.on_device) {
            t = Ten::make(const_cast<double *>(in.ptr), names2, {rows, cols});
        } else {
            t = ws_tensor(names2, {rows, cols});
            h2d(t.p, in.ptr, n);
        }
        return t;
    }
    const uint64_t st = (which >= 5) ? 0 : (uint64_t)cfg.step;   // gauge references are step independent
    t = ws_tensor(names2, {rows, cols});
    device_fill_gauss(t.p, (unsigned long long)n, si_subseed(cfg.seed, st, (uint64_t)which));
    return t;
}

void stage_mark(int i)
{
    Ctx &c = ctx();
    if (!c.ev_ok) {
        for (auto &e : c.ev) TATRG_CUDA_CHECK(cudaEventCreate(&e));
        c.ev_ok = true;
    }
    TATRG_CUDA_CHECK(cudaEventRecord(c.ev[i], c.stream));
    c.cur_stage = i < ST_COUNT ? i : ST_COUNT - 1;
    c.host_t[i] = std::chrono::duration<double>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

// Symmetric PSD eigenproblem of the n x n matrix S (overwritten): on exit the rows of Vt
// (row-major n x n) are the eigenvectors, lam (device, n) descending; returns lam on the host.
std::vector<double> sym_eig(double *S, int n, double *Vt, double *lam)
{
    if (n <= 64) {
        eig_small(S, n, Vt, lam);
        return d2h(lam, n);
    }
    symmetrize(S, n);
    jacobi_svd(S, n, n, Vt, lam, 1, 0, 0, 0);
    return d2h(lam, n);
}

// ---------------------------------------------------------------------------------------
// RSVD by subspace iteration (reading O9).  apply / apply_t map a
// (cols x z) block to (rows x z) and back.  Returns Q u[:, :k], s, Q_B v[:, :k].
struct RsvdOut {
    int k;
    std::vector<double> s_full;
    double *s_dev;
};

template <class F1, class F2>
RsvdOut rsvd(F1 apply, F2 apply_t, const Ten &omega, long long rows, long long cols, int ell, int q, int keep,
             double *left, double *right)
{
    double *Rtmp = ws_doubles((long long)ell * ell);
    Ten Yb = ws_tensor("rz", {rows, ell});
    Ten Yt = ws_tensor("rz", {cols, ell});
    double *Rb = ws_doubles((long long)ell * ell);
    // Fast route for tall blocks: asynchronous Cholesky-QR -- between iterations one shifted pass (only
    // the span is carried on), two passes for the two blocks that define the result (Q and Q_B); the
    // flags / condition estimates are read once at the end, and if they are bad everything is redone
    // with the robust synchronous QR.
    bool done = false;
    if (!(ctx().routes & ROUTE_HOUSEHOLDER_QR) && ell <= 256 && rows >= 16LL * ell && cols >= 16LL * ell && rows >= 512 && cols >= 512) {
        int *flag = (int *)ws_alloc(sizeof(int));
        double *ratio = ws_doubles(4);
        TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(int), stream()));
        const double it_shift = 1e-13;
        apply(omega.p, Yb.p);
        cholqr_async(Yb.p, rows, ell, q == 0 ? 2 : 1, q == 0 ? 0.0 : it_shift, flag, q == 0 ? ratio : nullptr, nullptr);
        for (int it = 0; it < q; ++it) {
            const bool last = it == q - 1;
            apply_t(Yb.p, Yt.p);
            cholqr_async(Yt.p, cols, ell, 1, it_shift, flag, nullptr, nullptr);
            apply(Yt.p, Yb.p);
            cholqr_async(Yb.p, rows, ell, last ? 2 : 1, last ? 0.0 : it_shift, flag, last ? ratio : nullptr, nullptr);
        }
        apply_t(Yb.p, Yt.p);             // B^T = Op^T Q
        cholqr_async(Yt.p, cols, ell, 2, 0.0, flag, ratio + 2, Rb);
        struct {
            int f;
            double r[4];
        } h;
        trace_mark("rsvd: subspace iteration");
        TATRG_CUDA_CHECK(cudaMemcpyAsync(&h.f, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
        TATRG_CUDA_CHECK(cudaMemcpyAsync(h.r, ratio, 4 * sizeof(double), cudaMemcpyDeviceToHost, stream()));
        TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
        done = h.f == 0 && h.r[0] > 1e-5 * h.r[1] && h.r[2] > 1e-5 * h.r[3];
    }
    if (!done) {
        apply(omega.p, Yb.p);
        tsqr(Yb.p, rows, ell, Rtmp);
        for (int it = 0; it < q; ++it) {
            apply_t(Yb.p, Yt.p);
            tsqr(Yt.p, cols, ell, Rtmp);
            apply(Yt.p, Yb.p);
            tsqr(Yb.p, rows, ell, Rtmp);
        }
        apply_t(Yb.p, Yt.p);             // B^T = Op^T Q
        tsqr(Yt.p, cols, ell, Rb);       // B^T = Q_B R_B; the row-major R_B buffer is R_B^T column-major
    }
    double *V = ws_doubles((long long)ell * ell);
    double *s = ws_doubles(ell);
    jacobi_svd(Rb, ell, ell, V, s, 1, 0, 0, 0);   // R_B^T V = U diag(s)
    trace_mark("rsvd: svd of the core");
    RsvdOut out;
    out.s_full = d2h(s, ell);
    out.s_dev = s;
    out.k = num_rank(out.s_full, keep);
    const int k = out.k;
    if (k < 1) fail(-34, "rsvd: operator is numerically zero");
    scale_leg(Rb, (long long)k * ell, ell, k, s, 1);   // columns of U
    Ten U = Ten::make(Rb, "gz", {ell, ell});           // [g][z] = U[z, g]
    Ten Vv = Ten::make(V, "gz", {ell, ell});
    Ten Uk = U, Vk = Vv;
    Uk.legs[0].n = k;
    Vk.legs[0].n = k;
    contract(Yb, Uk, Ten::make(left, "rg", {rows, k}));
    contract(Yt, Vk, Ten::make(right, "rg", {cols, k}));
    return out;
}

// Seeded Gaussian start block of an iterative solver (not a method input: the iteration is run to
// convergence, so the result does not depend on it beyond rounding).
Ten solver_start_block(long long rows, long long cols, int tag, const char *names2)
{
    Ten t = ws_tensor(names2, {rows, cols});
    device_fill_gauss(t.p, (unsigned long long)(rows * cols), si_subseed(0x7a7e6ULL, 0, 100 + (uint64_t)tag));
    return t;
}

// Squeezer of one direction without a dense eigensolver: any factors
// G^L = R1^T R1, G^R = R2 R2^T give the same M = R2 V s^-1/2, N = s^-1/2 U^T R1 (reading O6), so
// R1 = L_L^T, R2 = L_R from two Cholesky factorisations (tensor-pipe GEMMs), and only the top
// chi singular triplets of F = R1 R2 are needed: subspace iteration with a block of width b >
// chi, iteration count from the measured decay s_b / s_chi so that the neglected part is below
// 1e-13.  Returns false (nothing written) when a Gram matrix is not numerically positive definite
// or fewer than chi significant triplets exist -- the caller then uses the dense path.
// It is written as a chain in phases (enqueue only; the host reads the page-locked read-back
// after synchronising the chain's stream), so that the three squeezers of a step run concurrently
// on three streams (Fork).
struct SqChain {
    int b = 64;            // block width of the subspace iteration (> chi): 64, or 128 for chi >= 64
    struct Back {          // page-locked read-back
        int flag;
        int pad;
        double ratio[4];
        double s[128];
    };
    Ten GLm, GRm;
    int N2 = 0, chi = 0, mu = 0;
    bool active = false, ok = false;
    Ten LL, LR, F;
    int *flag = nullptr;
    double *ratio = nullptr, *Q = nullptr, *Qt = nullptr, *Rb = nullptr, *V = nullptr, *sv = nullptr;
    Back *back = nullptr;
    std::vector<double> sh;
    int more = 0, k = 0, hist = 0, iters_done = 0, planned = 0;
    int grid = 0;          // > 0: the iteration runs as one launch of that many CTAs (sq_iter.cu), b = 64 only
    const double *start = nullptr;
    double *Ft = nullptr;  // F^T: both products of the fused iteration read rows
    std::vector<unsigned char> steps;
    double gap = INFINITY;
    Ten Mr, Nr;
    static constexpr double it_shift = 1e-13;

    void mulF(const double *w, double *out)    // F w
    {
        contract(F, Ten::make(const_cast<double *>(w), "jz", {N2, b}), Ten::make(out, "iz", {N2, b}));
    }
    void mulFt(const double *w, double *out)   // F^T w
    {
        contract(F, Ten::make(const_cast<double *>(w), "iz", {N2, b}), Ten::make(out, "jz", {N2, b}));
    }
    // Ritz step on the current Q (two Cholesky-QR passes have just been applied to it):
    // B^T = F^T Q = Q_B R_B, R_B^T V = U diag(s); read-back of flag, condition estimates, s
    // estimate: only the singular values are wanted, to two or three digits (iteration count)
    void enqueue_ritz(bool estimate = false)
    {
        if (grid > 0) {
            steps.push_back(SQ_TRANS | SQ_TWO_PASSES | (2 << SQ_RATIO_SHIFT) | SQ_WANT_R);
            launch_fused();
        } else {
            mulFt(Q, Qt);
            cholqr_async(Qt, N2, b, 2, 0.0, flag, ratio + 2, Rb);
        }
        if (b <= 64)
            svd_small_async(Rb, b, b, V, sv, flag, estimate ? 1e-4 : 0.0);
        else
            jacobi_svd(Rb, b, b, V, sv, 1, 0, 0, 0);       // multi-launch Jacobi (synchronises this chain)
        TATRG_CUDA_CHECK(cudaMemcpyAsync(&back->flag, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
        TATRG_CUDA_CHECK(cudaMemcpyAsync(back->ratio, ratio, 4 * sizeof(double), cudaMemcpyDeviceToHost, stream()));
        TATRG_CUDA_CHECK(cudaMemcpyAsync(back->s, sv, b * sizeof(double), cudaMemcpyDeviceToHost, stream()));
    }
    // the half steps collected in `steps` as one launch (sq_iter.cu)
    void launch_fused()
    {
        SqIterParams p{};
        p.F = F.p;
        p.Ft = Ft;
        p.start = start;
        p.buf[0] = Q;
        p.buf[1] = Qt;
        p.Rout = Rb;
        p.ratio = ratio;
        p.flag = flag;
        p.shift = it_shift;
        p.N2 = N2;
        p.nsteps = (int)steps.size();
        if (p.nsteps > SQ_MAXSTEPS) fail(-22, "squeezer: %d half steps in one launch", p.nsteps);
        std::copy(steps.begin(), steps.end(), p.steps);
        sq_iter_launch(p, grid, ws_doubles((long long)sq_iter_scratch_doubles(sq_iter_grid(N2, grid))));
        steps.clear();
    }
    // after the chain's stream has been synchronised
    bool read_back()
    {
        sh.assign(back->s, back->s + b);
        // a failed factorisation / Jacobi, or a block too ill conditioned for two Cholesky-QR passes
        return back->flag == 0 && back->ratio[0] > 1e-5 * back->ratio[1] && back->ratio[2] > 1e-5 * back->ratio[3];
    }
    // The block was too ill conditioned for two Cholesky-QR passes while no factorisation failed (s_b / s_1 below
    // ~1e-5: at the ordered fixed point the spectrum of F decays that fast): the same Ritz step with Householder
    // TSQR, which needs no condition.  Q still spans the right subspace.  Synchronous on the chain's stream.
    bool too_ill_conditioned() const
    {
        return back->flag == 0 && !(back->ratio[0] > 1e-5 * back->ratio[1] && back->ratio[2] > 1e-5 * back->ratio[3]) &&
               back->ratio[0] > 0.0 && back->ratio[2] > 0.0;
    }
    void ritz_robust()
    {
        double *Rtmp = ws_doubles((long long)b * b);
        tsqr(Q, N2, b, Rtmp);
        mulFt(Q, Qt);
        tsqr(Qt, N2, b, Rb);
        if (b <= 64)
            svd_small_async(Rb, b, b, V, sv, flag);
        else
            jacobi_svd(Rb, b, b, V, sv, 1, 0, 0, 0);
        TATRG_CUDA_CHECK(cudaMemcpyAsync(&back->flag, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
        TATRG_CUDA_CHECK(cudaMemcpyAsync(back->s, sv, b * sizeof(double), cudaMemcpyDeviceToHost, stream()));
        TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
        for (int i = 0; i < 4; ++i) back->ratio[i] = 1.0;   // orthonormal by construction
    }
    // on the main stream, before any fork: the buffers of the two Cholesky factors
    void prep()
    {
        LL = ws_tensor("ki", {N2, N2});
        LR = ws_tensor("kj", {N2, N2});
        d2d(LL.p, GLm.p, (long long)N2 * N2);
        d2d(LR.p, GRm.p, (long long)N2 * N2);
        flag = (int *)ws_alloc(sizeof(int));
        TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(int), stream()));
    }
    // the two factorisations G^L + delta = L_L L_L^T, G^R + delta = L_R L_R^T: independent chains
    void factor(int which)
    {
        const double shift = 3e-14;
        cholesky_lower_async(which == 0 ? LL.p : LR.p, N2, shift, nullptr, flag);
    }
    // hist > 0: the iteration count the same squeezer needed four steps ago (same direction): that many
    // iterations are done at once and the Ritz step that follows is the final one if the decay it measures
    // confirms the count (plan); else two iterations and a rough Ritz step to measure the decay first
    void phaseA(char *pinned)
    {
        back = reinterpret_cast<Back *>(pinned);
        F = ws_tensor("ij", {N2, N2});
        contract(LL, LR, F);                               // F = L_L^T L_R
        if (grid > 0) {
            Ft = ws_doubles((long long)N2 * N2);
            transpose_small(F.p, Ft, N2, N2);
        }
        ratio = ws_doubles(4);
        Ten om = solver_start_block(N2, b, mu, "jz");
        Q = ws_doubles((long long)N2 * b);
        Qt = ws_doubles((long long)N2 * b);
        Rb = ws_doubles((long long)b * b);
        V = ws_doubles((long long)b * b);
        sv = ws_doubles(b);
        // Subspace iteration Q <- orth(F orth(F^T Q)).  Between iterations one (shifted) Cholesky-QR
        // pass is enough: only the span is carried on; the blocks that enter a Ritz step get two.
        // (fused: a few iterations more than the last count cost less than a second Ritz step would)
        iters_done = hist > 0 ? hist + (grid > 0 ? 2 : 0) : 2;
        if (grid > 0) {
            start = om.p;
            steps.clear();
            steps.push_back(SQ_FROM_START);
            for (int it = 0; it < iters_done; ++it) {
                steps.push_back(SQ_TRANS);
                steps.push_back(it == iters_done - 1 ? (SQ_TWO_PASSES | (1 << SQ_RATIO_SHIFT)) : 0);
            }
        } else {
            mulF(om.p, Q);
            cholqr_async(Q, N2, b, 1, it_shift, flag, nullptr, nullptr);
            for (int it = 0; it < iters_done; ++it) {
                const bool last = it == iters_done - 1;
                mulFt(Q, Qt);
                cholqr_async(Qt, N2, b, 1, it_shift, flag, nullptr, nullptr);
                mulF(Qt, Q);
                cholqr_async(Q, N2, b, last ? 2 : 1, last ? 0.0 : it_shift, flag, last ? ratio : nullptr, nullptr);
            }
        }
        enqueue_ritz(hist <= 0);
    }
    // iteration count from the measured decay rho = s_b / s_chi: rho^(2p+1) < 1e-13
    bool plan()
    {
        if (getenv("TATRG_TRACE"))
            fprintf(stderr, "tatrg-trace squeezer mu %d read-back: flag %d ratios %.2e/%.2e %.2e/%.2e s_1 %.3e s_chi %.3e s_b %.3e\n", mu, back->flag,
                    back->ratio[0], back->ratio[1], back->ratio[2], back->ratio[3], back->s[0], back->s[chi - 1], back->s[b - 1]);
        if (!read_back()) return false;
        if (!(sh[chi - 1] > 1e-6 * sh[0])) return false;
        const double rho = sh[b - 1] / sh[chi - 1];
        const int need = (rho > 0.0 && rho < 1.0) ? (int)ceil((13.0 / -log10(rho) - 1.0) / 2.0) : 2;
        if (need + 1 > 80) return false;                   // decay too slow for this block width: dense route
        planned = need + 1;
        if (hist > 0 && iters_done >= planned)
            more = 0;                                      // the Ritz step just read back is the final one
        else
            more = std::max(1, planned - iters_done);
        return true;
    }
    void phaseB()
    {
        for (int it = 0; it < more; ++it) {
            const bool last = it == more - 1;
            if (grid > 0) {
                steps.push_back(last ? (SQ_TWO_PASSES | (1 << SQ_RATIO_SHIFT)) : 0);
                if (!last) steps.push_back(SQ_TRANS);
                continue;
            }
            mulF(Qt, Q);                                   // Qt = orth(F^T Q) from the Ritz step / the loop
            cholqr_async(Q, N2, b, last ? 2 : 1, last ? 0.0 : it_shift, flag, last ? ratio : nullptr, nullptr);
            if (!last) {
                mulFt(Q, Qt);
                cholqr_async(Qt, N2, b, 1, it_shift, flag, nullptr, nullptr);
            }
        }
        enqueue_ritz();
    }
    // M = L_R V s^-1/2, N = s^-1/2 U^T L_L^T from the converged triplets
    bool phaseC()
    {
        if (!read_back()) return false;
        k = num_rank(sh, chi);
        if (k < chi) return false;
        gap = rel_gap(sh, k);
        scale_leg(Rb, (long long)k * b, b, k, sv, 1);      // columns of U
        Ten Uk = Ten::make(Rb, "kz", {b, b}), Vk = Ten::make(V, "kz", {b, b});
        Uk.legs[0].n = k;
        Vk.legs[0].n = k;
        Ten left = ws_tensor("ik", {N2, k}), right = ws_tensor("jk", {N2, k});
        contract(Ten::make(Q, "iz", {N2, b}), Uk, left);
        contract(Ten::make(Qt, "jz", {N2, b}), Vk, right);
        Mr = ws_tensor("nk", {N2, k});
        Nr = ws_tensor("kn", {k, N2});
        contract(left, LL.as("ni"), Nr);
        contract(LR.as("nj"), right, Mr);
        scale_leg(Nr.p, Nr.size(), N2, k, sv, 3);
        scale_leg(Mr.p, Mr.size(), 1, k, sv, 3);
        return true;
    }
};

// Orthonormal basis of the column space of the matricisation T2[(pqt); (c,b)] of T[c,p,q,t,b]
// (nT x nk, nk = n0 * a), by two Cholesky-QR passes with explicit triangular inverses so that all
// O(nT nk^2) work is three full-size tensor-GEMMs:
//   G1 = T2^T T2 = L1 L1^T,  Q1 = T2 L1^-T,  G2 = Q1^T Q1 = L2 L2^T,  Q = Q1 L2^-T (kept implicit),
//   T2 = Q R,  R = L2^T L1^T.
// Used by the bond swap (reduced operator, below).  Returns false -- nothing the caller keeps has
// been written -- when T2 is rank deficient or too ill conditioned for two passes (|G2 - I| > 0.05).
struct RedBasis {
    Ten Q1;      // [p,q,t,k]
    Ten R;       // [k,c,b]
    Ten L2inv;   // [k,l] lower triangular: Q = Q1 L2inv^T
};

// One tensor's factorisation in three pieces, so that the two Cholesky factorisations (latency-bound,
// a few CTAs) run on side streams under the machine-filling GEMMs of the main stream.
struct OrthoChain {
    Ten T;
    RedBasis o;
    long long nk = 0;
    Ten G1, G1copy, G2, L1inv;
    int *flag = nullptr;
    double *dev = nullptr;
    struct Back {
        int flag;
        int pad;
        double err;
    } *back = nullptr;
    double err = INFINITY;
    bool transposed_r = false;

    void alloc(const Ten &T_, char *pinned)   // on the main stream, before the fork
    {
        T = T_;
        back = reinterpret_cast<Back *>(pinned);
        const long long n0 = T.legs[0].n, n1 = T.legs[1].n, n2 = T.legs[2].n, n3 = T.legs[3].n, a = T.legs[4].n;
        nk = n0 * a;
        o.Q1 = ws_tensor("pqtk", {n1, n2, n3, nk});
        o.R = ws_tensor("kcb", {nk, n0, a});
        o.L2inv = ws_tensor("kl", {nk, nk});
        G1 = ws_tensor("cbde", {n0, a, n0, a});
        G1copy = ws_tensor("cbde", {n0, a, n0, a});
        G2 = ws_tensor("kl", {nk, nk});
        L1inv = ws_tensor("kcb", {nk, n0, a});
        flag = (int *)ws_alloc(sizeof(int));
        dev = ws_doubles(1);
        TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(int), stream()));
    }
    void gram1()                                                                                 // main
    {
        contract(T.as("cpqtb"), T.as("dpqte"), G1, 1.0, false, true);
        d2d(G1copy.p, G1.p, nk * nk);
    }
    void factor1() { cholesky_lower_async(G1.p, (int)nk, 0.0, L1inv.p, flag); }                 // side
    // When T2 is numerically rank deficient (the ordered fixed point: cond(T2) beyond ~3e7) the plain
    // factorisation breaks down: it is redone with a shift of 1e-13 max diag (above the rounding noise of
    // G1).  T2 = Q1 L1^T holds by construction whatever the shift, which only decides how far Q1 is from
    // orthonormal -- the extra pass takes care of that.
    bool redo_shifted()
    {
        d2d(G1.p, G1copy.p, nk * nk);
        TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(int), stream()));   // the failed attempt raised it
        if (!cholesky_lower(G1.p, (int)nk, 1e-13, L1inv.p)) return false;
        contract(T.as("cpqtb"), L1inv, o.Q1, 1.0, false, false, true);
        contract(o.Q1.as("pqtk"), o.Q1.as("pqtl"), G2, 1.0, false, true);
        max_dev_identity(G2.p, (int)nk, dev);
        err = d2h(dev, 1)[0];
        if (getenv("TATRG_TRACE")) fprintf(stderr, "tatrg-trace ortho: shifted first pass, |G2 - I| = %.3e\n", err);
        return std::isfinite(err);
    }
    void basis()                                                                                 // main
    {
        // Q1 = T2 L1^-T: L1inv[k][(c,b)] = 0 for (c,b) > k, the k tiles of zeros are skipped (tri_b)
        contract(T.as("cpqtb"), L1inv, o.Q1, 1.0, false, false, true);
        contract(o.Q1.as("pqtk"), o.Q1.as("pqtl"), G2, 1.0, false, true);
        max_dev_identity(G2.p, (int)nk, dev);
        TATRG_CUDA_CHECK(cudaMemcpyAsync(&back->flag, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
        TATRG_CUDA_CHECK(cudaMemcpyAsync(&back->err, dev, sizeof(double), cudaMemcpyDeviceToHost, stream()));
    }
    bool usable()   // after the main stream has been synchronised
    {
        err = back->err;
        if (getenv("TATRG_TRACE")) fprintf(stderr, "tatrg-trace ortho: nk %lld |G2 - I| = %.3e flag %d\n", nk, err, back->flag);
        return back->flag == 0 && std::isfinite(err);
    }
    bool failed_factor() const { return back->flag != 0 || !std::isfinite(back->err); }
    // One more explicit pass when Q1 is too far from orthonormal for the implicit last pass (|G2 - I| >= 0.05:
    // T2 ill conditioned, the shifted first pass left cond(Q1) up to ~1e6): G2 = L2 L2^T, Q2 = Q1 L2^-T
    // written over Q1, G3 = Q2^T Q2; then the implicit pass on G3.  R = L3^T L2^T L1^T.
    bool extra_pass()
    {
        Ten L2inv = ws_tensor("kl", {nk, nk});
        if (!cholesky_lower(G2.p, (int)nk, 0.0, L2inv.p)) return false;
        // L21[i][(c,b)] = sum_k L2[k][i] L1[(c,b)][k]  (= (L1 L2)^T: the triangular factor so far)
        Ten L21 = ws_tensor("ij", {nk, nk});
        contract(G2.as("ki"), Ten::make(G1.p, "jk", {nk, nk}), L21);
        d2d(G1.p, L21.p, nk * nk);                      // G1 now holds (L1 L2)^T row-major, used as "L1^T" below
        {
            size_t mk = ws_mark();
            Ten Q2 = ws_tensor("pqtl", {o.Q1.legs[0].n, o.Q1.legs[1].n, o.Q1.legs[2].n, nk});
            contract(o.Q1.as("pqtk"), L2inv.as("lk"), Q2, 1.0, false, false, true);
            d2d(o.Q1.p, Q2.p, Q2.size());
            ws_release(mk);
        }
        contract(o.Q1.as("pqtk"), o.Q1.as("pqtl"), G2, 1.0, false, true);
        max_dev_identity(G2.p, (int)nk, dev);
        err = d2h(dev, 1)[0];
        if (getenv("TATRG_TRACE")) fprintf(stderr, "tatrg-trace ortho: extra pass, |G3 - I| = %.3e\n", err);
        transposed_r = true;
        return std::isfinite(err) && err < 0.05;
    }
    // the last factorisation, G2 (or G3) = L L^T: asynchronous, so that the two tensors' run side by side
    void phase2_factor()
    {
        if (err < 1e-8)
            near_identity_chol(G2.p, (int)nk, o.L2inv.p);
        else
            cholesky_lower_async(G2.p, (int)nk, 0.0, o.L2inv.p, flag);
        TATRG_CUDA_CHECK(cudaMemcpyAsync(&back->flag, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
    }
    bool phase2()   // after the factorisations have been synchronised
    {
        if (back->flag != 0) return false;
        if (transposed_r)   // after an extra pass G1 holds the accumulated factor transposed: R[i][j] = sum_k L3[k][i] G1[k][j]
            contract(G2.as("ki"), Ten::make(G1.p, "kj", {nk, nk}), Ten::make(o.R.p, "ij", {nk, nk}));
        else                // R[i][(c,b)] = sum_k L2[k][i] L1[(c,b)][k]
            contract(G2.as("ki"), Ten::make(G1.p, "jk", {nk, nk}), Ten::make(o.R.p, "ij", {nk, nk}));
        return true;
    }
};

// Both bases of the reduced bond swap; false when either matricisation is rank deficient or too
// ill conditioned for two Cholesky-QR passes (|G2 - I| > 0.05).
// Main stream: G1_A, G1_D, Q1_A, G2_A, Q1_D, G2_D; side streams: chol(G1_A) under G1_D, chol(G1_D) under Q1_A.
// during_last (optional): main-stream work that needs only the first factor Q1 of D's basis (the projection of the
// sketch) is enqueued beside the last, latency-bound factorisations of the two bases.
bool ortho_factor_pair(const Ten &A, const Ten &D, RedBasis &bA, RedBasis &bD,
                       const std::function<void(const RedBasis &)> &during_last = nullptr)
{
    Ctx &c = ctx();
    if (!c.pinned) TATRG_CUDA_CHECK(cudaMallocHost((void **)&c.pinned, Ctx::PINNED_BYTES));
    OrthoChain ch[2];
    ch[0].alloc(A, c.pinned);
    ch[1].alloc(D, c.pinned + 64);
    if (ch[0].nk > 0x7fffffff) return false;
    {
        Fork fk(2, true);
        for (int i = 0; i < 2; ++i) {
            ch[i].gram1();
            fk.side_after_main(i);
            fk.enter(i);
            ch[i].factor1();
            fk.leave();
        }
        for (int i = 0; i < 2; ++i) {
            fk.main_after_side(i);
            ch[i].basis();
        }
        fk.join();
    }
    TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
    bool ok = true;
    for (int i = 0; i < 2 && ok; ++i) ok = ch[i].usable() || (ch[i].failed_factor() && ch[i].redo_shifted());
    for (int i = 0; i < 2 && ok; ++i)
        if (ch[i].err >= 0.05) ok = ch[i].extra_pass();
    bool during_done = false;
    if (ok) {
        const size_t chain_bytes = std::max<size_t>((size_t)32 << 20, (size_t)(4 * ch[0].nk * ch[0].nk * 8));
        const bool beside = during_last && c.hi - c.lo > 2 * chain_bytes + ((size_t)64 << 20);
        Fork fk(2, beside, beside ? chain_bytes : 0);
        if (beside) c.chol_ctas = CHAIN_SM_RESERVE / 2;
        for (int i = 0; i < 2; ++i) {
            fk.enter(i);
            ch[i].phase2_factor();
            fk.leave();
        }
        c.chol_ctas = 16;
        if (beside) {
            c.sm_reserve = CHAIN_SM_RESERVE;
            during_last(ch[1].o);
            c.sm_reserve = 0;
            during_done = true;
        }
        for (int i = 0; i < 2; ++i) fk.sync(i);
        fk.join();
    }
    for (int i = 0; i < 2 && ok; ++i) ok = ch[i].phase2();
    if (ok && during_last && !during_done) during_last(ch[1].o);
    bA = ch[0].o;
    bD = ch[1].o;
    return ok;
}

}  // namespace

// =======================================================================================
void do_init(double beta, double h)
{
    Ctx &c = ctx();
    if (!(beta > 0) || !std::isfinite(beta) || !std::isfinite(h)) fail(-22, "init_ising_tensor: beta must be finite and > 0, h finite");
    if (!c.ws) fail(-1, "init_ising_tensor: no workspace set");
    // PAPER.md:128-137 Eqs. 16-17, readings G1 (square roots) and G2 (field weight)
    double W[2][2];
    const double sgn[2] = {1.0, -1.0};
    for (int a = 0; a < 2; ++a) {
        W[a][0] = sqrt(cosh(beta));
        W[a][1] = sgn[a] * sqrt(sinh(beta));
    }
    std::vector<double> phi(32), psi(32);
    for (int i = 0; i < 16; ++i)
        for (int a = 0; a < 2; ++a) {
            double v = 1.0;
            for (int mu = 0; mu < 4; ++mu) v *= W[a][(i >> (3 - mu)) & 1];
            phi[i * 2 + a] = v;
            psi[i * 2 + a] = v * exp(beta * h * sgn[a]);
        }
    c.lo = 0;
    c.hi = c.ws_bytes;
    c.state_low = true;
    c.state_bytes = 512;
    if (c.ws_bytes < 4096) fail(-12, "workspace too small");
    c.phi = (double *)c.ws;
    c.psi = c.phi + 32;
    h2d(c.phi, phi.data(), 32);
    h2d(c.psi, psi.data(), 32);
    TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
    for (int i = 0; i < 4; ++i) c.dims[i] = 2;
    c.bond = 2;
    c.step = 0;
    c.log_acc = 0.0;
    c.beta = beta;
    c.h = h;
    // normalise (reading O8): c_0 = |Phi||Psi|
    c.lo = c.state_bytes;
    double *ss = ws_doubles(2);
    sumsq(c.phi, 32, ss);
    sumsq(c.psi, 32, ss + 1);
    scale_by_rsqrt(c.phi, 32, ss);
    scale_by_rsqrt(c.psi, 32, ss + 1);
    std::vector<double> v = d2h(ss, 2);
    c.log_acc = 0.5 * (log(v[0]) + log(v[1]));
    for (auto &s : c.spec) s.clear();
    for (int i = 0; i < 4; ++i) {
        c.iso_pending[i] = false;
        c.iso_H[i].clear();
        for (int mu = 0; mu < 3; ++mu) c.sq_hist[i][mu] = 0;
    }
    for (auto &i : c.in) i = Input();
    c.inited = true;
}

double do_log_z()
{
    Ctx &c = ctx();
    if (!c.inited) return NAN;
    c.lo = c.state_low ? c.state_bytes : 0;
    c.hi = c.state_low ? c.ws_bytes : c.ws_bytes - c.state_bytes;
    long long n = (long long)c.dims[0] * c.dims[1] * c.dims[2] * c.dims[3] * c.bond;
    double *o = ws_doubles(1);
    dot(c.phi, c.psi, n, o);
    double t = d2h(o, 1)[0];
    if (!(t > 0)) return NAN;
    return c.log_acc + ldexp(1.0, -c.step) * log(t);
}

// X^(m) = (Tr A)^2 / Tr(A^2), A_kl = sum T_{..k..;..l..}
double do_order_parameter(int leg)
{
    Ctx &c = ctx();
    if (!c.inited || leg < 1 || leg > 4) return NAN;
    c.lo = c.state_low ? c.state_bytes : 0;
    c.hi = c.state_low ? c.ws_bytes : c.ws_bytes - c.state_bytes;
    const char *names[4] = {"kuvwg", "ukvwg", "uvkwg", "uvwkg"};
    const char *namel[4] = {"luvwg", "ulvwg", "uvlwg", "uvwlg"};
    Ten phi = Ten::make(c.phi, names[leg - 1], {c.dims[0], c.dims[1], c.dims[2], c.dims[3], c.bond});
    Ten psi = Ten::make(c.psi, namel[leg - 1], {c.dims[0], c.dims[1], c.dims[2], c.dims[3], c.bond});
    int n = c.dims[leg - 1];
    Ten Am = ws_tensor("kl", {n, n});
    contract(phi, psi, Am);
    Ten A2 = ws_tensor("km", {n, n});
    contract(Am, Am.as("lm"), A2);
    std::vector<double> a = d2h(Am.p, (long long)n * n), a2 = d2h(A2.p, (long long)n * n);
    double tr = 0, tr2 = 0;
    for (int i = 0; i < n; ++i) {
        tr += a[(size_t)i * n + i];
        tr2 += a2[(size_t)i * n + i];
    }
    return tr * tr / tr2;
}

// Wide isometries (r chi > 64) leave their Ritz step out of the path (see do_coarse_grain): the spectra
// S^A..S^D and, for tatrg_get_isometry, the Ritz vectors U = Q V are computed here, when asked for, from
// the kk x kk Ritz matrices the step kept.
void resolve_iso_spectra()
{
    Ctx &c = ctx();
    bool any = false;
    for (int i = 0; i < 4; ++i) any = any || c.iso_pending[i];
    if (!any || !c.inited) return;
    c.lo = c.state_low ? c.state_bytes : 0;
    c.hi = c.state_low ? c.ws_bytes : c.ws_bytes - c.state_bytes;
    for (int i = 0; i < 4; ++i) {
        if (!c.iso_pending[i]) continue;
        const int kk = (int)llround(sqrt((double)c.iso_H[i].size()));
        size_t mk = ws_mark();
        Ten Hm = ws_tensor("zy", {kk, kk}), Vt = ws_tensor("kz", {kk, kk});
        double *lam = ws_doubles(kk);
        h2d(Hm.p, c.iso_H[i].data(), (long long)kk * kk);
        std::vector<double> lh = sym_eig(Hm.p, kk, Vt.p, lam);
        c.spec[2 + i].resize(kk);
        for (int j = 0; j < kk; ++j) c.spec[2 + i][j] = sqrt(std::max(lh[j], 0.0));
        if (!c.iso[i].empty() && c.iso_cols == kk) {   // kept isometry: Q -> Q V
            const long long n12 = c.iso_rows;
            Ten Qd = ws_tensor("rz", {n12, kk}), Ud = ws_tensor("rk", {n12, kk});
            h2d(Qd.p, c.iso[i].data(), n12 * kk);
            contract(Qd, Vt, Ud);
            c.iso[i] = d2h(Ud.p, n12 * kk);
        }
        ws_release(mk);
        c.iso_pending[i] = false;
        c.iso_H[i].clear();
    }
}

// =======================================================================================
void do_coarse_grain(int direction, int chi, int r, int q, uint64_t seed, int mode)
{
    Ctx &c = ctx();
    if (!c.inited) fail(-1, "coarse_grain: call init_ising_tensor first");
    if (direction < 1 || direction > 4 || chi < 1 || r < 1 || q < 0) fail(-22, "coarse_grain: bad arguments");
    if ((long long)r * chi > 256 || chi > 64) fail(-22, "coarse_grain: r*chi = %d > 256 (or chi > 64) not supported", r * chi);
    StepCfg cfg{seed, c.step};
    c.prof_rec.clear();

    // ---- frames (reading G8)
    int perm[4];
    perm[0] = direction - 1;
    for (int i = 0, j = 1; i < 4; ++i)
        if (i != direction - 1) perm[j++] = i;
    long long sd[4];   // strides of the standard layout [d1,d2,d3,d4,bond]
    const int g0 = c.bond;
    sd[3] = g0;
    for (int i = 2; i >= 0; --i) sd[i] = sd[i + 1] * c.dims[i + 1];
    const long long n0 = c.dims[perm[0]], n1 = c.dims[perm[1]], n2 = c.dims[perm[2]], n3 = c.dims[perm[3]];
    const long long R = n0 * n1 * n2 * n3, nT = n1 * n2 * n3, n12 = n1 * n2;
    auto rot_view = [&](double *p, long long bond) {
        Ten t;
        t.p = p;
        for (int i = 0; i < 4; ++i) t.legs.push_back(Leg{'?', (long long)c.dims[perm[i]], sd[perm[i]] / g0 * bond});
        t.legs.push_back(Leg{'?', bond, 1});
        return t;
    };

    // ---- workspace: new state at the end opposite to the current one
    const long long m1cap = std::min<long long>(chi, n1 * n1), m2cap = std::min<long long>(chi, n2 * n2),
                    m3cap = std::min<long long>(chi, n3 * n3), gcap = std::min<long long>(chi, g0 * nT);
    const size_t new_cap = (((size_t)(n0 * m1cap * m2cap * m3cap * gcap) * 8 + 255) / 256) * 256;
    double *phi_new, *psi_new;
    if (c.state_low) {
        c.lo = c.state_bytes;
        c.hi = c.ws_bytes;
        if (c.hi < c.lo + 2 * new_cap) fail(-12, "workspace too small for the new state");
        c.hi -= 2 * new_cap;
        phi_new = (double *)(c.ws + c.hi);
    } else {
        c.lo = 0;
        c.hi = c.ws_bytes - c.state_bytes;
        if (c.hi < 2 * new_cap) fail(-12, "workspace too small for the new state");
        phi_new = (double *)(c.ws + c.lo);
        c.lo += 2 * new_cap;
    }
    psi_new = phi_new + new_cap / 8;
    c.peak = std::max(c.peak, c.lo + (c.ws_bytes - c.hi));
    prefetch_inputs();
    std::vector<double> spec[10];
    double gaps[4] = {INFINITY, INFINITY, INFINITY, INFINITY};

    stage_mark(0);
    trace_mark("step begin");
    // =================== O2 canonical form ===================
    // A, D and sigma^T outlive this stage; everything else of it (the chi^5-sized Q factors included)
    // is released once A and D are formed
    double *Abuf = ws_doubles(R * g0), *Dbuf = ws_doubles(R * g0);
    double *sT = ws_doubles(g0);
    const size_t canon_mark = ws_mark();
    Ten Qp = ws_tensor("rg", {R, g0}), Qs = ws_tensor("rg", {R, g0});
    Ten Rp = ws_tensor("gr", {g0, g0}), Rs = ws_tensor("hr", {g0, g0});
    // the last Cholesky-QR factor of each side is not applied to the chi^5-sized block: Q = Q' L2inv^T, and every
    // use of Q below is a product with a small matrix that absorbs it (one pass over the block less per side)
    Ten L2ip = ws_tensor("gc", {g0, g0}), L2is = ws_tensor("gc", {g0, g0});
    {
        // the two tall QRs are independent: asynchronous Cholesky-QR2 on two streams; a side that is
        // rank deficient or too ill conditioned for it (the early steps) is redone by the robust route
        bool qr_done[2] = {false, false};
        double *Yq[2] = {Qp.p, Qs.p};
        const double *src[2] = {c.phi, c.psi};
        double *Rq[2] = {Rp.p, Rs.p};
        double *L2q[2] = {L2ip.p, L2is.p};
        if (!(c.routes & ROUTE_HOUSEHOLDER_QR) && R >= 16LL * g0 && R >= 512) {
            struct QrBack {
                int flag;
                int pad;
                double ratio[2];
            };
            Fork fk(2);
            for (int i = 0; i < 2; ++i) {
                fk.enter(i);
                QrBack *bk = reinterpret_cast<QrBack *>(fk.pinned(i));
                int *flag = (int *)ws_alloc(sizeof(int));
                double *ratio = ws_doubles(2);
                TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(int), stream()));
                cholqr_async(Yq[i], R, g0, 2, 0.0, flag, ratio, Rq[i], src[i], L2q[i]);   // reads Phi / Psi, writes Q'
                TATRG_CUDA_CHECK(cudaMemcpyAsync(&bk->flag, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
                TATRG_CUDA_CHECK(cudaMemcpyAsync(bk->ratio, ratio, 2 * sizeof(double), cudaMemcpyDeviceToHost, stream()));
                fk.leave();
            }
            for (int i = 0; i < 2; ++i) {
                fk.sync(i);
                const QrBack *bk = reinterpret_cast<QrBack *>(fk.pinned(i));
                qr_done[i] = bk->flag == 0 && bk->ratio[0] > 1e-5 * bk->ratio[1];
            }
            fk.join();
        }
        for (int i = 0; i < 2; ++i)
            if (!qr_done[i]) {
                d2d(Yq[i], src[i], R * g0);
                tsqr(Yq[i], R, g0, Rq[i]);
                fill_identity(L2q[i], (int)g0);
            }
    }
    trace_mark("canon: two tall QRs");
    // C = R_Phi R_Psi^T, stored transposed ([h][g]) so that the buffer is column-major C
    Ten Cm = ws_tensor("hg", {g0, g0});
    contract(Rs, Rp, Cm);
    Ten Vc = ws_tensor("ah", {g0, g0});    // rows = right singular vectors v_a[h]
    jacobi_svd(Cm.p, g0, g0, Vc.p, sT, 1, 0, 0, 0);   // C V = U diag(sT); Cm rows -> u_a[g] sT_a
    spec[0] = d2h(sT, g0);
    const int a = num_rank(spec[0], -1);
    if (a < 1) fail(-34, "coarse_grain: tensor is numerically zero");
    spec[0].resize(a);
    scale_leg(Cm.p, (long long)a * g0, g0, a, sT, 1);
    Ten u = Ten::make(Cm.p, "ag", {a, g0});   // u[a][g] = u_a[g]
    Ten v = Ten::make(Vc.p, "ah", {a, g0});
    trace_mark("canon: core svd");
    // gauge (reading G12): P = A^T G_ref = u^T (Q_Phi^T G_ref)
    Ten QpR = rot_view(Qp.p, g0), QsR = rot_view(Qs.p, g0);
    Ten ref = get_input(5, R, a, cfg, "rb");
    Ten ref5 = Ten::make(ref.p, "xpqtb", {n0, n1, n2, n3, a});
    Ten T1y = ws_tensor("cb", {g0, a}), T1 = ws_tensor("gb", {g0, a});
    contract(QpR.as("xpqtc"), ref5, T1y);
    contract(L2ip, T1y, T1);                // Q_Phi^T G_ref = L2inv (Q'^T G_ref)
    Ten Pg = ws_tensor("ab", {a, a});
    contract(u, T1, Pg);
    Ten Wg = gauge_rotation(Pg, spec[0], a);
    Ten u2 = ws_tensor("bg", {a, g0}), v2 = ws_tensor("bg", {a, g0});
    contract(Wg, u, u2);                    // u2[b][g] = sum_a W[a,b] u[a][g]
    contract(Wg, v.as("ag"), v2);
    trace_mark("canon: gauge");
    Ten A = Ten::make(Abuf, "xpqta", {n0, n1, n2, n3, a}), D = Ten::make(Dbuf, "xpqta", {n0, n1, n2, n3, a});
    Ten u3 = ws_tensor("ac", {a, g0}), v3 = ws_tensor("ac", {a, g0});
    contract(u2.as("ag"), L2ip, u3);        // A = Q u2^T = Q' (L2inv^T u2^T)
    contract(v2.as("ag"), L2is, v3);
    contract(QpR.as("xpqtc"), u3, A);
    contract(QsR.as("xpqtc"), v3, D);
    trace_mark("canon: A, D");
    ws_release(canon_mark);
    stage_mark(1);

    // =================== O3 bond swap (Table 1 row 1) ===================
    const long long dim = a * nT;
    const int ell = (int)std::min<long long>((long long)r * chi, dim);
    double *Xbuf = ws_doubles(dim * std::min<long long>(chi, ell));
    double *Ybuf = ws_doubles(dim * std::min<long long>(chi, ell));
    int gs = 0;
    double *sig = nullptr;
    bool swapped = false, x_scaled = false;
    // Reduced operator: M = (1 x Q_A) m (1 x Q_D)^T with A[c,I',b] = sum_k Q_A[I',k] R_A[k,c,b] and
    // D likewise (Q_A, Q_D orthonormal, nT x n0 a), m[(a k),(b l)] = sum_c sT_a R_D[l,c,a] R_A[k,c,b] sT_b.
    // Every iterate of the subspace iteration lies in the range of 1 x Q_A (resp. 1 x Q_D) and
    // qr+((1 x Q) y) = (1 x Q) qr+(y), so the RSVD of M with the sketch Omega is the RSVD of m with the
    // sketch (1 x Q_D)^T Omega, expanded at the end: the same X, sigma, Y at 1/chi of the flops.
    const long long nk = n0 * a;
    if (!(c.routes & ROUTE_PLAIN_SWAP) && nT >= 2 * nk && nk >= 16) {
        size_t mk = ws_mark();
        RedBasis bA, bD;
        // Omega_red[b,l,z] = sum_l' L2inv_D[l,l'] sum_uvw Q1_D[uvw,l'] Omega[b,uvw,z]: the first product (the
        // chi^4 x r chi sketch against Q1_D, a machine-filling GEMM) needs Q1_D only and runs beside the last
        // factorisations of the two bases
        Ten om_red = ws_tensor("blz", {a, nk, ell});
        Ten t1 = ws_tensor("bmz", {a, nk, ell});
        auto project = [&](const RedBasis &bd) {
            Ten omega = get_input(0, dim, ell, cfg, "rz");
            contract(bd.Q1.as("uvwm"), Ten::make(omega.p, "buvwz", {a, n1, n2, n3, ell}), t1);
        };
        if (ortho_factor_pair(A, D, bA, bD, project)) {
            trace_mark("swap: bases of A, D, sketch projection");
            const long long rdim = a * nk;
            const int ellr = (int)std::min<long long>(ell, rdim);
            contract(bD.L2inv.as("lm"), t1, om_red);
            Ten Z = ws_tensor("cabz", {n0, a, a, ell});
            auto apply = [&](const double *w, double *out) {     // m w : [(b,l), z] -> [(a,k), z]
                contract(bD.R.as("lca"), Ten::make(const_cast<double *>(w), "blz", {a, nk, ell}), Z);
                scale_leg(Z.p, Z.size(), (long long)a * ell, a, sT, 0);
                scale_leg(Z.p, Z.size(), ell, a, sT, 0);
                contract(bA.R.as("kcb"), Z, Ten::make(out, "akz", {a, nk, ell}));
            };
            auto apply_t = [&](const double *w, double *out) {   // m^T w : [(a,k), z] -> [(b,l), z]
                contract(bA.R.as("kcb"), Ten::make(const_cast<double *>(w), "akz", {a, nk, ell}), Z.as("cbaz"));
                scale_leg(Z.p, Z.size(), (long long)a * ell, a, sT, 0);
                scale_leg(Z.p, Z.size(), ell, a, sT, 0);
                contract(bD.R.as("lca"), Z.as("cbaz"), Ten::make(out, "blz", {a, nk, ell}));
            };
            double *xr = ws_doubles(rdim * std::min<long long>(chi, ellr)), *yr = ws_doubles(rdim * std::min<long long>(chi, ellr));
            if (ellr == ell) {
                size_t mk2 = ws_mark();
                RsvdOut ro = rsvd(apply, apply_t, om_red, rdim, rdim, ell, q, chi, xr, yr);
                gs = ro.k;
                spec[1].assign(ro.s_full.begin(), ro.s_full.begin() + gs);
                gaps[0] = rel_gap(ro.s_full, gs);
                ws_release(mk2);
                trace_mark("swap: rsvd of the core");
                // expand: X[a,pqt,g] = sum_m Q1_A[pqt,m] sum_k L2inv_A[k,m] x[a,k,g]
                double *sg = ws_doubles(gs);    // (the device copy inside rsvd's workspace has just been released)
                h2d(sg, spec[1].data(), gs);
                Ten t2 = ws_tensor("amg", {a, nk, gs});
                contract(bA.L2inv.as("km"), Ten::make(xr, "akg", {a, nk, gs}), t2);
                scale_leg(t2.p, t2.size(), 1, gs, sg, 0);   // X enters the rest of the step only as X sigma (Eq. 5)
                x_scaled = true;
                contract(bA.Q1.as("pqtm"), t2, Ten::make(Xbuf, "apqtg", {a, n1, n2, n3, gs}));
                contract(bD.L2inv.as("km"), Ten::make(yr, "akg", {a, nk, gs}), t2);
                contract(bD.Q1.as("pqtm"), t2, Ten::make(Ybuf, "apqtg", {a, n1, n2, n3, gs}));
                swapped = true;
            }
        }
        std::vector<double> keep(spec[1]);
        ws_release(mk);
        if (swapped) {
            sig = ws_doubles(gs);
            h2d(sig, keep.data(), gs);
            TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
        }
    }
    if (!swapped) {
        size_t mk = ws_mark();
        Ten omega = get_input(0, dim, ell, cfg, "rz");
        Ten Z = ws_tensor("cabz", {n0, a, a, ell});
        auto sw_apply = [&](const double *w, double *out) {   // M w : [(b,J), z] -> [(a,I'), z]
            contract(D.as("cuvwa"), Ten::make(const_cast<double *>(w), "buvwz", {a, n1, n2, n3, ell}), Z);
            scale_leg(Z.p, Z.size(), (long long)a * ell, a, sT, 0);
            scale_leg(Z.p, Z.size(), ell, a, sT, 0);
            contract(A.as("cpqtb"), Z, Ten::make(out, "apqtz", {a, n1, n2, n3, ell}));
        };
        auto sw_apply_t = [&](const double *w, double *out) {  // M^T w : [(a,I'), z] -> [(b,J), z]
            contract(A.as("cpqtb"), Ten::make(const_cast<double *>(w), "apqtz", {a, n1, n2, n3, ell}), Z.as("cbaz"));
            scale_leg(Z.p, Z.size(), (long long)a * ell, a, sT, 0);
            scale_leg(Z.p, Z.size(), ell, a, sT, 0);
            contract(D.as("cuvwa"), Z.as("cbaz"), Ten::make(out, "buvwz", {a, n1, n2, n3, ell}));
        };
        RsvdOut ro = rsvd(sw_apply, sw_apply_t, omega, dim, dim, ell, q, chi, Xbuf, Ybuf);
        gs = ro.k;
        spec[1].assign(ro.s_full.begin(), ro.s_full.begin() + gs);
        gaps[0] = rel_gap(ro.s_full, gs);
        std::vector<double> keep(ro.s_full.begin(), ro.s_full.begin() + gs);
        ws_release(mk);
        sig = ws_doubles(gs);
        h2d(sig, keep.data(), gs);
        TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
    }
    Ten X = Ten::make(Xbuf, "apqtg", {a, n1, n2, n3, gs});
    Ten Y = Ten::make(Ybuf, "buvwg", {a, n1, n2, n3, gs});
    // X enters the rest of the step only as X sigma (Eq. 5): scaled in place; Y is needed both ways
    Ten Xs = X, Ys = ws_tensor("buvwg", {a, n1, n2, n3, gs});
    if (!x_scaled) scale_leg(Xs.p, Xs.size(), 1, gs, sig, 0);
    scale_inner_copy(Y.p, Ys.p, Y.size(), gs, sig);
    trace_mark("swap: expansion, scaling");
    stage_mark(2);

    bool overlapped = false;   // the squeezers run beside the Gram chains and steps (i), (ii) of the contraction
    size_t gram_mark = 0;
    Ten U[4];   // A, X, Y, D : [p,q,k]
    bool iso_lazy[4] = {false, false, false, false};
    double *Hkeep[4] = {nullptr, nullptr, nullptr, nullptr};
    int iso_kk = 0;
    struct RitzBack {   // page-locked read-back of the deferred Ritz steps (r chi <= 64)
        int flag[4];
        double lam[4][64];
    } *ritz_back = nullptr;
    bool ritz_deferred[4] = {false, false, false, false};
    double *ritz_V = nullptr, *ritz_lam = nullptr;
    int *ritz_flag = nullptr;
    Ten E, F, G, H;
    long long kd = 0;
    Ten GL[3], GR[3];
    const long long nn[3] = {n1, n2, n3};
    Ten Ms[3], Ns[3];
    int kq[3] = {0, 0, 0};
    for (int mu = 0; mu < 3; ++mu) {
        GL[mu] = ws_tensor("psrv", {nn[mu], nn[mu], nn[mu], nn[mu]});
        GR[mu] = ws_tensor("psrv", {nn[mu], nn[mu], nn[mu], nn[mu]});
        const long long N2 = nn[mu] * nn[mu];
        Ms[mu] = ws_tensor("uok", {nn[mu], nn[mu], std::min<long long>(chi, N2)});
        Ns[mu] = ws_tensor("kuo", {std::min<long long>(chi, N2), nn[mu], nn[mu]});
    }
    // M^(4) once more as [t, w, T]: step (i) of Eq. 13 then writes E M^(4) with the legs summed in (ii) last
    Ten M3t = ws_tensor("twT", {n3, std::min<long long>(chi, n3 * n3), n3});
    bool done[3] = {false, false, false};
    // gauge (reading G12) P = N G_ref, then M W and W^T N into the step's squeezer buffers
    auto finish = [&](int mu, const Ten &Mr, const Ten &Nr, const std::vector<double> &sh, int k) {
        const long long N2 = nn[mu] * nn[mu];
        kq[mu] = k;
        spec[6 + mu].assign(sh.begin(), sh.begin() + k);
        Ten rf = get_input(6 + mu, N2, k, cfg, "nb");
        Ten Pq = ws_tensor("kb", {k, k});
        contract(Nr, rf, Pq);
        Ten Wq = gauge_rotation(Pq.as("ab"), sh, k);
        Ms[mu] = Ten::make(Ms[mu].p, "uok", {nn[mu], nn[mu], k});
        Ns[mu] = Ten::make(Ns[mu].p, "kuo", {k, nn[mu], nn[mu]});
        contract(Mr.as("na"), Wq, Ten::make(Ms[mu].p, "nb", {N2, k}));
        contract(Wq, Nr.as("an"), Ten::make(Ns[mu].p, "bn", {k, N2}));
        if (mu == 2) {
            M3t = Ten::make(M3t.p, "twT", {nn[2], k, nn[2]});
            Ten Mr3;   // Mr[(t, T), a] with its row index split into the two legs
            Mr3.p = Mr.p;
            Mr3.legs = {Leg{'t', nn[2], nn[2] * Mr.legs[0].stride}, Leg{'T', nn[2], Mr.legs[0].stride}, Leg{'a', Mr.legs[1].n, Mr.legs[1].stride}};
            contract(Mr3, Wq.as("aw"), M3t);
        }
    };
    // The subspace-iteration squeezers of the directions `mus` as concurrent chains (large legs only; the
    // others, and chains that give up, are left to squeeze_dense).  main_work (may be empty) is enqueued on
    // the main stream once the chains' factorisations are under way and runs beside them: the persistent GEMM
    // leaves SM_RESERVE SMs to the chains meanwhile.
    constexpr int SM_RESERVE = CHAIN_SM_RESERVE;
    int sq_hist_new[3] = {0, 0, 0};
    auto squeeze_wave = [&](const std::vector<int> &mus, const std::function<void()> &main_work,
                            const std::function<void()> &tail_work = nullptr, int reserve = -1) {
        SqChain ch[3];
        std::vector<int> act;
        long long n2max = 0;
        for (int mu : mus) {
            const long long N2 = nn[mu] * nn[mu];
            ch[mu].b = chi < 64 ? 64 : 128;
            ch[mu].active = !(c.routes & ROUTE_DENSE_SQUEEZER) && N2 >= 4 * ch[mu].b && chi < ch[mu].b;
            ch[mu].GLm = GL[mu];
            ch[mu].GRm = GR[mu];
            ch[mu].N2 = (int)N2;
            ch[mu].chi = chi;
            ch[mu].mu = mu;
            ch[mu].hist = c.sq_hist[direction - 1][mu];
            if (ch[mu].active) {
                act.push_back(mu);
                n2max = std::max(n2max, N2);
            }
        }
        if (act.empty()) {
            if (main_work) main_work();
            if (tail_work) tail_work();
            return;
        }
        for (int mu : act) ch[mu].prep();
        const int na = (int)act.size();
        const int rsv = reserve >= 0 ? reserve : SM_RESERVE;
        // the iteration of a chain as one resident grid (sq_iter.cu), one CTA per SM: beside the main stream's GEMMs
        // it takes the SMs those leave free, so two chains run their grids one after the other (resident grids that
        // do not fit into the reserve together would hold back CTAs of the persistent GEMM)
        bool fused = !(c.routes & ROUTE_UNFUSED_SQUEEZER);
        for (int mu : act) fused = fused && ch[mu].b == 64;
        for (int mu : act) ch[mu].grid = fused ? (main_work ? rsv : 32) : 0;
        const bool one_grid_at_a_time = fused && main_work && na > 1;
        const size_t chain_bytes = main_work ? std::max<size_t>((size_t)64 << 20, (size_t)(6 * n2max * n2max * 8)) : 0;
        Fork fk(2 * na, (bool)main_work, chain_bytes);
        c.chol_ctas = main_work ? std::max(2, rsv / (2 * na)) : 16;   // resident grids (chol.cu) that fit into the reserve together
        for (int i = 0; i < na; ++i)           // the two Cholesky factorisations of a chain side by side
            for (int w = 0; w < 2; ++w) {
                fk.enter(2 * i + w);
                ch[act[i]].factor(w);
                fk.leave();
            }
        c.chol_ctas = 16;
        for (int i = 0; i < na; ++i) fk.side_after_side(2 * i, 2 * i + 1);
        fk.enter(0);
        trace_mark("sq chain 0: cholesky x2");
        fk.leave();
        if (main_work) {
            c.sm_reserve = rsv;
            main_work();
            c.sm_reserve = 0;
        }
        for (int i = 0; i < na; ++i) {
            if (one_grid_at_a_time && i > 0) fk.side_after_side(2 * i, 2 * (i - 1));
            fk.enter(2 * i);
            ch[act[i]].phaseA(fk.pinned(2 * i));
            fk.leave();
        }
        fk.enter(0);
        trace_mark("sq chain 0: phase A");
        fk.leave();
        for (int i = 0; i < na; ++i) {
            fk.sync(2 * i);
            if (ch[act[i]].too_ill_conditioned()) {
                fk.enter(2 * i);
                ch[act[i]].ritz_robust();
                fk.leave();
            }
            ch[act[i]].ok = ch[act[i]].plan();
            if (getenv("TATRG_TRACE"))
                fprintf(stderr, "tatrg-trace squeezer mu %d: hist %d done %d planned %d more %d ok %d\n", act[i], ch[act[i]].hist,
                        ch[act[i]].iters_done, ch[act[i]].planned, ch[act[i]].more, (int)ch[act[i]].ok);
        }
        for (int i = 0, prev = -1; i < na; ++i)
            if (ch[act[i]].ok && ch[act[i]].more > 0) {
                if (one_grid_at_a_time && prev >= 0) fk.side_after_side(2 * i, 2 * prev);
                prev = i;
                fk.enter(2 * i);
                ch[act[i]].phaseB();
                fk.leave();
            }
        for (int i = 0; i < na; ++i)
            if (ch[act[i]].ok) {
                const int mu = act[i];
                if (ch[mu].more > 0) fk.sync(2 * i);
                fk.enter(2 * i);
                if (ch[mu].more > 0 && ch[mu].too_ill_conditioned()) ch[mu].ritz_robust();
                if (ch[mu].phaseC()) {
                    gaps[1 + mu] = ch[mu].gap;
                    finish(mu, ch[mu].Mr, ch[mu].Nr, ch[mu].sh, ch[mu].k);
                    done[mu] = true;
                    sq_hist_new[mu] = std::max(3, ch[mu].planned);
                }
                fk.leave();
            }
        fk.enter(0);
        trace_mark("sq chain 0: phase B, C, gauge");
        fk.leave();
        if (tail_work) {   // the chains are enqueued to their end: what follows on the main stream gets every SM
            for (int i = 0; i < na; ++i) fk.sync(2 * i);
            tail_work();
        }
        fk.join();
    };
    // dense route = the oracle's algorithm: eigendecompositions of both Grams, SVD of R1 R2
    auto squeeze_dense = [&](int mu) {
        const int N2 = (int)(nn[mu] * nn[mu]);
        size_t mk = ws_mark();
        Ten Mr, Nr;
        std::vector<double> sh;
        double *sf;
        int k;
        {
            Ten V1 = ws_tensor("in", {N2, N2}), V2 = ws_tensor("jn", {N2, N2});
            double *l1 = ws_doubles(N2), *l2 = ws_doubles(N2);
            std::vector<double> lam1 = sym_eig(GL[mu].p, N2, V1.p, l1);
            std::vector<double> lam2 = sym_eig(GR[mu].p, N2, V2.p, l2);
            const int kl = num_rank(lam1, -1), kr = num_rank(lam2, -1);
            if (kl < 1 || kr < 1) fail(-34, "squeezer: Gram matrix is numerically zero");
            // R1 = Lambda^1/2 V^T (rows of V1 scaled), R2^T likewise
            scale_leg(V1.p, (long long)kl * N2, N2, kl, l1, 2);
            scale_leg(V2.p, (long long)kr * N2, N2, kr, l2, 2);
            Ten R1 = V1, R2 = V2;
            R1.legs[0].n = kl;
            R2.legs[0].n = kr;
            Ten Fm = ws_tensor("ji", {kr, kl});        // buffer = column-major F = R1 R2 (kl x kr)
            contract(R2, R1, Fm);
            Ten Vf = ws_tensor("kj", {kr, kr});
            sf = ws_doubles(kr);
            jacobi_svd(Fm.p, kl, kr, Vf.p, sf, 1, 0, 0, 0);   // F V = U diag(s): Fm rows -> U_k[i] s_k
            sh = d2h(sf, kr);
            sh.resize(std::min(kl, kr));
            k = num_rank(sh, chi);
            if (k < 1) fail(-34, "squeezer: R1 R2 is numerically zero");
            gaps[1 + mu] = rel_gap(sh, k);
            Ten Vk = Vf, Uk = Fm.as("ki");
            Vk.legs[0].n = k;
            Uk.legs[0].n = k;
            Mr = ws_tensor("nk", {N2, k});
            Nr = ws_tensor("kn", {k, N2});
            contract(R2, Vk, Mr);                       // M = R2 V s^-1/2
            contract(Uk, R1, Nr);                       // N = s^-1/2 U^T R1, U = Fm rows / s
            scale_leg(Mr.p, Mr.size(), 1, k, sf, 3);
            scale_leg(Nr.p, Nr.size(), N2, k, sf, 5);
        }
        finish(mu, Mr, Nr, sh, k);
        ws_release(mk);
        done[mu] = true;
    };
    if (mode == 0) {
    // =================== O4 oversampled isometries (Eqs. 2-3) ===================
    const int kk = (int)std::min<long long>((long long)r * chi, n12);
    if (kk >= n12) {
        for (int i = 0; i < 4; ++i) {
            U[i] = ws_tensor("pqk", {n1, n2, n12});
            fill_identity(U[i].p, (int)n12);
        }
    } else {
        Ten RX = ws_tensor("ab", {a, a}), RY = ws_tensor("ab", {a, a});
        contract(Xs.as("apqtg"), Xs.as("bpqtg"), RX);
        contract(Ys.as("apqtg"), Ys.as("bpqtg"), RY);
        for (int i = 0; i < 4; ++i) U[i] = ws_tensor("pqk", {n1, n2, kk});
        struct IsoBack {   // page-locked read-back of one chain
            int flag;
            int pad;
            double ratio[16];
            double lam[64];
        };
        // One isometry: subspace iteration on the symmetric PSD operator S = K K_w^T on the pair space
        // (reading G6b), then a Ritz step.  fast: asynchronous Cholesky-QR and one-CTA eigensolver, no
        // host synchronisation (the caller checks the read-back); else the robust synchronous route.
        auto iso_body = [&](int i, bool fast, IsoBack *back) {
            const Ten &Kt = (i == 0) ? A : (i == 1) ? Xs : (i == 2) ? Ys : D;
            const bool mid = (i == 0 || i == 3);
            const Ten &Rm = (i == 0) ? RX : RY;
            const long long e0 = Kt.legs[0].n, e3 = Kt.legs[3].n, e4 = Kt.legs[4].n;
            Ten t1 = ws_tensor("xtaz", {e0, e3, e4, kk}), t2 = ws_tensor("xtbz", {e0, e3, e4, kk});
            auto S_op = [&](const double *w, double *out) {
                contract(Kt.as("xpqta"), Ten::make(const_cast<double *>(w), "pqz", {n1, n2, kk}), t1);
                if (mid) {
                    contract(t1, Rm, t2);
                    contract(Kt.as("xpqtb"), t2, Ten::make(out, "pqz", {n1, n2, kk}));
                } else {
                    contract(Kt.as("xpqta"), t1, Ten::make(out, "pqz", {n1, n2, kk}));
                }
            };
            int *flag = nullptr;
            double *ratio = nullptr;
            if (fast) {
                flag = (int *)ws_alloc(sizeof(int));
                TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(int), stream()));
                ratio = ws_doubles(16);
            }
            int nqr = 0;
            // last: the block that enters the Ritz step (two passes); before it only the span is carried on
            auto orth = [&](double *Y, bool last) {
                if (fast) {
                    if (last) {
                        // wide lines (the paper's r = 7): r chi columns reach far down the spectrum of S and the
                        // block is often too ill conditioned for two plain passes (the chain was rejected and the
                        // isometry redone on the synchronous route, 25 ms each): a shifted pass first (shifted
                        // Cholesky-QR3; the span, all that enters Gamma^triad, is unchanged), the check on the next
                        if (kk > 64) cholqr_async(Y, n12, kk, 1, 1e-13, flag, nullptr, nullptr);
                        cholqr_async(Y, n12, kk, 2, 0.0, flag, ratio + 2 * nqr, nullptr);
                        ++nqr;
                    } else {
                        cholqr_async(Y, n12, kk, 1, 1e-13, flag, nullptr, nullptr);
                    }
                } else {
                    double *Rtmp = ws_doubles((long long)kk * kk);
                    tsqr(Y, n12, kk, Rtmp);
                }
            };
            Ten om = get_input(1 + i, n12, kk, cfg, "rz");
            Ten Qi = ws_tensor("rz", {n12, kk});
            S_op(om.p, Qi.p);
            orth(Qi.p, q == 0);
            for (int it = 0; it < q; ++it) {
                S_op(Qi.p, Qi.p);        // (the block is read by the first product only)
                orth(Qi.p, it == q - 1);
            }
            // Ritz matrix H = Q^T S Q = (K Q)^T (K_w Q): a Gram matrix of t1 = K Q (weighted with R for the two
            // middle chains) -- the product with K^T back to the pair space, half of an application of S, is
            // not needed for it
            Ten Hm = ws_tensor("zy", {kk, kk});
            contract(Kt.as("xpqta"), Ten::make(Qi.p, "pqz", {n1, n2, kk}), t1);
            if (mid) {
                contract(t1, Rm, t2);
                contract(t1.as("xtbz"), t2.as("xtby"), Hm);
            } else {
                contract(t1.as("xtaz"), t1.as("xtay"), Hm);
            }
            Ten Vt = ws_tensor("kz", {kk, kk});
            double *lam = ws_doubles(kk);
            if (fast) {
                // The Ritz rotation is left out of the path.  Gamma^triad depends on U only through its span
                // (E I = A U U^T etc.: every oversampled line is summed over in Eqs. 13-14 and in the Grams
                // of Eq. 12), so the orthonormal block Q itself is used as U.  r chi <= 64: the eigenvalues
                // of the Ritz matrix H (the spectrum S of the step) are computed by the one-CTA solver on a
                // stream of their own BESIDE the triad tensors and Gram chains (below) and read at the end of
                // the step -- four single-CTA kernels no longer hold up the machine.  Wider lines: H goes to
                // the host and S is computed from it when it is asked for (resolve_iso_spectra).
                d2d(U[i].p, Qi.p, n12 * kk);
                d2d(Hkeep[i], Hm.p, (long long)kk * kk);
                back->pad = nqr;
                TATRG_CUDA_CHECK(cudaMemcpyAsync(&back->flag, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
                TATRG_CUDA_CHECK(cudaMemcpyAsync(back->ratio, ratio, 2 * nqr * sizeof(double), cudaMemcpyDeviceToHost, stream()));
                return;
            }
            std::vector<double> lh = sym_eig(Hm.p, kk, Vt.p, lam);   // the robust synchronous route
            spec[2 + i].resize(kk);
            for (int j = 0; j < kk; ++j) spec[2 + i][j] = sqrt(std::max(lh[j], 0.0));
            contract(Ten::make(Qi.p, "pqz", {n1, n2, kk}), Vt, U[i]);
        };
        bool iso_done[4] = {false, false, false, false};
        const bool wide = kk > 64;
        for (int i = 0; i < 4; ++i) Hkeep[i] = ws_doubles((long long)kk * kk);   // outlives the chains' slices
        if (!wide) {
            ritz_V = ws_doubles(4LL * kk * kk);
            ritz_lam = ws_doubles(4LL * kk);
            ritz_flag = (int *)ws_alloc(4 * sizeof(int));
        }
        if (!(c.routes & ROUTE_SEQUENTIAL_ISO) && kk <= 256 && q + 1 <= 8 && n12 >= (wide ? 2LL : 4LL) * kk) {   // the four isometries as concurrent chains
            Fork fk(4);
            for (int i = 0; i < 4; ++i) {
                fk.enter(i);
                iso_body(i, true, reinterpret_cast<IsoBack *>(fk.pinned(i)));
                fk.leave();
            }
            for (int i = 0; i < 4; ++i) {
                fk.sync(i);
                const IsoBack *bk = reinterpret_cast<IsoBack *>(fk.pinned(i));
                bool ok = bk->flag == 0;
                for (int j = 0; j < bk->pad; ++j) ok = ok && bk->ratio[2 * j] > 1e-5 * bk->ratio[2 * j + 1];
                if (!ok) {           // ill conditioned block or no convergence: redone below
                    if (getenv("TATRG_TRACE")) fprintf(stderr, "tatrg-trace isometry %d: chain rejected (flag %d), robust route\n", i, bk->flag);
                    continue;
                }
                iso_kk = kk;
                if (wide)
                    iso_lazy[i] = true;
                else
                    ritz_deferred[i] = true;
                iso_done[i] = true;
            }
            fk.join();
            // the deferred Ritz steps: one single-CTA eigensolver per isometry on side streams 4..7 (no Fork of this
            // step has more than six chains), after everything the chains wrote; read back at the end of the step
            if (!wide) {
                TATRG_CUDA_CHECK(cudaMemsetAsync(ritz_flag, 0, 4 * sizeof(int), stream()));
                TATRG_CUDA_CHECK(cudaEventRecord(c.fork_ev, stream()));
                ritz_back = reinterpret_cast<RitzBack *>(fk.pinned(Ctx::MAX_CHAINS - 1));
                cudaStream_t main_stream = c.stream;
                for (int i = 0; i < 4; ++i) {
                    if (!ritz_deferred[i]) continue;
                    c.stream = c.side[4 + i];
                    TATRG_CUDA_CHECK(cudaStreamWaitEvent(c.stream, c.fork_ev, 0));
                    eig_small_async(Hkeep[i], kk, ritz_V + (long long)i * kk * kk, ritz_lam + (long long)i * kk, ritz_flag + i);
                    TATRG_CUDA_CHECK(cudaMemcpyAsync(&ritz_back->flag[i], ritz_flag + i, sizeof(int), cudaMemcpyDeviceToHost, c.stream));
                    TATRG_CUDA_CHECK(cudaMemcpyAsync(ritz_back->lam[i], ritz_lam + (long long)i * kk, kk * sizeof(double), cudaMemcpyDeviceToHost, c.stream));
                    c.stream = main_stream;
                }
            }
        }
        for (int i = 0; i < 4; ++i)
            if (!iso_done[i]) {
                size_t mk = ws_mark();
                iso_lazy[i] = false;
                ritz_deferred[i] = false;
                iso_body(i, false, nullptr);
                ws_release(mk);
            }
    }
    kd = U[0].legs[2].n;
    if (c.keep_iso) {   // tests: the gauge-invariant projectors U U^T are compared with the oracle's
        c.iso_rows = (int)n12;
        c.iso_cols = (int)kd;
        for (int i = 0; i < 4; ++i) c.iso[i] = d2h(U[i].p, n12 * kd);
    }
    stage_mark(3);

    // =================== O5 triad tensors (Eqs. 4-7) ===================
    E = ws_tensor("xkta", {n0, kd, n3, a});
    F = ws_tensor("aktg", {a, kd, n3, gs});
    G = ws_tensor("bktg", {a, kd, n3, gs});
    H = ws_tensor("xktb", {n0, kd, n3, a});
    contract(A.as("xpqta"), U[0], E);
    contract(Xs.as("apqtg"), U[1], F);     // sigma is inside Xs (Eq. 5)
    contract(Y.as("bpqtg"), U[2], G);
    contract(D.as("xpqtb"), U[3], H);
    stage_mark(4);

    // =================== O6 Gram matrices of Gamma^triad (Eq. 12) ===================
    {
        gram_mark = ws_mark();
        Ten HH0 = ws_tensor("bc", {a, a}), EE0 = ws_tensor("ab", {a, a});
        contract(H.as("xktb"), H.as("xktc"), HH0);
        contract(E.as("xkta"), E.as("xktb"), EE0);
        Ten Gh = ws_tensor("cktg", {a, kd, n3, gs}), Fh = ws_tensor("bktg", {a, kd, n3, gs});
        contract(HH0, G.as("bktg"), Gh);
        contract(EE0, F.as("aktg"), Fh);
        Ten Sm = ws_tensor("gd", {gs, gs}), Sp = ws_tensor("gd", {gs, gs});
        contract(Gh, G.as("cktd"), Sm);    // "-" half reduced to the swap bond
        contract(Fh, F.as("bktd"), Sp);    // "+" half
        Ten Fs = Fh, Gs = Gh;              // reuse: Fs[b,k,u,g] = sum_d F[b,k,u,d] Sm[g,d]
        contract(F.as("bkud"), Sm, Fs.as("bkug"));
        contract(G.as("ckud"), Sp, Gs.as("ckug"));
        {   // lone leg
            size_t mk2 = ws_mark();
            Ten EE3 = ws_tensor("taub", {n3, a, n3, a}), FF3 = ws_tensor("asbv", {a, n3, a, n3});
            contract(E.as("xkta"), E.as("xkub"), EE3);
            contract(F.as("aksg"), Fs.as("bkvg"), FF3);
            contract(EE3, FF3, GL[2].as("tsuv"));
            Ten GG3 = ws_tensor("btcu", {a, n3, a, n3}), HH3 = ws_tensor("sbvc", {n3, a, n3, a});
            contract(G.as("bktg"), Gs.as("ckug"), GG3);
            contract(H.as("xksb"), H.as("xkvc"), HH3);
            contract(GG3, HH3, GR[2].as("tsuv"));
            ws_release(mk2);
        }
        // grouped legs
        auto gram_grouped = [&]() {
            size_t mk1 = ws_mark();
            Ten EEk = ws_tensor("kalb", {kd, a, kd, a}), FFk = ws_tensor("kalb", {kd, a, kd, a});
            Ten GGk = ws_tensor("kblc", {kd, a, kd, a}), HHk = ws_tensor("kblc", {kd, a, kd, a});
            contract(E.as("xkta"), E.as("xltb"), EEk);
            contract(F.as("aktg"), Fs.as("bltg"), FFk);
            contract(G.as("bktg"), Gs.as("cltg"), GGk);
            contract(H.as("xktb"), H.as("xltc"), HHk);
            for (int mu = 0; mu < 2; ++mu) {
                size_t mk2 = ws_mark();
                const char *n1s = mu == 0 ? "pqk" : "qpk", *n2s = mu == 0 ? "rql" : "qrl";
                const long long np = nn[mu];
                Ten UU = ws_tensor("pkrl", {np, kd, np, kd});
                Ten Ta = ws_tensor("prab", {np, np, a, a}), Tb = ws_tensor("qsab", {np, np, a, a});
                contract(U[0].as(n1s), U[0].as(n2s), UU);
                contract(UU, EEk, Ta);
                contract(U[1].as(n1s), U[1].as(n2s), UU);
                contract(UU, FFk, Tb.as("prab"));
                contract(Ta, Tb, GL[mu].as("pqrs"));
                contract(U[2].as(n1s), U[2].as(n2s), UU);
                contract(UU, GGk.as("kalb"), Ta);
                contract(U[3].as(n1s), U[3].as(n2s), UU);
                contract(UU, HHk.as("kalb"), Tb.as("prab"));
                contract(Ta, Tb, GR[mu].as("pqrs"));
                ws_release(mk2);
            }
            ws_release(mk1);
        };
        // Large legs: the lone-leg squeezer (the only one steps (i), (ii) of Eqs. 13-14 need) runs as a chain
        // of small kernels BESIDE the grouped-leg Gram chains, and the two grouped-leg squeezers later beside
        // (i), (ii): their latency (Cholesky, ~17 subspace iterations, two 64 x 64 Jacobi each) disappears
        // behind machine-filling GEMMs.
        const int sq_b = chi < 64 ? 64 : 128;
        overlapped = !(c.routes & (ROUTE_DENSE_SQUEEZER | ROUTE_SEQUENTIAL_ISO)) && chi < sq_b;
        for (int mu = 0; mu < 3; ++mu) overlapped = overlapped && nn[mu] * nn[mu] >= 4 * sq_b;
        {   // room for the grouped-leg temporaries in the main stream's slice
            const double need = 8.0 * (4.0 * kd * a * kd * a + 2.0 * (double)n1 * kd * n1 * kd + 4.0 * (double)n1 * n1 * a * a) * 1.5 +
                                2.0 * std::max<double>(64 << 20, 6.0 * 8.0 * (double)n3 * n3 * n3 * n3);
            overlapped = overlapped && (double)(c.hi - c.lo) > need + (64 << 20);
        }
        if (overlapped) {
            stage_mark(5);
            squeeze_wave({2}, gram_grouped, nullptr, LONE_SM_RESERVE);
            if (!done[2]) squeeze_dense(2);
        } else {
            gram_grouped();
        }
        ws_release(gram_mark);
    }
    } else {
        // =================== plain ATRG (Table 1): squeezer Grams of A X sigma and of
        // sigma Y D only (the canonical form drops the other half; Table 1 "Squeezer step O(chi^7)")
        stage_mark(3);
        stage_mark(4);
        // leg letters of the three transverse legs: upper (p,q,t) / bar (P,Q,T); lower (r,s,u) / bar (R,S,U)
        const char up[3] = {'p', 'q', 't'}, ub[3] = {'P', 'Q', 'T'};
        for (int mu = 0; mu < 3; ++mu) {
            size_t mk = ws_mark();
            const long long nm = nn[mu];
            char n1s[6] = "xpqta", n2s[6] = "xpqtb";
            n2s[1 + mu] = ub[mu];
            char o[5] = {up[mu], 'a', ub[mu], 'b', 0};
            Ten AA = ws_tensor("taub", {nm, a, nm, a});
            contract(A.as(n1s), A.as(n2s), AA.as(o));                    // AA[i, al, ibar, albar]
            char x1[6] = "apqtg", x2[6] = "bpqtg";
            x2[1 + mu] = ub[mu];
            char ox[5] = {'a', up[mu], 'b', ub[mu], 0};
            Ten XX = ws_tensor("asbv", {a, nm, a, nm});
            contract(Xs.as(x1), Xs.as(x2), XX.as(ox));                   // XX[al, i', albar, ibar']
            contract(AA.as("taub"), XX.as("asbv"), GL[mu].as("tsuv"));   // G^L[(up,lo),(upbar,lobar)]
            Ten YY = AA, DD = XX;                                        // reuse the buffers
            YY = Ten::make(AA.p, "btcu", {a, nm, a, nm});
            DD = Ten::make(XX.p, "sbvc", {nm, a, nm, a});
            char oy[5] = {'a', up[mu], 'b', ub[mu], 0};
            contract(Ys.as(x1), Ys.as(x2), YY.as(oy));                   // YY[be, j, bebar, jbar]
            char od[5] = {up[mu], 'a', ub[mu], 'b', 0};
            contract(D.as(n1s), D.as(n2s), DD.as(od));                   // DD[j', be, jbar', bebar]
            contract(YY.as("btcu"), DD.as("sbvc"), GR[mu].as("tsuv"));
            ws_release(mk);
        }
    }
    if (!overlapped) stage_mark(5);

    // =================== O6 squeezers (Eq. 12; reading G10) ===================
    if (!overlapped) {
        squeeze_wave({0, 1, 2}, nullptr);
        for (int mu = 0; mu < 3; ++mu)
            if (!done[mu]) squeeze_dense(mu);
    }
    stage_mark(6);

    // =================== O7 contraction (Eqs. 13-14) ===================
    // (i) E M^(4) and (ii) . F need the lone-leg squeezer only: when the squeezers are overlapped, both sides'
    // (i), (ii) run on the main stream while the grouped-leg squeezers finish on their chains
    Ten Pt_pre[2];
    bool pre_done = false;
    if (overlapped) {
        const long long m3 = kq[2];
        const double per_x = 8.0 * ((double)kd * a * n3 * m3 + (double)kd * m3 * kd * gs);
        const long long xc = std::max<long long>(1, std::min<long long>(n0, (long long)(8.0e9 / per_x)));
        const double chains = 4.0 * std::max<double>(64 << 20, 6.0 * 8.0 * (double)n1 * n1 * n1 * n1);
        const double need = 8.0 * ((double)n0 * kd * a * n3 * m3 + 2.0 * (double)n0 * kd * m3 * kd * gs) + chains + (256 << 20);
        if (xc == n0 && (double)(c.hi - c.lo) > need) {
            // E M^(4) is stored with the legs summed in (ii) last, [x, k, w, (a, T)]: the A operand of (ii) is then
            // a plain row-major 65536 x 1024 matrix (summed index contiguous), the faster operand layout
            Ten EM = ws_tensor("xkwaT", {n0, kd, m3, a, n3});
            for (int side = 0; side < 2; ++side) Pt_pre[side] = ws_tensor("xkwlg", {n0, kd, m3, kd, gs});
            auto side0 = [&]() {
                contract(E.as("xkta"), M3t, EM);
                contract(EM, F.as("alTg"), Pt_pre[0]);
            };
            auto side1 = [&]() {
                // H is the lower site: its lone leg is the "lower" index of N3[w, upper, lower]
                contract(H.as("xkTa"), Ns[2].as("wtT"), EM.as("xkwat"));
                contract(EM.as("xkwat"), G.as("altg"), Pt_pre[1]);   // Pt[x, kD, w, kY, g]
            };
            // (handing the second side to the main stream only after the chains have ended, so that it gets every
            // SM, measured slower: the chains outlast the first side and the main stream idles meanwhile)
            squeeze_wave({0, 1}, [&]() {
                if (c.side_mask & 1) side0();
                if (c.side_mask & 2) side1();
            });
            pre_done = true;
        } else {
            squeeze_wave({0, 1}, nullptr);
        }
        for (int mu = 0; mu < 2; ++mu)
            if (!done[mu]) squeeze_dense(mu);
    }
    const long long m1 = kq[0], m2 = kq[1], m3 = kq[2];
    const long long nd[4] = {n0, m1, m2, m3};
    int new_dims[4];
    for (int i = 0; i < 4; ++i) new_dims[perm[i]] = (int)nd[i];
    long long nsd[4];
    nsd[3] = gs;
    for (int i = 2; i >= 0; --i) nsd[i] = nsd[i + 1] * new_dims[i + 1];
    auto new_view = [&](double *p) {
        Ten t;
        t.p = p;
        for (int i = 0; i < 4; ++i) t.legs.push_back(Leg{'?', nd[i], nsd[perm[i]]});
        t.legs.push_back(Leg{'?', (long long)gs, 1});
        return t;
    };
    if ((size_t)(n0 * m1 * m2 * m3 * gs) * 8 > new_cap) fail(-12, "internal: new state exceeds its reservation");
    for (int side = 0; side < 2 && mode == 0; ++side) {
        if (!(c.side_mask >> side & 1)) continue;   // the other GPU's half (tatrg_set_side_split)
        size_t mk = ws_mark();
        Ten W1 = ws_tensor("qkPm", {n2, kd, n1, m1}), V2 = ws_tensor("Plqn", {n1, kd, n2, m2});
        Ten Qt = ws_tensor("klmn", {kd, kd, m1, m2});
        if (side == 0) {
            contract(U[0].as("pqk"), Ms[0].as("pPm"), W1);
            contract(U[1].as("PQl"), Ms[1].as("qQn"), V2);
        } else {
            contract(U[2].as("pqk"), Ns[0].as("mpP"), W1);
            contract(U[3].as("PQl"), Ns[1].as("nqQ"), V2);
        }
        contract(W1, V2, Qt);
        Ten out = new_view(side == 0 ? phi_new : psi_new).as("xmnwg");
        if (pre_done) {   // (iv)
            if (side == 0)
                contract(Pt_pre[0], Qt, out);
            else
                contract(Pt_pre[1].as("xlwkg"), Qt, out);
            ws_release(mk);
            continue;
        }
        // (i)-(ii)-(iv) of Eqs. 13-14 in slabs of the direction-0 leg so that E M^(4) (r chi^5) and
        // P (r^2 chi^5) stay below ~8 GB (one slab = the whole tensor up to chi ~ 40)
        const double per_x = 8.0 * ((double)kd * a * n3 * m3 + (double)kd * m3 * kd * gs);
        const long long xc = std::max<long long>(1, std::min<long long>(n0, (long long)(8.0e9 / per_x)));
        Ten EM = ws_tensor("xkwaT", {xc, kd, m3, a, n3});
        Ten Pt = ws_tensor("xkwlg", {xc, kd, m3, kd, gs});
        auto slab = [](Ten t, long long x0, long long cnt) {   // legs[0] is the direction-0 leg
            t.p += x0 * t.legs[0].stride;
            t.legs[0].n = cnt;
            return t;
        };
        for (long long x0 = 0; x0 < n0; x0 += xc) {
            const long long cnt = std::min(xc, n0 - x0);
            Ten EMs = slab(EM, 0, cnt), Pts = slab(Pt, 0, cnt), outs = slab(out, x0, cnt);
            if (side == 0) {
                contract(slab(E.as("xkta"), x0, cnt), M3t, EMs);
                contract(EMs, F.as("alTg"), Pts);
                contract(Pts, Qt, outs);
            } else {
                // H is the lower site: its lone leg is the "lower" index of N3[w, upper, lower]
                contract(slab(H.as("xkTa"), x0, cnt), Ns[2].as("wtT"), EMs.as("xkwat"));
                contract(EMs.as("xkwat"), G.as("altg"), Pts);   // Pt[x, kD, w, kY, g]
                contract(Pts.as("xlwkg"), Qt, outs);
            }
        }
        ws_release(mk);
    }
    if (mode != 0) {
        // plain ATRG contraction, O(chi^9) (Table 1): Phi = sum A (X sigma) M1 M2 M3,
        // Psi = sum Y D N1 N2 N3, one slice of the direction-0 leg at a time (the chi^7-sized
        // intermediate of the whole tensor would not fit)
        size_t mk = ws_mark();
        Ten T1 = ws_tensor("qtarm", {n2, n3, a, n1, m1});          // per x: A[x] M1
        Ten T2 = ws_tensor("qtmsug", {n2, n3, m1, n2, n3, gs});    // . (X sigma) over (a, r)
        Ten T3 = ws_tensor("tmnug", {n3, m1, m2, n3, gs});         // . M2 over (q, s)
        Ten outP = new_view(phi_new), outS = new_view(psi_new);
        for (long long x = 0; x < n0 && (c.side_mask & 1); ++x) {
            Ten Ax = Ten::make(A.p + x * (n1 * n2 * n3 * a), "pqta", {n1, n2, n3, a});
            contract(Ax, Ms[0].as("prm"), T1);
            contract(T1, Xs.as("arsug"), T2);
            contract(T2, Ms[1].as("qsn"), T3);
            Ten ox = outP;
            ox.p += x * ox.legs[0].stride;
            ox.legs.erase(ox.legs.begin());
            contract(T3, Ms[2].as("tuw"), ox.as("mnwg"));
        }
        // Psi[x,m,n,w,g] = sum Y[b,p,q,t,g] D[x,r,s,u,b] N1[m,p,r] N2[n,q,s] N3[w,t,u]
        Ten S1 = ws_tensor("subpm", {n2, n3, a, n1, m1});          // per x: D[x] N1 over r
        Ten S2 = ws_tensor("sumqtg", {n2, n3, m1, n2, n3, gs});    // . Y over (b, p)
        Ten S3 = ws_tensor("umntg", {n3, m1, m2, n3, gs});         // . N2 over (q, s)
        for (long long x = 0; x < n0 && (c.side_mask & 2); ++x) {
            Ten Dx = Ten::make(D.p + x * (n1 * n2 * n3 * a), "rsub", {n1, n2, n3, a});
            contract(Dx, Ns[0].as("mpr"), S1);
            contract(S1, Y.as("bpqtg"), S2);
            contract(S2, Ns[1].as("nqs"), S3);
            Ten ox = outS;
            ox.p += x * ox.legs[0].stride;
            ox.legs.erase(ox.legs.begin());
            contract(S3, Ns[2].as("wtu"), ox.as("mnwg"));
        }
        ws_release(mk);
    }
    stage_mark(7);

    // =================== O8 normalise, accumulate ln Z ===================
    const long long nnew = n0 * m1 * m2 * m3 * gs;
    if (c.side_mask != 3 || c.exchange) {
        // Phi / Psi split over two GPUs: this process contracted one half;
        // the caller's exchange (one send / receive pair over NVLink in the binding) completes the other before
        // the norms (with both halves contracted here the callback is an observer of the finished tensors)
        if (!c.exchange) fail(-22, "coarse_grain: one half of the contraction is switched off and no exchange is set");
        const int xrc = c.exchange(c.exchange_user, phi_new, psi_new, nnew, (void *)stream());
        if (xrc != 0) fail(-5, "coarse_grain: the caller's exchange of the Phi / Psi halves failed (status %d)", xrc);
    }
    double *ss = ws_doubles(2);
    sumsq(phi_new, nnew, ss);
    sumsq(psi_new, nnew, ss + 1);
    scale_by_rsqrt(phi_new, nnew, ss);
    scale_by_rsqrt(psi_new, nnew, ss + 1);
    std::vector<double> nv = d2h(ss, 2);
    stage_mark(8);
    TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
    // an uploaded input that no stage consumed (wrong shape for this step) may still be in flight:
    // the caller's host buffers are read during the call only
    if (c.copy_stream) TATRG_CUDA_CHECK(cudaStreamSynchronize(c.copy_stream));
    if (c.pre_timed) {
        float ms = 0;
        if (cudaEventElapsedTime(&ms, c.pre_t0, c.pre_t1) == cudaSuccess) c.h2d_ms = ms;
    }
    if (!(nv[0] > 0) || !(nv[1] > 0) || !std::isfinite(nv[0]) || !std::isfinite(nv[1]))
        fail(-34, "coarse_grain: non-finite or zero norm of the renormalised tensor");
    // ---- commit
    const double lnc = 0.5 * (log(nv[0]) + log(nv[1]));
    c.step += 1;
    c.log_acc += ldexp(1.0, -c.step) * lnc;
    for (int i = 0; i < 4; ++i) c.dims[i] = new_dims[i];
    c.bond = gs;
    c.phi = phi_new;
    c.psi = psi_new;
    c.state_low = !c.state_low;
    c.state_bytes = 2 * new_cap;
    spec[9] = {lnc};
    for (int mu = 0; mu < 3; ++mu) c.sq_hist[direction - 1][mu] = sq_hist_new[mu];
    // the deferred Ritz steps of the isometries ended long ago: collect the spectra S^A..S^D; a solver that did not
    // converge, or kept isometries (tests: the Ritz vectors are wanted as well), leave the rest to resolve_iso_spectra
    for (int i = 0; i < 4; ++i) {
        if (!ritz_deferred[i]) continue;
        TATRG_CUDA_CHECK(cudaStreamSynchronize(c.side[4 + i]));
        if (ritz_back->flag[i] != 0 || c.keep_iso) {
            iso_lazy[i] = true;
            continue;
        }
        spec[2 + i].resize(iso_kk);
        for (int j = 0; j < iso_kk; ++j) spec[2 + i][j] = sqrt(std::max(ritz_back->lam[i][j], 0.0));
    }
    for (int i = 0; i < 10; ++i) c.spec[i] = spec[i];
    for (int i = 0; i < 4; ++i) {
        c.iso_pending[i] = iso_lazy[i];
        c.iso_H[i].clear();
        if (iso_lazy[i]) c.iso_H[i] = d2h(Hkeep[i], (long long)iso_kk * iso_kk);
    }
    for (int i = 0; i < 4; ++i) c.gaps[i] = gaps[i];
    for (int i = 0; i < ST_COUNT; ++i) {
        float ms = 0;
        cudaEventElapsedTime(&ms, c.ev[i], c.ev[i + 1]);
        c.stage_ms[i] = ms;
    }
    if (getenv("TATRG_TRACE")) {
        fprintf(stderr, "tatrg-trace stages (gpu ms / host enqueue ms):");
        for (int i = 0; i < ST_COUNT; ++i) fprintf(stderr, " %d: %.2f / %.2f", i, c.stage_ms[i], 1e3 * (c.host_t[i + 1] - c.host_t[i]));
        fprintf(stderr, "\n");
    }
    if (c.prof) prof_collect();
}

}  // namespace tatrg
