// api.cpp -- the C-ABI of libtatrg (include/tatrg.h): argument checking, the process-global
// context, the caller-owned workspace (bump allocator), error reporting.
#include <math.h>

#include <algorithm>
#include <stdarg.h>
#include <string.h>

#include "../../include/tatrg.h"
#include <stdlib.h>

#include "ctx.h"
#include "sq_iter.h"

namespace tatrg {

Ctx &ctx()
{
    static Ctx c;
    return c;
}

cudaStream_t stream() { return ctx().stream; }
void count_launch(int n) { ctx().launches += n; }
void count_flops(double f) { ctx().flops += f; }

int set_error(int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof(buf), fmt, ap);
    va_end(ap);
    ctx().err = buf;
    return code;
}

void fail(int code, const char *fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof(buf), fmt, ap);
    va_end(ap);
    ctx().err = buf;
    throw Err{code};
}

void trace_mark(const char *label)
{
    static const bool trace = getenv("TATRG_TRACE") != nullptr;
    if (!trace) return;
    Ctx &c = ctx();
    cudaEvent_t e;
    if (cudaEventCreate(&e) != cudaSuccess) return;
    cudaEventRecord(e, c.stream);
    c.tmarks.emplace_back(label, e);
}

int prof_begin(double flops, int big)
{
    Ctx &c = ctx();
    if (!c.prof || (c.prof == 1 && big != 1)) return -1;
    const size_t slot = c.prof_rec.size();
    if (2 * slot + 2 > c.prof_ev.size()) {
        const size_t old = c.prof_ev.size();
        c.prof_ev.resize(old + 1024);
        for (size_t i = old; i < c.prof_ev.size(); ++i)
            if (cudaEventCreate(&c.prof_ev[i]) != cudaSuccess) {
                c.prof_ev.resize(i & ~(size_t)1);
                return -1;
            }
    }
    Ctx::ProfRec rec{c.cur_stage, big, flops, {0, 0, 0, 0, 0}};
    for (int i = 0; i < 5; ++i) rec.shape[i] = c.prof_shape[i];
    c.prof_rec.push_back(rec);
    cudaEventRecord(c.prof_ev[2 * slot], c.stream);
    return (int)slot;
}

void prof_shape(int M, int N, int K, int batch, int ksplit)
{
    Ctx &c = ctx();
    c.prof_shape[0] = M;
    c.prof_shape[1] = N;
    c.prof_shape[2] = K;
    c.prof_shape[3] = batch;
    c.prof_shape[4] = ksplit;
}

void prof_end(int slot)
{
    if (slot < 0) return;
    Ctx &c = ctx();
    cudaEventRecord(c.prof_ev[2 * slot + 1], c.stream);
}

void prof_collect()
{
    Ctx &c = ctx();
    static const bool trace = getenv("TATRG_TRACE") != nullptr;   // per-launch GEMM log on stderr
    for (int i = 0; i < ST_COUNT; ++i)
        for (int j = 0; j < 2; ++j) c.gemm_ms[i][j] = c.gemm_fl[i][j] = 0.0, c.gemm_n[i][j] = 0;
    for (size_t i = 0; i < c.prof_rec.size(); ++i) {
        float ms = 0;
        if (cudaEventElapsedTime(&ms, c.prof_ev[2 * i], c.prof_ev[2 * i + 1]) != cudaSuccess) continue;
        const Ctx::ProfRec &r = c.prof_rec[i];
        if (r.stage < 0 || r.stage >= ST_COUNT) continue;
        if (trace)
            fprintf(stderr, "tatrg-trace stage %d tile %d M %d N %d K %d batch %d ksplit %d ms %.4f tflops %.2f\n", r.stage,
                    r.big, r.shape[0], r.shape[1], r.shape[2], r.shape[3], r.shape[4], ms, r.flops / (ms * 1e-3) / 1e12);
        c.gemm_ms[r.stage][r.big] += ms;
        c.gemm_fl[r.stage][r.big] += r.flops;
        c.gemm_n[r.stage][r.big] += 1;
    }
    c.prof_rec.clear();
    if (trace && !c.tmarks.empty()) {
        for (size_t i = 1; i < c.tmarks.size(); ++i) {
            float ms = 0;
            cudaEventElapsedTime(&ms, c.tmarks[i - 1].second, c.tmarks[i].second);
            fprintf(stderr, "tatrg-trace mark %-28s %.3f ms\n", c.tmarks[i].first.c_str(), ms);
        }
        for (auto &m : c.tmarks) cudaEventDestroy(m.second);
        c.tmarks.clear();
    }
    if (trace) {
        fprintf(stderr, "tatrg-trace host: %lld tensor_gemm calls, %.3f ms on the host (%.2f us each)\n", c.host_contract_n,
                1e3 * c.host_contract_s, c.host_contract_n ? 1e6 * c.host_contract_s / c.host_contract_n : 0.0);
        c.host_contract_s = 0;
        c.host_contract_n = 0;
    }
}

void *ws_alloc(size_t bytes)
{
    Ctx &c = ctx();
    if (!c.ws) fail(TATRG_ESTATE, "no workspace set (tatrg_set_workspace)");
    size_t b = (bytes + 255) & ~(size_t)255;
    if (c.lo + b > c.hi)
        fail(TATRG_ENOMEM, "workspace too small: need %zu more bytes (scratch %zu of %zu in use)", b, c.lo,
             c.ws_bytes);
    void *p = c.ws + c.lo;
    c.lo += b;
    size_t used = c.lo + (c.ws_bytes - c.hi);
    if (used > c.peak) c.peak = used;
    return p;
}

double *ws_doubles(long long n) { return (double *)ws_alloc(sizeof(double) * (size_t)(n > 0 ? n : 1)); }
size_t ws_mark() { return ctx().lo; }
void ws_release(size_t mark) { ctx().lo = mark; }

namespace {

// scratch region for the stand-alone entry points (tests, roofline measurements)
void scratch_begin()
{
    Ctx &c = ctx();
    if (!c.ws) fail(TATRG_ESTATE, "no workspace set (tatrg_set_workspace)");
    if (c.inited) {
        c.lo = c.state_low ? c.state_bytes : 0;
        c.hi = c.state_low ? c.ws_bytes : c.ws_bytes - c.state_bytes;
    } else {
        c.lo = 0;
        c.hi = c.ws_bytes;
    }
}

template <class F>
int guarded(F f)
{
    try {
        f();
        return TATRG_OK;
    } catch (const Err &e) {
        cudaDeviceSynchronize();   // nothing of a failed call (side streams included) is left in flight
        cudaGetLastError();
        return e.code;
    } catch (const std::exception &e) {
        return set_error(TATRG_ENUM, "exception: %s", e.what());
    }
}

Map4 map_from(const int64_t *m)
{
    Map4 r;
    r.n0 = m[0] > 0 ? (unsigned)m[0] : TATRG_RADIX_INF;
    r.n1 = m[1] > 0 ? (unsigned)m[1] : TATRG_RADIX_INF;
    r.n2 = m[2] > 0 ? (unsigned)m[2] : TATRG_RADIX_INF;
    r.pad = 0;
    r.s0 = m[3];
    r.s1 = m[4];
    r.s2 = m[5];
    r.s3 = m[6];
    return r;
}

}  // namespace
}  // namespace tatrg

using namespace tatrg;

extern "C" {

int init_ising_tensor(double beta, double h)
{
    return guarded([&] { do_init(beta, h); });
}

int coarse_grain(int direction, int chi, int r, int q, uint64_t seed)
{
    int rc = guarded([&] { do_coarse_grain(direction, chi, r, q, seed, 0); });
    for (auto &i : ctx().in) i = Input();
    return rc;
}

int coarse_grain_atrg(int direction, int chi, int r, int q, uint64_t seed)
{
    int rc = guarded([&] { do_coarse_grain(direction, chi, r, q, seed, 1); });
    for (auto &i : ctx().in) i = Input();
    return rc;
}

double log_Z_per_site(void)
{
    double v = NAN;
    guarded([&] { v = do_log_z(); });
    return v;
}

int tatrg_set_stream(void *cuda_stream)
{
    ctx().stream = (cudaStream_t)cuda_stream;
    return TATRG_OK;
}

int tatrg_set_workspace(void *dev_ptr, size_t bytes)
{
    Ctx &c = ctx();
    if (!dev_ptr || ((uintptr_t)dev_ptr & 255) || bytes < 4096) return set_error(TATRG_EINVAL, "workspace must be a 256-byte aligned device buffer of >= 4096 bytes");
    c.ws = (char *)dev_ptr;
    c.ws_bytes = bytes & ~(size_t)255;
    c.lo = 0;
    c.hi = c.ws_bytes;
    c.inited = false;   // the state lived in the old workspace
    c.peak = 0;
    return TATRG_OK;
}

static double workspace_doubles(int chi, int r)
{
    // steady state, all legs = chi, in units of u = chi^5 doubles: two generations of the state (4 u),
    // A, D (2 u), X sigma, Y (2 u), Y sigma (1 u) persist.  The largest transient sits on top of the first
    // 8 u: the reduced bond swap (Q1_A, Q1_D, the r u sketch: 2.5 + r), or, when the reduced operator
    // does not apply (ill-conditioned matricisation), the plain swap (sketch + two RSVD blocks + copies:
    // 3.5 r) -- the latter is provisioned only while it costs less than 40 GB; beyond that a plain-swap
    // fallback in the steady state fails with TATRG_ENOMEM.  The canonical form (3-4 u on 6 u) and the
    // slabbed contraction (<= 1.1e9 doubles on 9 u) need less.  Plus the chi^4-sized triad / Gram /
    // squeezer intermediates.
    const double c5 = pow((double)chi, 5), c4 = pow((double)chi, 4);
    const double swap_u = (c5 * 3.5 * r * 8.0 < 40e9) ? std::max(3.5 * r, 2.5 + r) : 2.5 + r;
    return c5 * (8.0 + swap_u) + std::min(c5 * r * (1.0 + r), 1.1e9) + c4 * (12.0 * r * r + 40) + (1 << 23);
}

size_t tatrg_workspace_bytes(int chi, int r)
{
    if (chi < 1 || r < 1) return 0;
    return (size_t)(workspace_doubles(chi, r) * 8.0 * 1.05) + ((size_t)64 << 20);
}

size_t tatrg_workspace_bytes_atrg(int chi, int r)
{
    if (chi < 1 || r < 1) return 0;
    const double c6 = pow((double)chi, 6);   // the chi^6 slices of the plain ATRG contraction
    return (size_t)((workspace_doubles(chi, r) + 2.2 * c6) * 8.0 * 1.05) + ((size_t)64 << 20);
}

size_t tatrg_workspace_peak(void) { return ctx().peak; }

int tatrg_set_sketch(int which, const double *data, size_t n, int on_device)
{
    if (which < 0 || which > 8) return set_error(TATRG_EINVAL, "tatrg_set_sketch: which must be 0..8");
    Input &i = ctx().in[which];
    i.ptr = data;
    i.n = data ? n : 0;
    i.on_device = on_device;
    return TATRG_OK;
}

int tatrg_sketch_shape(int which, int direction, int chi, int r, int64_t *rows, int64_t *cols)
{
    Ctx &c = ctx();
    if (!c.inited || which < 0 || which > 8 || direction < 1 || direction > 4 || !rows || !cols)
        return set_error(TATRG_EINVAL, "tatrg_sketch_shape: bad arguments or not initialised");
    int perm[4];
    perm[0] = direction - 1;
    for (int i = 0, j = 1; i < 4; ++i)
        if (i != direction - 1) perm[j++] = i;
    int64_t n0 = c.dims[perm[0]], n1 = c.dims[perm[1]], n2 = c.dims[perm[2]], n3 = c.dims[perm[3]];
    int64_t a = c.bond, nT = n1 * n2 * n3, rc = (int64_t)r * chi;
    *rows = *cols = 0;
    if (which == 0) {
        *rows = a * nT;
        *cols = rc < a * nT ? rc : a * nT;
    } else if (which <= 4) {
        if (rc < n1 * n2) {
            *rows = n1 * n2;
            *cols = rc;
        }
    } else if (which == 5) {
        *rows = n0 * nT;
        *cols = a;
    } else {
        int64_t nn = which == 6 ? n1 : which == 7 ? n2 : n3;
        *rows = nn * nn;
        *cols = chi < nn * nn ? chi : nn * nn;
    }
    return TATRG_OK;
}

int tatrg_get_spectrum(int which, double *host_out, int cap)
{
    if (which < 0 || which > 9 || !host_out) return set_error(TATRG_EINVAL, "tatrg_get_spectrum: bad arguments");
    if (which >= 2 && which <= 5 && ctx().iso_pending[which - 2]) {
        int rc = guarded([&] { resolve_iso_spectra(); });
        if (rc != TATRG_OK) return rc;
    }
    const std::vector<double> &s = ctx().spec[which];
    int n = (int)s.size() < cap ? (int)s.size() : cap;
    for (int i = 0; i < n; ++i) host_out[i] = s[i];
    return n;
}

int tatrg_set_routes(int mask)
{
    if (mask < 0 || mask > 63) return set_error(TATRG_EINVAL, "tatrg_set_routes: mask must be in 0..63");
    ctx().routes = mask;
    return TATRG_OK;
}

int tatrg_set_side_split(int sides, void *exchange_fn, void *user)
{
    if (sides < 1 || sides > 3) return set_error(TATRG_EINVAL, "tatrg_set_side_split: sides must be 1 (Phi), 2 (Psi) or 3 (both)");
    if (sides != 3 && !exchange_fn)
        return set_error(TATRG_EINVAL, "tatrg_set_side_split: computing one half needs an exchange that supplies the other");
    ctx().side_mask = sides;
    ctx().exchange = reinterpret_cast<int (*)(void *, double *, double *, long long, void *)>(exchange_fn);
    ctx().exchange_user = exchange_fn ? user : nullptr;
    return TATRG_OK;
}

int tatrg_keep_isometries(int on)
{
    ctx().keep_iso = on != 0;
    if (!on)
        for (auto &v : ctx().iso) v.clear();
    return TATRG_OK;
}

int tatrg_get_isometry(int which, double *host_out, size_t cap, int *rows, int *cols)
{
    Ctx &c = ctx();
    if (which < 0 || which > 3) return set_error(TATRG_EINVAL, "tatrg_get_isometry: which must be 0..3 (A, X, Y, D)");
    if (c.iso_pending[which]) {
        int rc = guarded([&] { resolve_iso_spectra(); });
        if (rc != TATRG_OK) return rc;
    }
    const std::vector<double> &v = c.iso[which];
    if (v.empty()) return set_error(TATRG_ESTATE, "tatrg_get_isometry: nothing kept (tatrg_keep_isometries(1) before the step; Triad-ATRG steps only)");
    if (rows) *rows = c.iso_rows;
    if (cols) *cols = c.iso_cols;
    if (host_out) {
        if (cap < v.size()) return set_error(TATRG_EINVAL, "tatrg_get_isometry: need %zu doubles", v.size());
        memcpy(host_out, v.data(), v.size() * sizeof(double));
    }
    return TATRG_OK;
}

int tatrg_get_gaps(double out[4])
{
    for (int i = 0; i < 4; ++i) out[i] = ctx().gaps[i];
    return TATRG_OK;
}

int tatrg_get_dims(int dims_out[6])
{
    Ctx &c = ctx();
    if (!c.inited) return set_error(TATRG_ESTATE, "not initialised");
    for (int i = 0; i < 4; ++i) dims_out[i] = c.dims[i];
    dims_out[4] = c.bond;
    dims_out[5] = c.step;
    return TATRG_OK;
}

int tatrg_get_tensors(double *phi_out, double *psi_out, size_t cap_each)
{
    Ctx &c = ctx();
    if (!c.inited) return set_error(TATRG_ESTATE, "not initialised");
    size_t n = (size_t)c.dims[0] * c.dims[1] * c.dims[2] * c.dims[3] * c.bond;
    if (cap_each < n) return set_error(TATRG_EINVAL, "tatrg_get_tensors: need %zu doubles each", n);
    return guarded([&] {
        TATRG_CUDA_CHECK(cudaMemcpyAsync(phi_out, c.phi, n * 8, cudaMemcpyDeviceToHost, c.stream));
        TATRG_CUDA_CHECK(cudaMemcpyAsync(psi_out, c.psi, n * 8, cudaMemcpyDeviceToHost, c.stream));
        TATRG_CUDA_CHECK(cudaStreamSynchronize(c.stream));
    });
}

double tatrg_order_parameter(int leg)
{
    double v = NAN;
    guarded([&] { v = do_order_parameter(leg); });
    return v;
}

static const char *kStageNames[ST_COUNT] = {"canonical_form", "bond_swap",  "isometries", "triad_tensors",
                                            "gram_chains",    "squeezers",  "contraction", "normalise"};

int tatrg_get_stage_ms(double *host_out, int cap)
{
    int n = ST_COUNT < cap ? ST_COUNT : cap;
    for (int i = 0; i < n; ++i) host_out[i] = ctx().stage_ms[i];
    return ST_COUNT;
}

int tatrg_set_profile(int on)
{
    ctx().prof = on < 0 ? 0 : (on > 2 ? 2 : on);
    ctx().prof_rec.clear();
    return TATRG_OK;
}

int tatrg_get_gemm_profile(double *host_out, int cap)
{
    Ctx &c = ctx();
    int k = 0;
    for (int i = 0; i < ST_COUNT; ++i)
        for (int j = 0; j < 2; ++j) {
            if (k + 3 > cap) return k;
            host_out[k++] = c.gemm_ms[i][j];
            host_out[k++] = c.gemm_fl[i][j];
            host_out[k++] = (double)c.gemm_n[i][j];
        }
    return k;
}

int tatrg_get_h2d(double *ms_out, size_t *bytes_out)
{
    if (ms_out) *ms_out = ctx().h2d_ms;
    if (bytes_out) *bytes_out = ctx().h2d_bytes;
    return TATRG_OK;
}

const char *tatrg_stage_name(int i) { return (i >= 0 && i < ST_COUNT) ? kStageNames[i] : ""; }

long long tatrg_launch_count(int reset)
{
    long long v = ctx().launches;
    if (reset) ctx().launches = 0;
    return v;
}

double tatrg_gemm_flops(int reset)
{
    double v = ctx().flops;
    if (reset) ctx().flops = 0;
    return v;
}

double tatrg_probe_fp64_peak(int mode, int iters)
{
    double v = -1.0;
    guarded([&] {
        if (mode < 0 || mode > 2 || iters < 1) fail(TATRG_EINVAL, "tatrg_probe_fp64_peak: bad arguments");
        scratch_begin();
        v = probe_fp64_peak(mode, iters);
    });
    return v;
}

int tatrg_tensor_gemm(const double *A, const double *B, double *C, int M, int N, int K, int batch,
                      const int64_t *maps, double alpha, int accumulate)
{
    return guarded([&] {
        if (!A || !B || !C || !maps || M < 0 || N < 0 || K < 1 || batch < 1) fail(TATRG_EINVAL, "tatrg_tensor_gemm: bad arguments");
        scratch_begin();
        GemmParams p;
        memset(&p, 0, sizeof(p));
        p.A = A;
        p.B = B;
        p.C = C;
        p.M = M;
        p.N = N;
        p.K = K;
        p.batch = batch;
        p.am = map_from(maps + 0);
        p.ak = map_from(maps + 7);
        p.bk = map_from(maps + 14);
        p.bn = map_from(maps + 21);
        p.cm = map_from(maps + 28);
        p.cn = map_from(maps + 35);
        p.ab = map_from(maps + 42);
        p.bb = map_from(maps + 49);
        p.cb = map_from(maps + 56);
        p.alpha = alpha;
        p.accumulate = accumulate & 1;
        p.tri_b = (accumulate & 2) ? 1 : 0;
        p.a_kfast = llabs(p.ak.s0) < llabs(p.am.s0) || p.am.s0 == 0;
        p.b_kfast = llabs(p.bk.s0) < llabs(p.bn.s0) || p.bn.s0 == 0;
        tensor_gemm(p);
    });
}

extern "C" uint64_t si_subseed(uint64_t seed, uint64_t step, uint64_t which);

int tatrg_fill_gauss(double *out, uint64_t n, uint64_t seed, uint64_t step, uint64_t which)
{
    return guarded([&] {
        if (!out && n) fail(TATRG_EINVAL, "tatrg_fill_gauss: null pointer");
        device_fill_gauss(out, n, si_subseed(seed, step, which));
    });
}

int tatrg_qr_pos(double *Y, int64_t m, int n, double *R)
{
    return guarded([&] {
        if (!Y || !R || m < n) fail(TATRG_EINVAL, "tatrg_qr_pos: need m >= n >= 1");
        scratch_begin();
        tsqr(Y, m, n, R);
    });
}

int tatrg_cholesky(double *A, int n, double shift_rel, double *Linv)
{
    bool ok = false;
    int rc = guarded([&] {
        if (!A || n < 1) fail(TATRG_EINVAL, "tatrg_cholesky: need A and n >= 1");
        scratch_begin();
        ok = cholesky_lower(A, n, shift_rel, Linv);
    });
    return rc < 0 ? rc : (ok ? 0 : 1);
}

int tatrg_cholqr(double *Y, int64_t m, int n, int passes, double shift_rel, double *R)
{
    int h = 0;
    int rc = guarded([&] {
        if (!Y || m < n || n < 1) fail(TATRG_EINVAL, "tatrg_cholqr: need m >= n >= 1");
        scratch_begin();
        int *flag = (int *)ws_alloc(sizeof(int));
        TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(int), stream()));
        cholqr_async(Y, m, n, passes, shift_rel, flag, nullptr, R);
        TATRG_CUDA_CHECK(cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
        TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
    });
    return rc < 0 ? rc : (h ? 1 : 0);
}

int tatrg_subspace_iteration(const double *F, int n, const double *start, double *Q, double *Qt, int iters, int grid,
                             double *R, double *minmax)
{
    int h = 0;
    int rc = guarded([&] {
        if (!F || !start || !Q || !Qt || n < 64 || iters < 1 || 2 * iters + 2 > SQ_MAXSTEPS || grid < 1)
            fail(TATRG_EINVAL, "tatrg_subspace_iteration: need F, start, Q, Qt, n >= 64, 1 <= iters <= %d, grid >= 1", SQ_MAXSTEPS / 2 - 1);
        scratch_begin();
        int *flag = (int *)ws_alloc(sizeof(int));
        TATRG_CUDA_CHECK(cudaMemsetAsync(flag, 0, sizeof(int), stream()));
        SqIterParams p{};
        double *Ft = ws_doubles((long long)n * n);
        transpose_small(F, Ft, n, n);
        p.F = F;
        p.Ft = Ft;
        p.start = start;
        p.buf[0] = Q;
        p.buf[1] = Qt;
        p.Rout = R;
        p.ratio = ws_doubles(4);
        p.flag = flag;
        p.shift = 1e-13;
        p.N2 = n;
        int ns = 0;
        p.steps[ns++] = SQ_FROM_START;
        for (int it = 0; it < iters; ++it) {
            p.steps[ns++] = SQ_TRANS;
            p.steps[ns++] = it == iters - 1 ? (SQ_TWO_PASSES | (1 << SQ_RATIO_SHIFT)) : 0;
        }
        p.steps[ns++] = SQ_TRANS | SQ_TWO_PASSES | (2 << SQ_RATIO_SHIFT) | SQ_WANT_R;
        p.nsteps = ns;
        sq_iter_launch(p, grid, ws_doubles((long long)sq_iter_scratch_doubles(sq_iter_grid(n, grid))));
        if (minmax) TATRG_CUDA_CHECK(cudaMemcpyAsync(minmax, p.ratio, 4 * sizeof(double), cudaMemcpyDeviceToDevice, stream()));
        TATRG_CUDA_CHECK(cudaMemcpyAsync(&h, flag, sizeof(int), cudaMemcpyDeviceToHost, stream()));
        TATRG_CUDA_CHECK(cudaStreamSynchronize(stream()));
    });
    return rc < 0 ? rc : (h ? 1 : 0);
}

int tatrg_jacobi_svd(double *G, int m, int n, double *V, double *s)
{
    return guarded([&] {
        if (!G || !V || !s) fail(TATRG_EINVAL, "tatrg_jacobi_svd: null pointer");
        scratch_begin();
        jacobi_svd(G, m, n, V, s, 1, 0, 0, 0);
    });
}

int tatrg_sumsq(const double *x, int64_t n, double *out_dev)
{
    return guarded([&] {
        scratch_begin();
        sumsq(x, n, out_dev);
    });
}

int tatrg_sumsq_static(const double *x, int64_t n, double *out_dev)
{
    return guarded([&] {
        if (!out_dev || n < 0 || (n > 0 && !x)) fail(TATRG_EINVAL, "tatrg_sumsq_static: need out_dev, n >= 0 and x for n > 0");
        if (n > (int64_t)TATRG_SUMSQ_STATIC_MAX_N)
            fail(TATRG_EINVAL, "tatrg_sumsq_static: n = %lld exceeds the maximum of %lld elements", (long long)n,
                 (long long)TATRG_SUMSQ_STATIC_MAX_N);
        sumsq_static(x, n, out_dev);
    });
}

int tatrg_dot(const double *x, const double *y, int64_t n, double *out_dev)
{
    return guarded([&] {
        scratch_begin();
        dot(x, y, n, out_dev);
    });
}

int tatrg_scale_by_rsqrt(double *x, int64_t n, const double *sumsq_dev)
{
    return guarded([&] { scale_by_rsqrt(x, n, sumsq_dev); });
}

const char *tatrg_last_error(void) { return ctx().err.c_str(); }

void tatrg_destroy(void)
{
    Ctx &c = ctx();
    if (c.ev_ok)
        for (auto &e : c.ev) cudaEventDestroy(e);
    for (auto &e : c.prof_ev) cudaEventDestroy(e);
    if (c.side_ok) {
        for (auto &st : c.side) cudaStreamDestroy(st);
        for (auto &e : c.join_ev) cudaEventDestroy(e);
        for (auto &e : c.dep_ev) cudaEventDestroy(e);
        cudaEventDestroy(c.fork_ev);
    }
    if (c.copy_stream) {
        cudaStreamDestroy(c.copy_stream);
        for (auto &e : c.pre_ev) cudaEventDestroy(e);
        cudaEventDestroy(c.pre_t0);
        cudaEventDestroy(c.pre_t1);
    }
    if (c.pinned) cudaFreeHost(c.pinned);
    c = Ctx();
}

}  // extern "C"
