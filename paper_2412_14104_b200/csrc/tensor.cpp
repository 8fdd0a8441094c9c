// tensor.cpp -- leg bookkeeping: classifies the legs of a pairwise contraction into
// (batch, rows, columns, summed), orders them by the operand's memory stride (so that the
// kernel's loader walks the contiguous leg), merges legs that are adjacent in every tensor
// involved, and emits the mixed-radix maps of one tensor_gemm launch.
#include "ctx.h"

#include <chrono>

#include <algorithm>
#include <string.h>

namespace tatrg {

Ten Ten::make(double *p, const char *names, std::initializer_list<long long> dims)
{
    Ten t;
    t.p = p;
    size_t n = strlen(names);
    if (n != dims.size()) fail(-22, "Ten::make: %s has %zu names for %zu dims", names, n, dims.size());
    std::vector<long long> d(dims);
    long long s = 1;
    t.legs.resize(n);
    for (int i = (int)n - 1; i >= 0; --i) {
        t.legs[i] = Leg{names[i], d[i], s};
        s *= d[i];
    }
    return t;
}

Ten Ten::as(const char *names) const
{
    if (strlen(names) != legs.size()) fail(-22, "Ten::as: %s for %zu legs", names, legs.size());
    Ten t = *this;
    for (size_t i = 0; i < legs.size(); ++i) t.legs[i].name = names[i];
    return t;
}

long long Ten::dim(char c) const
{
    for (auto &l : legs)
        if (l.name == c) return l.n;
    fail(-22, "Ten::dim: no leg %c", c);
}

Ten ws_tensor(const char *names, std::initializer_list<long long> dims)
{
    long long s = 1;
    for (auto d : dims) s *= d;
    return Ten::make(ws_doubles(s > 0 ? s : 1), names, dims);
}

namespace {

struct GLeg {
    long long n;
    long long s[3];  // strides in up to three tensors (unused = 0)
};

const Leg *find(const Ten &t, char c)
{
    for (auto &l : t.legs)
        if (l.name == c) return &l;
    return nullptr;
}

// sort by stride in tensor `key`, drop size-1 legs, merge legs adjacent in all `nt` tensors
void canon(std::vector<GLeg> &g, int key, int nt)
{
    std::vector<GLeg> v;
    for (auto &l : g)
        if (l.n != 1) v.push_back(l);
    std::stable_sort(v.begin(), v.end(), [key](const GLeg &a, const GLeg &b) { return a.s[key] < b.s[key]; });
    std::vector<GLeg> out;
    for (auto &l : v) {
        if (!out.empty()) {
            GLeg &o = out.back();
            bool ok = true;
            for (int t = 0; t < nt; ++t) ok = ok && (l.s[t] == o.s[t] * o.n);
            if (ok) {
                o.n *= l.n;
                continue;
            }
        }
        out.push_back(l);
    }
    g = out;
}

Map4 to_map(const std::vector<GLeg> &g, int t, const char *what)
{
    if (g.size() > 4) fail(-22, "contract: %s index needs %zu levels (max 4)", what, g.size());
    Map4 m = map1(0);
    long long s[4] = {0, 0, 0, 0};
    unsigned n[3] = {TATRG_RADIX_INF, TATRG_RADIX_INF, TATRG_RADIX_INF};
    for (size_t i = 0; i < g.size(); ++i) {
        s[i] = g[i].s[t];
        if (i < 3 && i + 1 < g.size()) n[i] = (unsigned)g[i].n;
    }
    m.n0 = n[0];
    m.n1 = n[1];
    m.n2 = n[2];
    m.s0 = s[0];
    m.s1 = s[1];
    m.s2 = s[2];
    m.s3 = s[3];
    return m;
}

long long total(const std::vector<GLeg> &g)
{
    long long s = 1;
    for (auto &l : g) s *= l.n;
    return s;
}

}  // namespace

void contract(const Ten &A, const Ten &B, const Ten &C, double alpha, bool accumulate, bool lower_only, bool tri_b)
{
    std::vector<GLeg> gb, gm, gn, gk;  // strides: batch (A,B,C); m (A,C); n (B,C); k (A,B)
    std::string seen;
    auto visit = [&](char c) {
        if (seen.find(c) != std::string::npos) return;
        seen.push_back(c);
        const Leg *a = find(A, c), *b = find(B, c), *cc = find(C, c);
        long long n = a ? a->n : (b ? b->n : cc->n);
        if ((a && a->n != n) || (b && b->n != n) || (cc && cc->n != n))
            fail(-22, "contract: leg %c has inconsistent sizes", c);
        if (a && b && cc)
            gb.push_back(GLeg{n, {a->stride, b->stride, cc->stride}});
        else if (a && cc)
            gm.push_back(GLeg{n, {a->stride, cc->stride, 0}});
        else if (b && cc)
            gn.push_back(GLeg{n, {b->stride, cc->stride, 0}});
        else if (a && b)
            gk.push_back(GLeg{n, {a->stride, b->stride, 0}});
        else
            fail(-22, "contract: leg %c appears in one tensor only", c);
    };
    for (auto &l : A.legs) visit(l.name);
    for (auto &l : B.legs) visit(l.name);
    for (auto &l : C.legs) visit(l.name);
    canon(gb, 2, 3);
    canon(gm, 0, 2);
    canon(gn, 0, 2);
    canon(gk, 0, 2);

    GemmParams p;
    memset(&p, 0, sizeof(p));
    p.A = A.p;
    p.B = B.p;
    p.C = C.p;
    long long M = total(gm), N = total(gn), K = total(gk), Bt = total(gb);
    if (M <= 64 && N > 64 && !lower_only) {   // the wide index goes to the 128-row side of the CTA tile
        contract(B, A, C, alpha, accumulate);
        return;
    }
    if (M > 0x7fffffff || N > 0x7fffffff || K > 0x7fffffff || Bt > 65535)
        fail(-22, "contract: index range too large (M=%lld N=%lld K=%lld batch=%lld)", M, N, K, Bt);
    p.M = (int)M;
    p.N = (int)N;
    p.K = (int)K;
    p.batch = (int)Bt;
    p.am = to_map(gm, 0, "row");
    p.cm = to_map(gm, 1, "row");
    p.bn = to_map(gn, 0, "column");
    p.cn = to_map(gn, 1, "column");
    p.ak = to_map(gk, 0, "summed");
    p.bk = to_map(gk, 1, "summed");
    p.ab = to_map(gb, 0, "batch");
    p.bb = to_map(gb, 1, "batch");
    p.cb = to_map(gb, 2, "batch");
    p.alpha = alpha;
    p.accumulate = accumulate ? 1 : 0;
    p.lower_only = (lower_only && M == N) ? 1 : 0;
    p.tri_b = tri_b ? 1 : 0;
    // loader order: walk whichever index has the smaller leading stride in that operand
    long long am0 = gm.empty() ? (1LL << 60) : gm[0].s[0];
    long long ak0 = gk.empty() ? (1LL << 60) : gk[0].s[0];
    p.a_kfast = ak0 < am0;
    long long bn0 = gn.empty() ? (1LL << 60) : gn[0].s[0];
    long long bk0 = gk.empty() ? (1LL << 60) : gk[0].s[1];
    p.b_kfast = bk0 < bn0;
    const auto t0 = std::chrono::steady_clock::now();
    tensor_gemm(p);
    Ctx &c = ctx();
    c.host_contract_s += std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    c.host_contract_n += 1;
}

}  // namespace tatrg
