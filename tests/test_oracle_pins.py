"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these retype the oracle's formulas: they compare it with exact enumeration, Onsager's
solution, the high-temperature series, brute-force einsum of the paper's defining equations,
LAPACK dense SVD, and invariants the paper states (isometries PAPER.md:37, :41; r*chi >= d2*d3
=> ATRG).
"""
import numpy as np
import pytest

from exact_refs import brute_force_lnZ, ht_series_lnZ, onsager_lnZ
from oracle import driver
from oracle import tatrg_oracle as orc

BETA = 1.0 / 6.0


# ------------------------------------------------------------------ golden values (P2-values)
def _golden():
    out = {}
    import os
    with open(os.path.join(os.path.dirname(__file__), "golden", "enumeration_beta_1_6.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            ext, h, val = line.split()
            out[(tuple(int(c) for c in ext.split("x")), float(h))] = float(val)
    return out


def test_enumeration_reproduces_survey_values():
    """SURVEY.md 8(c) 'P2-values' were computed by an independent spin sum; ours must agree."""
    for (ext, h), val in _golden().items():
        assert abs(brute_force_lnZ(BETA, h, ext) - val) < 2e-15 * 16


def test_ring_closed_form():
    """(4,1,1,1): 4-site ring with three self bonds per site, Z = e^{12b}((2cosh b)^4+(2sinh b)^4)."""
    z = np.exp(12 * BETA) * ((2 * np.cosh(BETA)) ** 4 + (2 * np.sinh(BETA)) ** 4)
    assert abs(np.exp(4 * brute_force_lnZ(BETA, 0.0, (4, 1, 1, 1))) / z - 1) < 1e-13


def test_W_reading_G1():
    """Eq. 17 as printed gives (W W^T) = (cosh 2b, 1); with the square roots restored it is
    (e^b, e^-b) (reading G1)."""
    st = orc.init_ising_tensor(0.3, 0.0, active=(1, 0, 0, 0))
    # 1 leg pair: T[i,j] = sum_a W[a,i] W[a,j]; tTr over a 1-site ring with a self bond: Z = 2 e^b
    assert abs(orc.log_Z_per_site(st) - np.log(2 * np.exp(0.3))) < 1e-14


# ------------------------------------------------------------------ P2: exact enumeration
@pytest.mark.parametrize("h", [0.0, 0.01])
@pytest.mark.parametrize("dirs,ext", [
    ([1], (2, 1, 1, 1)), ([2], (1, 2, 1, 1)), ([3], (1, 1, 2, 1)), ([4], (1, 1, 1, 2)),
    ([1, 2], (2, 2, 1, 1)), ([2, 1], (2, 2, 1, 1)), ([3, 4], (1, 1, 2, 2)), ([4, 2], (1, 2, 1, 2)),
    ([1, 1], (4, 1, 1, 1)), ([3, 3], (1, 1, 4, 1)),
])
def test_P2_tiny_lattices(h, dirs, ext):
    st = driver.run(BETA, h, 16, 2, 2, len(dirs), 7, directions=dirs)
    assert abs(orc.log_Z_per_site(st) / brute_force_lnZ(BETA, h, ext) - 1) < 1e-12


@pytest.mark.parametrize("mode", ["triad", "atrg"])
def test_P2prime_partial_trace_closure(mode):
    """Lattice (2,2,2,1): two untruncated steps (dirs 1,2), then Z = Tr(A~^2) with the
    partial-trace matrix of PAPER.md:177 (open leg moved to direction 3)."""
    st = driver.run(BETA, 0.01, 16, 2, 2, 2, 7, directions=[1, 2], mode=mode)
    g = st.phi.shape[4]
    ph = np.moveaxis(st.phi, 2, 3).reshape(-1, st.phi.shape[2], g)
    ps = np.moveaxis(st.psi, 2, 3).reshape(-1, st.psi.shape[2], g)
    At = np.einsum("xkg,xlg->kl", ph, ps)
    lnz = st.log_acc + np.log(np.trace(At @ At)) / 8.0
    assert abs(lnz / brute_force_lnZ(BETA, 0.01, (2, 2, 2, 1)) - 1) < 1e-12


# ------------------------------------------------------------------ P1: Onsager (d=2 embedding)
@pytest.mark.parametrize("T", [2.0, 3.0])
def test_P1_onsager(T):
    """d=2 run of the same code (legs 2,3 dummy => no (2,3) pair => pure ATRG).  Truncation
    limited: the error must shrink with chi and be <= 1e-6 at chi=16."""
    ex = onsager_lnZ(1 / T)
    err = []
    for chi in (8, 16):
        st = driver.run(1 / T, 0.0, chi, 2, 2, 30, 11, active=(1, 0, 0, 1), directions=[1, 4])
        err.append(abs(orc.log_Z_per_site(st) / ex - 1))
    assert err[1] < err[0] < 1e-5 and err[1] < 1e-6


def test_onsager_matches_2d_series():
    # beta=0.02: the neglected 12 v^10 term is 1e-16
    assert abs(onsager_lnZ(0.02) - ht_series_lnZ(0.02, 2)) < 1e-13


# ------------------------------------------------------------------ P3: high-temperature series
@pytest.mark.parametrize("T", [50.0, 20.0])
def test_P3_high_temperature_4d(T):
    """Infinite-volume path (24 steps, L = 64 per direction: winding loops ~ v^64 vanish).  SURVEY P3:
    series value 0.693948091615655 at T=50 (neglected v^10 term < 1e-12) and 0.698183708674986 at T=20
    (< 1e-8).  The oracle reproduces ln 2 + 4 ln cosh(beta) exactly and loses, by truncation, a fraction of
    the plaquette term 6 v^4 (the first term that needs a bond dimension above 2) that strictly shrinks with
    chi: measured 0.43, 0.21, 0.17 of it at chi = 4, 8, 12 at T=50.  A wrong bond weight, sign or leg
    pairing shows at order v^2 >> 6 v^4."""
    ex = ht_series_lnZ(1 / T, 4)
    assert abs(ex - {50.0: 0.693948091615655, 20.0: 0.698183708674986}[T]) < 1e-14
    plaq = 6 * np.tanh(1 / T) ** 4
    e = [orc.log_Z_per_site(driver.run(1 / T, 0.0, chi, 2, 2, 24, 13)) - ex for chi in (4, 8, 12)]
    assert all(v < 0 for v in e)                       # truncation only removes weight
    assert abs(e[2]) < abs(e[1]) < abs(e[0]) < 0.5 * plaq
    assert abs(e[2]) < 0.2 * plaq
    _P3_ERR[T] = e


_P3_ERR = {}


def test_P3_truncation_error_scales_like_the_plaquette_term():
    """The chi-limited error is a fixed fraction of 6 v^4 at both temperatures (to the next order, v^6):
    e(T=20) / e(T=50) = (tanh(1/20) / tanh(1/50))^4 = 38.9 within 15 % for every chi -- no O(v^2) or O(1)
    piece is wrong."""
    if len(_P3_ERR) < 2:
        pytest.skip("runs after both parametrisations of test_P3_high_temperature_4d")
    ratio = (np.tanh(1 / 20.0) / np.tanh(1 / 50.0)) ** 4
    for a, b in zip(_P3_ERR[20.0], _P3_ERR[50.0]):
        assert abs((a / b) / ratio - 1) < 0.15, (a, b, ratio)


# ------------------------------------------------------------------ helpers for step-level pins
def _mid_state(chi=3, n_steps=3, seed=5, r=1):
    return driver.run(BETA, 0.02, chi, r, 1, n_steps, seed)


def _step_pieces(st, direction, chi, r, q, seed, iso_mode="rsvd", q_iso=None):
    inputs = driver.seeded_inputs_for(seed, st.step)
    perm = orc.frame_perm(direction)
    phi = np.transpose(st.phi, perm + [4])
    psi = np.transpose(st.psi, perm + [4])
    n0, n1, n2, n3, _ = phi.shape
    A, sT, D = orc.canonicalise(phi, psi, lambda a: inputs("ref_ad", n0 * n1 * n2 * n3, a))
    a = len(sT)
    dim = a * n1 * n2 * n3
    ell = min(r * chi, dim)
    X, sig, Y, _ = orc.bond_swap(A, sT, D, chi, r, q, inputs("swap", dim, ell))
    k = min(r * chi, n1 * n2)
    om = {t: inputs(t, n1 * n2, k) for t in "AXYD"} if k < n1 * n2 else {}
    U, spec = orc.make_isometries(A, X, sig, Y, D, chi, r, q if q_iso is None else q_iso, om, iso_mode)
    return dict(phi=phi, psi=psi, A=A, sT=sT, D=D, X=X, sig=sig, Y=Y, U=U, spec=spec)


def _gamma(p):
    return np.einsum("xpqta,arsug,g,bPQTg,yRSUb->xpqtrsuPQTyRSU",
                     p["A"], p["X"], p["sig"], p["Y"], p["D"], optimize=True)


def _gamma_triad(E, F, G, H, U):
    return np.einsum("xkta,pqk,alug,rsl,bmTg,PQm,ynUb,RSn->xpqtrsuPQTyRSU",
                     E, U["A"], F, U["X"], G, U["Y"], H, U["D"], optimize=True)


# ------------------------------------------------------------------ P4: isometries
def test_P4_isometries_and_projectors():
    st = _mid_state(chi=4, n_steps=5, r=1)
    p = _step_pieces(st, 2, 4, 1, 2, 9)
    for name in ("A", "D"):
        m = p[name].reshape(-1, p[name].shape[4])
        assert np.abs(m.T @ m - np.eye(m.shape[1])).max() < 1e-12
    for name in ("X", "Y"):
        m = p[name].reshape(-1, p[name].shape[4])
        assert np.abs(m.T @ m - np.eye(m.shape[1])).max() < 1e-12
    for t in "AXYD":
        u = p["U"][t].reshape(-1, p["U"][t].shape[2])
        assert u.shape[1] < u.shape[0]          # genuinely oversampled-truncated here
        assert np.abs(u.T @ u - np.eye(u.shape[1])).max() < 1e-12
    E, F, G, H = orc.triad_tensors(p["A"], p["X"], p["sig"], p["Y"], p["D"], p["U"])
    GL, GR = orc.triad_grams(E, F, G, H, p["U"])
    for mu in (1, 2, 3):
        M, N, s, _ = orc.squeezer(GL[mu], GR[mu], 4)
        assert np.abs(N @ M - np.eye(len(s))).max() < 1e-10
        PMN = M @ N
        assert np.abs(PMN @ PMN - PMN).max() < 1e-10
        assert np.all(np.diff(s) <= 0)


def test_canonical_form_is_exact():
    """A sigT D^T reproduces T = Phi Psi^T (reading O2 is exact)."""
    st = _mid_state()
    phi, psi = st.phi, st.psi
    A, sT, D = orc.canonicalise(phi, psi)
    g = phi.shape[4]
    T = phi.reshape(-1, g) @ psi.reshape(-1, g).T
    T2 = (A.reshape(-1, len(sT)) * sT) @ D.reshape(-1, len(sT)).T
    assert np.abs(T - T2).max() < 1e-14


# ------------------------------------------------------------------ P6: RSVD
def test_P6_rsvd_full_width_equals_lapack():
    """l >= rank => RSVD = exact truncated SVD of the dense swap matrix M (LAPACK gesdd)."""
    st = _mid_state(chi=3, n_steps=2)
    phi = st.phi
    A, sT, D = orc.canonicalise(st.phi, st.psi)
    n0, n1, n2, n3, a = A.shape
    nT = n1 * n2 * n3
    Mdense = np.einsum("cJa,cIb->aIbJ", (D * sT).reshape(n0, nT, a), (A * sT).reshape(n0, nT, a))
    Mdense = Mdense.reshape(a * nT, a * nT)
    import seeded_inputs as si
    om = si.gauss_matrix(3, 0, 0, a * nT, a * nT)
    X, s, Y, _ = orc.bond_swap(A, sT, D, 5, a * nT, 0, om)     # r*chi >= dim: full width
    u, s_ref, vt = np.linalg.svd(Mdense)
    assert np.abs(s - s_ref[:5]).max() < 1e-13 * s_ref[0]
    approx = (X.reshape(a * nT, -1) * s) @ Y.reshape(a * nT, -1).T
    best = (u[:, :5] * s_ref[:5]) @ vt[:5]
    assert np.abs(approx - best).max() < 1e-12
    del phi


def test_P6_truncated_bond_swap_meets_eckart_young():
    """The q-loop of `rsvd` with l < rank (what every truncated config runs).  On a dense M small enough
    for LAPACK: (i) || M - X sigma Y^T ||_F is never below the Eckart-Young bound sqrt(sum_{i>chi} s_i^2) and
    falls to it monotonically in q; (ii) the computed singular values approach the exact ones from below;
    (iii) the rate: one iteration = one application of M^T and one of M, so the error of sigma_l shrinks by
    (s_{l+1}/s_l)^4 per iteration -- an iterate with a missing or doubled application has another rate."""
    import seeded_inputs as si
    st = driver.run(BETA, 0.02, 4, 1, 1, 3, 5)
    A, sT, D = orc.canonicalise(st.phi, st.psi)
    n0, n1, n2, n3, a = A.shape
    nT = n1 * n2 * n3
    Md = np.einsum("cJa,cIb->aIbJ", (D * sT).reshape(n0, nT, a), (A * sT).reshape(n0, nT, a)).reshape(a * nT, a * nT)
    s_ref = np.linalg.svd(Md, compute_uv=False)
    assert np.sum(s_ref > 1e-12 * s_ref[0]) > 8            # l = 3 or 8 is well below the rank (64)
    for chi, r in ((4, 2), (3, 1)):
        ell = r * chi
        om = si.gauss_matrix(3, 0, 0, a * nT, ell)
        bound = np.sqrt(np.sum(s_ref[chi:] ** 2))
        errs, devs = [], []
        for q in (0, 1, 2, 4, 8, 30):
            X, s, Y, s_full = orc.bond_swap(A, sT, D, chi, r, q, om)
            assert len(s) == chi and len(s_full) == ell
            approx = (X.reshape(a * nT, -1) * s) @ Y.reshape(a * nT, -1).T
            errs.append(np.linalg.norm(Md - approx))
            devs.append(s_ref[:ell] - s_full)
            assert np.all(devs[-1] > -1e-14 * s_ref[0])    # from below
        assert all(e >= bound * (1 - 1e-13) for e in errs)
        assert all(errs[i + 1] < errs[i] for i in range(4)) and errs[5] <= errs[4] * (1 + 1e-13)
        assert errs[5] / bound - 1 < 1e-13 and errs[0] / bound - 1 > 1e-2
        if r == 1:                                         # l = chi = 3: rate of the last kept value
            rate = (s_ref[ell] / s_ref[ell - 1]) ** 4
            for (i, j, n) in ((1, 2, 1), (2, 3, 2), (3, 4, 4)):     # q = 1->2, 2->4, 4->8
                got = (devs[j][ell - 1] / devs[i][ell - 1]) ** (1.0 / n)
                assert 0.7 * rate < got < 1.4 * rate, (i, j, got, rate)


def test_P6_isometry_rsvd_converges_to_exact():
    """q -> large: the randomized projector U U^T tends to the exact Eq. 3 projector."""
    st = _mid_state(chi=4, n_steps=5, r=1)
    pe = _step_pieces(st, 1, 4, 1, 2, 9, iso_mode="exact")
    err = []
    for q in (0, 2, 8, 30):
        pr = _step_pieces(st, 1, 4, 1, 2, 9, iso_mode="rsvd", q_iso=q)
        ue = pe["U"]["A"].reshape(16, -1)
        ur = pr["U"]["A"].reshape(16, -1)
        err.append(np.abs(ue @ ue.T - ur @ ur.T).max())
    assert err[3] < 1e-6 and err[3] < err[2] < err[1] < err[0]


# ------------------------------------------------------------------ P7: brute-force einsum
def test_P7_gamma_is_the_two_site_tensor():
    """Untruncated swap: Gamma = A X sig Y D (Eq. 1) equals the two original tensors joined
    along direction 0 (upper j0 with lower i0)."""
    st = driver.run(BETA, 0.02, 16, 2, 1, 1, 5)
    p = _step_pieces(st, 3, 64, 2, 1, 9)
    g = p["phi"].shape[4]
    T = np.einsum("xpqtg,yrsug->xpqtyrsu", p["phi"], p["psi"])
    two = np.einsum("xpqtcPQT,crsuyRSU->xpqtrsuPQTyRSU", T, T, optimize=True)
    assert np.abs(_gamma(p) - two).max() < 1e-13 * np.abs(two).max()
    del g


def test_P7_exact_isometry_is_optimal_for_gamma():
    """Eq. 2-3: U^T (exact mode) spans the top-k left singular space of the *full* Gamma
    matricised on the pair legs -- pins the canonical-form reduction (R_X, R_Y)."""
    st = _mid_state(chi=3, n_steps=4)
    p = _step_pieces(st, 1, 3, 1, 1, 9, iso_mode="exact")
    Gm = _gamma(p)
    # axes: x p q t | r s u | P Q T | y R S U
    for name, ax in (("A", (1, 2)), ("X", (4, 5)), ("Y", (7, 8)), ("D", (11, 12))):
        mat = np.moveaxis(Gm, ax, (0, 1)).reshape(Gm.shape[ax[0]] * Gm.shape[ax[1]], -1)
        lam, V = np.linalg.eigh(mat @ mat.T)
        k = p["U"][name].shape[2]
        Pex = V[:, -k:] @ V[:, -k:].T
        u = p["U"][name].reshape(-1, k)
        assert np.abs(u @ u.T - Pex).max() < 1e-9
        np.testing.assert_allclose(p["spec"][name] ** 2, lam[::-1][:k], rtol=1e-9, atol=1e-14)


def test_P7_triad_tensors_grams_and_contraction():
    """Eqs. 4-14 against brute-force einsum on the full 14-leg Gamma^triad at chi=3."""
    st = _mid_state(chi=3, n_steps=4)
    p = _step_pieces(st, 4, 3, 1, 1, 9)
    U = p["U"]
    E, F, G, H = orc.triad_tensors(p["A"], p["X"], p["sig"], p["Y"], p["D"], U)
    Gt = _gamma_triad(E, F, G, H, U)
    # Gamma^triad = Gamma with the four projectors U U^T applied
    Gp = _gamma(p)
    for name, ax in (("A", (1, 2)), ("X", (4, 5)), ("Y", (7, 8)), ("D", (11, 12))):
        Pj = np.einsum("pqk,rsk->pqrs", U[name], U[name])
        Gp = np.moveaxis(np.tensordot(Pj, Gp, axes=([2, 3], list(ax))), (0, 1), ax)
    assert np.abs(Gt - Gp).max() < 1e-13
    GL, GR = orc.triad_grams(E, F, G, H, U)
    # axes of Gt: 0:x 1:p 2:q 3:t | 4:r 5:s 6:u | 7:P 8:Q 9:T | 10:y 11:R 12:S 13:U
    plus = {1: (1, 4), 2: (2, 5), 3: (3, 6)}
    minus = {1: (7, 11), 2: (8, 12), 3: (9, 13)}
    for mu in (1, 2, 3):
        for ax, got in ((plus[mu], GL[mu]), (minus[mu], GR[mu])):
            m = np.moveaxis(Gt, ax, (0, 1))
            m = m.reshape(m.shape[0] * m.shape[1], -1)
            assert np.abs(m @ m.T - got).max() < 1e-13
    Ms, Ns = {}, {}
    for mu in (1, 2, 3):
        Ms[mu], Ns[mu], _, _ = orc.squeezer(GL[mu], GR[mu], 3)
    phi2, psi2 = orc.contract_triad(E, F, G, H, U, Ms, Ns)
    n = 3
    T2 = np.einsum("xpqtrsuPQTyRSU,prm,qsn,tuw,aPR,bQS,cTU->xmnwyabc", Gt,
                   Ms[1].reshape(n, n, -1), Ms[2].reshape(n, n, -1), Ms[3].reshape(n, n, -1),
                   Ns[1].reshape(-1, n, n), Ns[2].reshape(-1, n, n), Ns[3].reshape(-1, n, n),
                   optimize=True)
    got = np.einsum("xmnwg,yabcg->xmnwyabc", phi2, psi2)
    assert np.abs(T2 - got).max() < 1e-12 * np.abs(T2).max()
    # plain ATRG contraction against the same brute force on the un-projected Gamma
    GLa, GRa = orc.atrg_grams(p["A"], p["X"], p["sig"], p["Y"], p["D"])
    Gfull = _gamma(p)
    for mu in (1, 2, 3):
        for ax, got_ in ((plus[mu], GLa[mu]), (minus[mu], GRa[mu])):
            m = np.moveaxis(Gfull, ax, (0, 1))
            m = m.reshape(m.shape[0] * m.shape[1], -1)
            assert np.abs(m @ m.T - got_).max() < 1e-13
        Ms[mu], Ns[mu], _, _ = orc.squeezer(GLa[mu], GRa[mu], 3)
    phi3, psi3 = orc.contract_atrg(p["A"], p["X"], p["sig"], p["Y"], p["D"], Ms, Ns)
    T3 = np.einsum("xpqtrsuPQTyRSU,prm,qsn,tuw,aPR,bQS,cTU->xmnwyabc", Gfull,
                   Ms[1].reshape(n, n, -1), Ms[2].reshape(n, n, -1), Ms[3].reshape(n, n, -1),
                   Ns[1].reshape(-1, n, n), Ns[2].reshape(-1, n, n), Ns[3].reshape(-1, n, n),
                   optimize=True)
    got3 = np.einsum("xmnwg,yabcg->xmnwyabc", phi3, psi3)
    assert np.abs(T3 - got3).max() < 1e-12 * np.abs(T3).max()


def test_P7_squeezer_minimises_eq12():
    """M N is the best rank-chi insertion between Gamma_L and Gamma_R (Eq. 12): with factors
    L^T L = G^L, R R^T = G^R the optimum is the truncated SVD of L R."""
    rng = np.random.default_rng(0)
    L = rng.standard_normal((40, 9))
    R = rng.standard_normal((9, 50))
    M, N, s, _ = orc.squeezer(L.T @ L, R @ R.T, 4)
    u, sv, vt = np.linalg.svd(L @ R)
    np.testing.assert_allclose(s, sv[:4], rtol=1e-10)
    assert np.abs(L @ M @ N @ R - (u[:, :4] * sv[:4]) @ vt[:4]).max() < 1e-10


# ------------------------------------------------------------------ P5: Triad == ATRG
def test_P5_triad_equals_atrg_when_r_chi_covers_pair():
    """r = chi (here r*chi >= d2*d3) => Triad-ATRG is the ATRG."""
    a = driver.run(BETA, 0.0, 4, 4, 2, 8, 3, mode="triad")
    b = driver.run(BETA, 0.0, 4, 4, 2, 8, 3, mode="atrg")
    assert abs(orc.log_Z_per_site(a) / orc.log_Z_per_site(b) - 1) < 1e-12
    c = driver.run(BETA, 0.0, 4, 2, 2, 8, 3, mode="triad")       # r*chi = 8 < 16: differs
    assert abs(orc.log_Z_per_site(c) / orc.log_Z_per_site(b) - 1) > 1e-9


# ------------------------------------------------------------------ P8: invariances
def test_P8_field_sign_and_rescaling():
    # h -> -h is a sign gauge transformation on every leg: exact while nothing is truncated,
    # and only truncation-level once the seeded sketches see the flipped basis (reading G12).
    a2 = driver.run(BETA, 0.01, 16, 2, 2, 2, 3)
    b2 = driver.run(BETA, -0.01, 16, 2, 2, 2, 3)
    assert abs(orc.log_Z_per_site(a2) / orc.log_Z_per_site(b2) - 1) < 1e-13
    a = driver.run(BETA, 0.01, 6, 2, 2, 6, 3)
    b = driver.run(BETA, -0.01, 6, 2, 2, 6, 3)
    assert abs(orc.log_Z_per_site(a) / orc.log_Z_per_site(b) - 1) < 1e-4
    st = orc.init_ising_tensor(BETA, 0.01)
    st.phi *= 7.0
    st.psi *= 0.3
    st.log_acc -= np.log(7.0 * 0.3)
    for m in range(6):
        orc.coarse_grain(st, (m % 4) + 1, 6, 2, 2, driver.seeded_inputs_for(3, m))
    assert abs(orc.log_Z_per_site(st) / orc.log_Z_per_site(a) - 1) < 1e-12


def test_bad_arguments():
    with pytest.raises(ValueError):
        orc.init_ising_tensor(-1.0)
    st = orc.init_ising_tensor(BETA)
    with pytest.raises(ValueError):
        orc.coarse_grain(st, 5, 4, 2, 2, driver.seeded_inputs_for(1, 0))


# --------------------------------------------------------------------------- order parameter
def test_order_parameter_definition_on_the_dense_tensor():
    """X = (Tr A)^2 / Tr(A^2), A_kl = sum_{i1 i2 i3} T_{i1 i2 i3 k; i1 i2 i3 l} written out
    with explicit loops on the dense initial tensor T = Phi Psi^T (2^8 elements), for every open leg."""
    beta, h = 0.3, 0.07
    st = orc.init_ising_tensor(beta, h)
    T = np.tensordot(st.phi, st.psi, axes=([4], [4]))          # T[i1..i4, j1..j4]
    for leg in range(4):
        A = np.zeros((2, 2))
        for idx in np.ndindex(2, 2, 2, 2):
            for l in range(2):
                jdx = list(idx)
                jdx[leg] = l
                A[idx[leg], l] += T[idx + tuple(jdx)]
        X = np.trace(A) ** 2 / np.trace(A @ A)
        assert abs(orc.order_parameter_X(st, leg) - X) < 1e-13


def test_order_parameter_counts_degenerate_ground_states():
    """Deep in the ordered phase (T = 3 << T_c = 6.65, h = 0) two degenerate states dominate: X -> 2;
    deep in the disordered phase (T = 12) one: X -> 1."""
    def X_after(T, steps):
        st = orc.init_ising_tensor(1 / T, 0.0)
        for m in range(steps):
            orc.coarse_grain(st, m % 4 + 1, 4, 2, 2, driver.seeded_inputs_for(7, m))
        return orc.order_parameter_X(st, 3)
    assert abs(X_after(3.0, 8) - 2.0) < 1e-2
    assert abs(X_after(12.0, 16) - 1.0) < 2e-2
