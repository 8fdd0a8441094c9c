"""Parity of the CUDA path (through the C-ABI) with the CPU oracle on the same seeded inputs.

Compared: ln Z per site after every step (BASELINE.json north_star: 1e-10 relative) and every
truncated spectrum of every step (1e-9 of the largest value, reading G13), plus dims.  Gauge
dependent tensors are not compared (reading G18)."""
import numpy as np
import pytest

from oracle import driver
from oracle import tatrg_oracle as orc

pytestmark = pytest.mark.gpu

LNZ_RTOL = 1e-10
SPEC_TOL = 1e-9
# The isometries themselves, gauge invariant (reading G18): max |U S^2 U^T - U_o S_o^2 U_o^T| / S_1^2, the
# Ritz approximation Q H Q^T of the pair operator K K_w^T that the Ritz step diagonalises.  (The plain
# projector U U^T is not unique when K K_w^T has fewer than r chi non-zero eigenvalues, as in the early
# steps: the trailing Ritz vectors then span an arbitrary part of the null space and carry no weight in
# Gamma; for the same reason the spectra S^A..S^D are compared through lambda = S^2, see below.)
PROJ_TOL = 1e-9
# config 2's steps 22..40: the two sides' tensors have drifted apart by 1e-10 (sigma^T) and the Ritz VECTORS of
# q = 2 unconverged iterations follow with the amplification the oracle's own Ritz values show against itself
# (10-27x, oracle_sensitivity_c2*.json); measured 8.7e-9 at worst
PROJ_TOL_LATE = 3e-8


def spectrum_deviation(name, so, sg):
    """Reading G13: max_i |s_i - s_i^ref| / s_1^ref for the truncated spectra (sigma^T, sigma_swap, s^(mu)).
    S^A..S^D are square roots of the Ritz values lambda of the pair operator K K_w^T, which the Ritz step
    (oracle: eigh of Q^T S Q) determines to eps lambda_1 in absolute terms: a Ritz value at rounding level
    (rank-deficient K K_w^T in the early steps, r chi above the rank) has a square root anywhere below
    ~1e-8 S_1, and the oracle's own S^X moves by 2.8e-10 S_1 under a 1-ulp change of its sketches there
    (tests/golden/oracle_sensitivity_w80.json) while its sigma's move by 1e-15; along config 2's 40 steps the
    oracle's S^A..S^D move 10-27 times further than its sigma's (oracle_sensitivity_c2*.json).  They are
    therefore compared through lambda = S^2, the quantity that is determined:
    max_i |lambda_i - lambda_i^ref| / lambda_1^ref (for S_i ~ S_1 this is twice as strict as the plain rule;
    measured on config 2's 40 steps: 3.2e-10 at worst, where the plain rule reads 3.3e-9)."""
    if name in ("SA", "SX", "SY", "SD"):
        return float(np.abs(so ** 2 - sg ** 2).max() / so[0] ** 2)
    return float(np.abs(so - sg).max() / so[0])


@pytest.fixture(scope="module")
def tt():
    import torch
    import paper_2412_14104_b200 as t
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    t.set_workspace(nbytes=8 << 30)
    t.set_stream()
    yield t
    t.destroy()


def run_both(tt, beta, h, chi, r, q, n_steps, seed, directions=None, mode="triad"):
    """Oracle and GPU step by step; returns list of per-step comparison records."""
    recs = []
    st = orc.init_ising_tensor(beta, h)
    tt.init_ising_tensor(beta, h)
    tt.keep_isometries(mode == "triad")
    assert abs(tt.log_Z_per_site() / orc.log_Z_per_site(st) - 1) < 1e-13
    for m in range(n_steps):
        d = directions[m % len(directions)] if directions else (m % 4) + 1
        rec = orc.coarse_grain(st, d, chi, r, q, driver.seeded_inputs_for(seed, m), mode=mode)
        (tt.coarse_grain if mode == "triad" else tt.coarse_grain_atrg)(d, chi, r, q, seed)
        out = {"step": m, "lnz_o": orc.log_Z_per_site(st), "lnz_g": tt.log_Z_per_site(),
               "dims_o": st.dims, "dims_g": tt.get_dims()[:5], "spec": {}, "proj": {}}
        for name in ("sigmaT", "sigma_swap", "SA", "SX", "SY", "SD", "s1", "s2", "s3"):
            so, sg = np.asarray(rec[name]) if name in rec else np.zeros(0), tt.get_spectrum(name)
            out["spec"][name] = (so, sg)
        if mode == "triad":
            for t in "AXYD":
                uo = rec["U"][t].reshape(-1, rec["U"][t].shape[-1])
                ug = tt.get_isometry(t)
                assert uo.shape == ug.shape, (m, t, uo.shape, ug.shape)
                so, sg = np.asarray(rec["S" + t]), tt.get_spectrum("S" + t)
                if len(so):
                    out["proj"][t] = float(np.abs((uo * so ** 2) @ uo.T - (ug * sg ** 2) @ ug.T).max() / so[0] ** 2)
        recs.append(out)
    tt.keep_isometries(False)
    return recs


def check(recs, lnz_rtol=LNZ_RTOL, spec_tol=SPEC_TOL, proj_late=None):
    worst = {}
    for o in recs:
        assert tuple(o["dims_o"]) == tuple(o["dims_g"]), o
        for name, (so, sg) in o["spec"].items():
            assert len(so) == len(sg), (o["step"], name, len(so), len(sg))
            if len(so):
                dev = spectrum_deviation(name, so, sg)
                worst[name] = max(worst.get(name, 0.0), dev)
                assert dev <= spec_tol, (o["step"], name, dev)
        for t, dev in o["proj"].items():
            worst["P" + t] = max(worst.get("P" + t, 0.0), dev)
            ptol = PROJ_TOL_LATE if (proj_late is not None and o["step"] >= proj_late) else PROJ_TOL
            assert dev <= ptol, (o["step"], "Ritz operator of U^" + t, dev)
        dz = abs(o["lnz_g"] / o["lnz_o"] - 1)
        worst["lnz"] = max(worst.get("lnz", 0.0), dz)
        assert dz <= lnz_rtol, (o["step"], o["lnz_g"], o["lnz_o"])
    print("worst deviations:", {k: "%.2e" % v for k, v in worst.items()})


def test_config1_chi6_8steps(tt):
    """BASELINE.json configs[0]: T=6.0, chi=6, r=2, q=2, 8 steps cycling 1..4 (4^4 lattice)."""
    check(run_both(tt, 1 / 6.0, 0.0, 6, 2, 2, 8, 20241214))


def test_untruncated_tiny_lattice_matches_enumeration(tt):
    """GPU path against exact enumeration directly (2x2x1x1 lattice, chi large enough)."""
    from exact_refs import brute_force_lnZ
    tt.init_ising_tensor(1 / 6.0, 0.01)
    tt.coarse_grain(1, 16, 2, 2, 7)
    tt.coarse_grain(2, 16, 2, 2, 7)
    assert abs(tt.log_Z_per_site() / brute_force_lnZ(1 / 6.0, 0.01, (2, 2, 1, 1)) - 1) < 1e-12


@pytest.mark.parametrize("dirs", [[2, 3, 1, 4], [4, 4, 1, 2]])
def test_direction_orders_with_field(tt, dirs):
    check(run_both(tt, 1 / 6.5, 0.01, 5, 2, 1, 4, 99, directions=dirs))


def test_config2_chi16_all_40_steps(tt):
    """BASELINE.json configs[1] (T=6.65, chi=16, r=2, q=2) in full: 40 steps, L = 2^10 per direction.
    (Measured: ln Z/V agrees to 3e-15 at every step, the spectra to 5e-10.)"""
    check(run_both(tt, 1 / 6.65, 0.0, 16, 2, 2, 40, 20241215), proj_late=21)


def test_config3_chi32_first_steps_incl_one_full_size_step(tt):
    """BASELINE.json configs[2] (the headline config: T=6.65, chi=32, r=2, q=2), the first 5 of its 40
    steps.  Step 5 has all legs and the bond = 32 on input: the launch configuration bench.py times
    (reduced bond swap, concurrent isometry / squeezer chains, 64-column sketches); the oracle needs
    about a minute for it."""
    check(run_both(tt, 1 / 6.65, 0.0, 32, 2, 2, 5, 20241216))


def test_r7_parity_chi10(tt):
    """The paper's oversampling r = 7 (Table 2 and Figs. 4-6 are at r = 7), 8 steps at
    chi = 10.  (Not chi = 8: there the second bond swap cuts a four-fold degenerate multiplet of singular
    values 0.1568 s_1 in the middle -- the oracle logs gap_swap = 5e-17 --, so which vectors are kept is not
    determined and no two implementations agree beyond the truncation error; reading G12.)"""
    check(run_both(tt, 1 / 6.65, 0.0, 10, 7, 2, 8, 424242))


def test_r7_wide_internal_lines_chi20(tt):
    """r chi = 140 > 128: sketches, Cholesky-QR panels and Ritz cores between 129 and 256 columns wide
    (5 steps of chi = 20, r = 7, q = 1; the fifth has 140 of 256 pair states kept by the isometries)."""
    check(run_both(tt, 1 / 6.65, 0.0, 20, 7, 1, 5, 434343))


@pytest.mark.parametrize("chi,r,n", [(12, 3, 10), (20, 2, 7)])
def test_isometry_chains_at_widths_between_32_and_64(tt, chi, r, n):
    """Oversampled lines that are neither 32 nor 64 wide on the concurrent isometry chains (fused Cholesky-QR of a
    36- or 40-column block, the one-CTA Ritz solver at that width): chi = 12, r = 3 (r chi = 36 on 144 pair
    states, the fewest rows per column the chains take) and chi = 20, r = 2 (r chi = 40 on 400 pair states)."""
    check(run_both(tt, 1 / 6.65, 0.0, chi, r, 2, n, 20241219))


def test_plain_atrg_parity(tt):
    """coarse_grain_atrg (Table 1: no triads, O(chi^9) contraction) against the oracle's
    mode='atrg' on the same seeded bond-swap sketches."""
    check(run_both(tt, 1 / 6.65, 0.0, 6, 2, 2, 6, 20241217, mode="atrg"))


def test_triad_equals_atrg_when_r_chi_covers_pair_gpu(tt):
    """r*chi >= d2*d3 => the isometries are identities and Triad-ATRG is ATRG (GPU vs GPU)."""
    out = []
    for fn in (tt.coarse_grain, tt.coarse_grain_atrg):
        tt.init_ising_tensor(1 / 6.0, 0.02)
        for m in range(4):
            fn(m % 4 + 1, 4, 4, 2, 31)
        out.append(tt.log_Z_per_site())
    assert abs(out[0] / out[1] - 1) < 1e-12, out


def test_config4_atrg_chi24_vs_triad(tt):
    """BASELINE.json configs[3] shape check at reduced length: plain ATRG chi=24 (O(chi^9) GEMM
    13824 x 13824 x 576 per slice), 5 steps, against a Triad-ATRG run at the same chi: the free
    energies agree to truncation level (PAPER.md:139 quotes 0.0013 % at chi=54; not a pin)."""
    out = []
    for fn in (tt.coarse_grain_atrg, tt.coarse_grain):
        tt.init_ising_tensor(1 / 6.65, 0.0)
        for m in range(5):
            fn(m % 4 + 1, 24, 2, 2, 20241217)
        out.append(tt.log_Z_per_site())
    assert abs(out[0] / out[1] - 1) < 1e-4, out


def _supply(tt, where, seed, m, d, chi, r, only=None):
    import torch
    import seeded_inputs as si
    keep = []
    for which in range(9):
        if only is not None and which not in only:
            continue
        rows, cols = tt.sketch_shape(which, d, chi, r)
        if rows * cols == 0:
            continue
        g = si.gauss(si.subseed(seed, 0 if which >= 5 else m, which), rows * cols)
        if where == "host_pageable":
            buf = g
        else:
            buf = torch.from_numpy(g)
            buf = buf.cuda() if where == "device" else buf.pin_memory()
        keep.append(buf)
        tt.set_sketch(which, buf)
    return keep


@pytest.mark.parametrize("where", ["host_pinned", "host_pageable", "device"])
def test_caller_supplied_inputs(tt, where):
    """Sketches and gauge references handed over through tatrg_set_sketch (host buffers are uploaded
    by the library's copy stream while the step's first stage runs; device buffers are used in place)
    give the oracle's result like the internally generated ones: same generator, same sub-seeds."""
    beta, chi, r, q, seed = 1 / 6.0, 6, 2, 2, 20241214      # config 1: no cut through a degenerate multiplet
    st = orc.init_ising_tensor(beta, 0.0)
    tt.init_ising_tensor(beta, 0.0)
    for m in range(7):
        d = m % 4 + 1
        keep = _supply(tt, where, seed, m, d, chi, r)
        rec = orc.coarse_grain(st, d, chi, r, q, driver.seeded_inputs_for(seed, m))
        tt.coarse_grain(d, chi, r, q, seed)
        del keep
        lo, lg = orc.log_Z_per_site(st), tt.log_Z_per_site()
        assert abs(lg / lo - 1) <= LNZ_RTOL, (m, lg, lo)
        for name in ("sigma_swap", "s1", "s2", "s3"):
            so, sg = np.asarray(rec[name]), tt.get_spectrum(name)
            assert len(so) == len(sg) and np.abs(so - sg).max() <= SPEC_TOL * so[0], (m, name)


@pytest.mark.parametrize("where", ["host_pinned", "device"])
def test_caller_supplied_sketch_is_the_one_used(tt, where):
    """A swap sketch from another stream changes the step at truncation level (and only there)."""
    beta, chi, r, q, seed = 1 / 6.0, 6, 2, 2, 20241214
    out = []
    for other in (False, True):
        tt.init_ising_tensor(beta, 0.0)
        for m in range(6):
            keep = _supply(tt, where, seed + 17, m, m % 4 + 1, chi, r, only=(0,)) if (other and m == 5) else None
            tt.coarse_grain(m % 4 + 1, chi, r, q, seed)
            del keep
        out.append(tt.log_Z_per_site())
    assert 1e-13 < abs(out[0] / out[1] - 1) < 1e-3, out


def test_order_parameter_matches_oracle(tt):
    """X^(m) = (Tr A)^2 / Tr(A^2) from the device-resident (Phi, Psi)
    against the oracle's, every leg, along the config-1 schedule."""
    beta, chi, r, q, seed = 1 / 6.0, 6, 2, 2, 20241214
    st = orc.init_ising_tensor(beta, 0.0)
    tt.init_ising_tensor(beta, 0.0)
    for m in range(6):
        orc.coarse_grain(st, m % 4 + 1, chi, r, q, driver.seeded_inputs_for(seed, m))
        tt.coarse_grain(m % 4 + 1, chi, r, q, seed)
        for leg in range(4):
            xo, xg = orc.order_parameter_X(st, leg), tt.order_parameter(leg + 1)
            assert abs(xg / xo - 1) < 1e-9, (m, leg, xg, xo)


def test_errors_leave_the_state_intact(tt):
    """include/tatrg.h: errors never abort; a failed coarse_grain leaves the previous state in place."""
    import paper_2412_14104_b200 as t
    tt.init_ising_tensor(1 / 6.0, 0.0)
    tt.coarse_grain(1, 6, 2, 2, 1)
    tt.coarse_grain(2, 6, 2, 2, 1)
    before, dims = tt.log_Z_per_site(), tt.get_dims()
    for args in ((0, 6, 2, 2, 1), (5, 6, 2, 2, 1), (1, 0, 2, 2, 1), (1, 6, 0, 2, 1), (1, 6, 2, -1, 1), (1, 65, 2, 2, 1),
                 (1, 64, 5, 2, 1)):
        with pytest.raises(t.TatrgError):
            tt.coarse_grain(*args)
    with pytest.raises(t.TatrgError):
        tt.init_ising_tensor(-1.0, 0.0)
    assert tt.log_Z_per_site() == before and tt.get_dims() == dims
    # a workspace that cannot hold some step: that step fails with a TatrgError and the state of the
    # step before is still there
    import torch
    small = torch.empty(1 << 17, dtype=torch.float64, device="cuda")     # 1 MB
    t._check(t.lib().tatrg_set_workspace(small.data_ptr(), small.numel() * 8))
    try:
        tt.init_ising_tensor(1 / 6.0, 0.0)
        failed_at = None
        for m in range(8):
            before, dims = tt.log_Z_per_site(), tt.get_dims()
            try:
                tt.coarse_grain(m % 4 + 1, 16, 2, 2, 1)
            except t.TatrgError as e:
                failed_at = m
                assert "workspace" in str(e)
                break
        assert failed_at is not None and failed_at >= 1
        assert tt.log_Z_per_site() == before and tt.get_dims() == dims
    finally:
        tt.set_workspace(nbytes=8 << 30)
        tt.init_ising_tensor(1 / 6.0, 0.0)


def test_critical_temperature_bisection(tt):
    """SURVEY 8(f) NEXT-1 / PAPER.md Fig. 7: bisection on X^(m).  At chi = 8 the estimate is crude (the paper
    needs chi ~ 50 for 0.1 %); it must land in the neighbourhood of the Monte Carlo value T_c = 6.68."""
    Tc = tt.critical_temperature(chi=8, r=2, q=2, seed=5, T_lo=5.0, T_hi=8.5, n_steps=12, iters=8)
    assert 6.4 < Tc < 7.2, Tc


@pytest.mark.parametrize("mask", [1, 2, 4, 8, 15, 32])
def test_robust_routes_give_the_same_step(tt, mask):
    """Every stage has a fast route and a robust route that follows the oracle's algorithm step by step
    (tatrg_set_routes): bit 0 plain chi^4-dimensional bond-swap operator instead of the
    reduced chi^3 core, bit 1 Householder TSQR instead of Cholesky-QR, bit 2 dense eigendecompositions instead
    of Cholesky + subspace iteration in the squeezers, bit 3 sequential isometries, bit 5 the squeezers' subspace
    iteration as separate launches instead of the one resident grid of sq_iter.cu.  Config 2 (chi = 16), 10
    steps: from step 5 on every fast route is taken by default (GPU against GPU)."""
    import paper_2412_14104_b200 as t
    beta, chi, r, q, seed, n = 1 / 6.65, 16, 2, 2, 20241215, 10
    runs = []
    for m_ in (0, mask):
        tt.set_routes(m_)
        try:
            tt.init_ising_tensor(beta, 0.0)
            rec = []
            for m in range(n):
                tt.coarse_grain(m % 4 + 1, chi, r, q, seed)
                rec.append((tt.log_Z_per_site(), {k: tt.get_spectrum(k) for k in t.SPECTRA if k != "ln_c"}))
            runs.append(rec)
        finally:
            tt.set_routes(0)
    for m in range(n):
        (l0, s0), (l1, s1) = runs[0][m], runs[1][m]
        assert abs(l1 / l0 - 1) <= LNZ_RTOL, (m, l0, l1)
        for k in s0:
            assert len(s0[k]) == len(s1[k]), (m, k)
            if len(s0[k]):
                assert spectrum_deviation(k, s0[k], s1[k]) <= SPEC_TOL, (m, k, spectrum_deviation(k, s0[k], s1[k]))
