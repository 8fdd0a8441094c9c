"""Two-GPU Phi / Psi split of the step (tatrg_set_side_split; "two GPUs are used", SURVEY.md 8(f)
NEXT-4) on ONE GPU: the two processes of the split are played one after the other, never side by side.

  whole : the step as it is (both halves), recording ln Z/V, every spectrum and the tensors after each step, and,
          through the exchange callback as an observer, the two tensors before the normalisation;
  rank 1: contracts Psi only (sides = 2); its exchange keeps a copy of its Psi ("sent") and receives the Phi the
          whole run produced;
  rank 0: contracts Phi only (sides = 1); its exchange receives exactly what rank 1 sent.

The split rests on one assumption: two processes that run the same kernels on the same bits get the same bits
(the squeezers and the swap bond are shared by the two halves, and a rounding-level difference would turn a
degenerate pair of their spectra -- the Z2 symmetry at h = 0 makes pairs -- into two different gauges).  So the
halves are compared BIT FOR BIT with the whole run's, step by step; rank 0's run must then reproduce the whole run:
ln Z/V to 1e-10, every spectrum to 1e-9, the tensors element by element.  GPU against GPU; the whole run itself is compared
with the oracle in tests/test_gpu_parity.py.  The exchange over two processes (exchange_halves) is covered on CPU
with gloo in tests/test_multi_rank_host_logic.py."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

LNZ_RTOL = 1e-10     # as tests/test_gpu_parity.py
SPEC_TOL = 1e-9
ELEM_TOL = 1e-9      # tensors have unit Frobenius norm; measured ~1e-15


@pytest.fixture(scope="module")
def tt():
    import torch
    import paper_2412_14104_b200 as t
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    t.set_workspace(nbytes=8 << 30)
    t.set_stream()
    yield t
    t.set_side_split(3)
    t.destroy()


def _run(tt, step, beta, chi, r, q, seed, n, sides, exchange):
    import paper_2412_14104_b200 as t
    tt.set_side_split(sides, exchange)
    try:
        tt.init_ising_tensor(beta, 0.0)
        rec = []
        for m in range(n):
            exchange_state["m"] = m
            step(m % 4 + 1, chi, r, q, seed)
            phi, psi = tt.get_tensors()
            rec.append({"lnz": tt.log_Z_per_site(), "phi": phi, "psi": psi,
                        "spec": {k: tt.get_spectrum(k) for k in t.SPECTRA}})
        return rec
    finally:
        tt.set_side_split(3)


exchange_state = {"m": 0}


@pytest.mark.parametrize("mode,chi,r,q,n", [("triad", 16, 2, 2, 10), ("triad", 6, 2, 1, 6), ("atrg", 6, 2, 2, 6)])
def test_split_halves_reproduce_the_whole_step(tt, mode, chi, r, q, n):
    """chi = 16, 10 steps of config 2: from step 5 on the halves' products (i), (ii) run beside the squeezer chains
    (the default route of config 3 too); chi = 6: the slab route; plain ATRG: the two O(chi^9) products."""
    beta, seed = 1 / 6.65, 20241215
    step = tt.coarse_grain if mode == "triad" else tt.coarse_grain_atrg
    un = {"phi": [], "psi": []}

    def observe(phi, psi):
        un["phi"].append(phi.clone())
        un["psi"].append(psi.clone())

    whole = _run(tt, step, beta, chi, r, q, seed, n, 3, observe)
    assert len(un["phi"]) == n

    sent_by_rank1, diff = [], {"r0": [], "r1": []}

    def exchange_rank1(phi, psi):
        m = exchange_state["m"]
        assert phi.numel() == psi.numel() == whole[m]["phi"].size
        sent_by_rank1.append(psi.clone())
        diff["r1"].append(float((psi - un["psi"][m]).abs().max()))
        phi.copy_(un["phi"][m])

    rank1 = _run(tt, step, beta, chi, r, q, seed, n, 2, exchange_rank1)

    def exchange_rank0(phi, psi):
        m = exchange_state["m"]
        diff["r0"].append(float((phi - un["phi"][m]).abs().max()))
        psi.copy_(sent_by_rank1[m])

    rank0 = _run(tt, step, beta, chi, r, q, seed, n, 1, exchange_rank0)
    assert len(diff["r0"]) == len(diff["r1"]) == n        # once per step
    assert diff["r1"] == [0.0] * n, diff["r1"]            # each half: the same bits as in the whole step
    assert diff["r0"] == [0.0] * n, diff["r0"]
    for m in range(n):
        w, g = whole[m], rank0[m]
        assert abs(g["lnz"] / w["lnz"] - 1) <= LNZ_RTOL, (m, w["lnz"], g["lnz"])
        for k in w["spec"]:
            assert len(w["spec"][k]) == len(g["spec"][k]), (m, k)
            if len(w["spec"][k]):
                dev = np.abs(w["spec"][k] - g["spec"][k]).max() / max(abs(w["spec"][k][0]), 1e-300)
                assert dev <= SPEC_TOL, (m, k, dev)
        for name in ("phi", "psi"):
            assert w[name].shape == g[name].shape
            assert np.abs(w[name] - g[name]).max() <= ELEM_TOL, (m, name, np.abs(w[name] - g[name]).max())
        assert rank1[m]["lnz"] == w["lnz"] and g["lnz"] == w["lnz"]          # the same bits in, the same bits out
        for name in ("phi", "psi"):
            assert np.array_equal(w[name], rank1[m][name]) and np.array_equal(w[name], g[name]), (m, name)


def test_split_errors(tt):
    import paper_2412_14104_b200 as t
    with pytest.raises(t.TatrgError):
        tt.set_side_split(1, None)
    assert tt.lib().tatrg_set_side_split(0, None, None) == -22
    assert tt.lib().tatrg_set_side_split(2, None, None) == -22      # one half without an exchange
    # an exchange that fails: the step fails, the previous state stays
    beta, chi, r, q, seed = 1 / 6.65, 6, 2, 1, 7
    tt.init_ising_tensor(beta, 0.0)
    tt.coarse_grain(1, chi, r, q, seed)
    before = (tt.get_dims(), tt.log_Z_per_site())

    def broken(phi, psi):
        raise ValueError("no peer")

    tt.set_side_split(1, broken)
    try:
        with pytest.raises(t.TatrgError) as e:
            tt.coarse_grain(2, chi, r, q, seed)
        assert isinstance(e.value.__cause__, ValueError)
    finally:
        tt.set_side_split(3)
    assert (tt.get_dims(), tt.log_Z_per_site()) == before
    tt.coarse_grain(2, chi, r, q, seed)                              # and the whole step still runs
    assert tt.get_dims()[5] == 2
