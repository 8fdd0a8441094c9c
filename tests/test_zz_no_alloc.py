"""tatrg_sumsq_static: the one entry point of libtatrg that allocates nothing (include/tatrg.h) -- the squared
Frobenius norm of the step's normalisation (Eq. 15) with the per-CTA partial sums in a static device
array of the library instead of the caller's workspace.  Checked against the existing path (tatrg_sumsq, partial
sums in the workspace) and against numpy, on two calls in a row that share the static array: a large input that
fills every slot, then a smaller one that uses a few slots only (stale partial sums of the first call must not
leak into the second).  The file sorts last on purpose (the suite runs with -x); it passes alone in a fresh process
and after the other tests (every fixture there ends with tatrg_destroy, so the library is without a workspace
when this starts)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

RTOL = 1e-14   # the tolerance of the norm checks in tests/test_gpu_kernels.py


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def test_sumsq_static_matches_the_workspace_path_on_two_calls_in_a_row():
    torch = _torch()
    import paper_2412_14104_b200 as tt
    tt.destroy()                      # no workspace, default stream: the state of a caller that never set one
    rng = np.random.default_rng(20241214)
    sizes = [(1 << 22) + 3, 4097]     # 1184 CTAs (every slot of the static array), then 3 CTAs
    xs = [rng.standard_normal(n) for n in sizes]
    dxs = [torch.from_numpy(x).cuda() for x in xs]
    out_static = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    # two calls in a row, no workspace set
    tt.sumsq_static(dxs[0], out_static[0:1])
    tt.sumsq_static(dxs[1], out_static[1:2])
    torch.cuda.synchronize()
    got = out_static.cpu().numpy()
    # the existing path needs a workspace
    out_ws = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    tt.set_workspace(nbytes=1 << 20)
    tt.set_stream()
    try:
        tt.sumsq(dxs[0], out_ws[0:1])
        tt.sumsq(dxs[1], out_ws[1:2])
        torch.cuda.synchronize()
        ref = out_ws.cpu().numpy()
        for i, x in enumerate(xs):
            assert abs(got[i] / ref[i] - 1) <= RTOL, (i, got[i], ref[i])
            assert got[i] == ref[i], "same kernels on the same grid: expected the same bits"
            assert abs(got[i] / float(np.dot(x, x)) - 1) <= 1e-13, (i, got[i], float(np.dot(x, x)))
        # and again in the other order, with the workspace set (the static path must not depend on it either way)
        tt.sumsq_static(dxs[1], out_static[1:2])
        tt.sumsq_static(dxs[0], out_static[0:1])
        torch.cuda.synchronize()
        np.testing.assert_array_equal(out_static.cpu().numpy(), ref)
    finally:
        tt.destroy()


def test_sumsq_static_edge_cases_and_size_limit():
    torch = _torch()
    import paper_2412_14104_b200 as tt
    tt.destroy()
    x = torch.arange(1, 8, dtype=torch.float64, device="cuda")
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    tt.sumsq_static(x, out)
    torch.cuda.synchronize()
    assert out.item() == 140.0
    tt.sumsq_static(x[1:], out)           # a pointer that is not 16-byte aligned: the scalar loads
    torch.cuda.synchronize()
    assert out.item() == 139.0
    tt.sumsq_static(x, out, n=0)          # empty input
    torch.cuda.synchronize()
    assert out.item() == 0.0
    # beyond the stated maximum: rejected before anything is launched, with a message that names the limit
    out.fill_(-1.0)
    with pytest.raises(tt.TatrgError) as e:
        tt.sumsq_static(x, out, n=tt.SUMSQ_STATIC_MAX_N + 1)
    assert "maximum" in str(e.value) and str(tt.SUMSQ_STATIC_MAX_N) in str(e.value)
    with pytest.raises(tt.TatrgError):
        tt.sumsq_static(x, out, n=-1)
    torch.cuda.synchronize()
    assert out.item() == -1.0
