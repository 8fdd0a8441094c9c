"""paper_2412_14104_b200 -- Triad-ATRG coarse-graining of the 4D Ising tensor network on one
NVIDIA B200 (sm_100a), FP64.

Thin ctypes binding of libtatrg.so (C-ABI: include/tatrg.h).  Argument marshalling only: every
step of the path runs in the library's CUDA kernels.  PyTorch is used for device memory and
streams.  There is no CPU fallback: importing works without a GPU (so that the symbols can be
checked), but every compute call needs the CUDA library and a device, and fails loudly otherwise.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtatrg.so")

EXPORTS = [
    "init_ising_tensor", "coarse_grain", "coarse_grain_atrg", "log_Z_per_site",
    "tatrg_set_stream", "tatrg_set_workspace", "tatrg_workspace_bytes", "tatrg_workspace_bytes_atrg",
    "tatrg_workspace_peak",
    "tatrg_set_sketch", "tatrg_sketch_shape", "tatrg_set_routes", "tatrg_set_side_split", "tatrg_keep_isometries", "tatrg_get_isometry", "tatrg_get_spectrum", "tatrg_get_gaps", "tatrg_get_dims",
    "tatrg_get_tensors", "tatrg_order_parameter", "tatrg_get_stage_ms", "tatrg_stage_name", "tatrg_get_h2d",
    "tatrg_set_profile", "tatrg_get_gemm_profile",
    "tatrg_launch_count", "tatrg_gemm_flops", "tatrg_probe_fp64_peak", "tatrg_tensor_gemm",
    "tatrg_fill_gauss", "tatrg_qr_pos", "tatrg_cholesky", "tatrg_cholqr", "tatrg_subspace_iteration", "tatrg_jacobi_svd", "tatrg_sumsq", "tatrg_sumsq_static", "tatrg_dot", "tatrg_scale_by_rsqrt",
    "tatrg_last_error", "tatrg_destroy",
]

SPECTRA = {"sigmaT": 0, "sigma_swap": 1, "SA": 2, "SX": 3, "SY": 4, "SD": 5, "s1": 6, "s2": 7, "s3": 8,
           "ln_c": 9}

_lib = None
_keep = {}     # keeps the workspace / sketch tensors alive while the library points into them


class TatrgError(RuntimeError):
    pass


def lib():
    """Loads libtatrg.so (built in-tree by build.py / __graft_entry__.build()); no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise TatrgError("libtatrg.so is missing: run `python paper_2412_14104_b200/build.py` "
                             "(there is no CPU fallback)")
        L = ctypes.CDLL(_SO)
        c_d, c_i, c_vp, c_sz = ctypes.c_double, ctypes.c_int, ctypes.c_void_p, ctypes.c_size_t
        c_i64, c_u64 = ctypes.c_int64, ctypes.c_uint64
        sig = {
            "init_ising_tensor": (c_i, [c_d, c_d]),
            "coarse_grain": (c_i, [c_i, c_i, c_i, c_i, c_u64]),
            "coarse_grain_atrg": (c_i, [c_i, c_i, c_i, c_i, c_u64]),
            "log_Z_per_site": (c_d, []),
            "tatrg_set_stream": (c_i, [c_vp]),
            "tatrg_set_workspace": (c_i, [c_vp, c_sz]),
            "tatrg_workspace_bytes": (c_sz, [c_i, c_i]),
            "tatrg_workspace_bytes_atrg": (c_sz, [c_i, c_i]),
            "tatrg_workspace_peak": (c_sz, []),
            "tatrg_set_sketch": (c_i, [c_i, c_vp, c_sz, c_i]),
            "tatrg_sketch_shape": (c_i, [c_i, c_i, c_i, c_i, ctypes.POINTER(c_i64), ctypes.POINTER(c_i64)]),
            "tatrg_get_spectrum": (c_i, [c_i, c_vp, c_i]),
            "tatrg_set_routes": (c_i, [c_i]),
            "tatrg_set_side_split": (c_i, [c_i, c_vp, c_vp]),
            "tatrg_keep_isometries": (c_i, [c_i]),
            "tatrg_get_isometry": (c_i, [c_i, c_vp, c_sz, ctypes.POINTER(c_i), ctypes.POINTER(c_i)]),
            "tatrg_get_gaps": (c_i, [c_vp]),
            "tatrg_get_dims": (c_i, [c_vp]),
            "tatrg_get_tensors": (c_i, [c_vp, c_vp, c_sz]),
            "tatrg_order_parameter": (c_d, [c_i]),
            "tatrg_get_stage_ms": (c_i, [c_vp, c_i]),
            "tatrg_stage_name": (ctypes.c_char_p, [c_i]),
            "tatrg_get_h2d": (c_i, [c_vp, c_vp]),
            "tatrg_set_profile": (c_i, [c_i]),
            "tatrg_get_gemm_profile": (c_i, [c_vp, c_i]),
            "tatrg_launch_count": (ctypes.c_longlong, [c_i]),
            "tatrg_gemm_flops": (c_d, [c_i]),
            "tatrg_probe_fp64_peak": (c_d, [c_i, c_i]),
            "tatrg_tensor_gemm": (c_i, [c_vp, c_vp, c_vp, c_i, c_i, c_i, c_i, c_vp, c_d, c_i]),
            "tatrg_fill_gauss": (c_i, [c_vp, c_u64, c_u64, c_u64, c_u64]),
            "tatrg_qr_pos": (c_i, [c_vp, c_i64, c_i, c_vp]),
            "tatrg_cholesky": (c_i, [c_vp, c_i, c_d, c_vp]),
            "tatrg_cholqr": (c_i, [c_vp, c_i64, c_i, c_i, c_d, c_vp]),
            "tatrg_subspace_iteration": (c_i, [c_vp, c_i, c_vp, c_vp, c_vp, c_i, c_i, c_vp, c_vp]),
            "tatrg_jacobi_svd": (c_i, [c_vp, c_i, c_i, c_vp, c_vp]),
            "tatrg_sumsq": (c_i, [c_vp, c_i64, c_vp]),
            "tatrg_sumsq_static": (c_i, [c_vp, c_i64, c_vp]),
            "tatrg_dot": (c_i, [c_vp, c_vp, c_i64, c_vp]),
            "tatrg_scale_by_rsqrt": (c_i, [c_vp, c_i64, c_vp]),
            "tatrg_last_error": (ctypes.c_char_p, []),
            "tatrg_destroy": (None, []),
        }
        for name, (res, args) in sig.items():
            f = getattr(L, name)
            f.restype = res
            f.argtypes = args
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        cause = _keep.pop("exchange_error", None)    # an exception of the caller's exchange (set_side_split)
        raise TatrgError("libtatrg error %d: %s" % (rc, lib().tatrg_last_error().decode())) from cause


def _require_cuda():
    import torch
    if not torch.cuda.is_available():
        raise TatrgError("no CUDA device: libtatrg has no CPU fallback")
    return torch


# ------------------------------------------------------------------ plumbing
def set_workspace(nbytes: int | None = None, chi: int | None = None, r: int = 2, device="cuda:0", atrg: bool = False):
    """Allocates the workspace as a torch tensor (PyTorch owns device memory) and hands it over.
    atrg: size it for coarse_grain_atrg (the chi^6 slices of the plain ATRG contraction)."""
    torch = _require_cuda()
    if nbytes is None:
        f = lib().tatrg_workspace_bytes_atrg if atrg else lib().tatrg_workspace_bytes
        nbytes = int(f(int(chi), int(r)))
    buf = torch.empty((nbytes + 255) // 256 * 32, dtype=torch.float64, device=device)
    _keep["ws"] = buf
    _check(lib().tatrg_set_workspace(buf.data_ptr(), buf.numel() * 8))
    return buf


def set_stream(stream=None):
    torch = _require_cuda()
    s = stream if stream is not None else torch.cuda.current_stream()
    _keep["stream"] = s
    _check(lib().tatrg_set_stream(ctypes.c_void_p(s.cuda_stream)))


def workspace_bytes(chi, r):
    return int(lib().tatrg_workspace_bytes(int(chi), int(r)))


def workspace_peak():
    return int(lib().tatrg_workspace_peak())


# ------------------------------------------------------------------ the three calls of the path
def init_ising_tensor(beta: float, h: float = 0.0):
    _require_cuda()
    _check(lib().init_ising_tensor(float(beta), float(h)))


def coarse_grain(direction: int, chi: int, r: int, q: int, seed: int):
    _require_cuda()
    _check(lib().coarse_grain(int(direction), int(chi), int(r), int(q), int(seed) & (2**64 - 1)))
    for k in [k for k in _keep if isinstance(k, tuple)]:
        del _keep[k]


def coarse_grain_atrg(direction: int, chi: int, r: int, q: int, seed: int):
    _require_cuda()
    _check(lib().coarse_grain_atrg(int(direction), int(chi), int(r), int(q), int(seed) & (2**64 - 1)))
    for k in [k for k in _keep if isinstance(k, tuple)]:
        del _keep[k]


def log_Z_per_site() -> float:
    _require_cuda()
    return float(lib().log_Z_per_site())


# ------------------------------------------------------------------ inputs / outputs
def set_sketch(which: int, data):
    """data: torch CUDA float64 tensor (device pointer) or C-contiguous numpy / pinned CPU torch
    tensor (host pointer, copied inside the next coarse_grain)."""
    if isinstance(data, np.ndarray):
        assert data.dtype == np.float64 and data.flags.c_contiguous
        ptr, n, dev = data.ctypes.data, data.size, 0
    else:
        import torch
        assert data.dtype == torch.float64 and data.is_contiguous()
        ptr, n, dev = data.data_ptr(), data.numel(), int(data.is_cuda)
    _keep[("sketch", which)] = data
    _check(lib().tatrg_set_sketch(int(which), ctypes.c_void_p(ptr), n, dev))


def sketch_shape(which, direction, chi, r):
    rows, cols = ctypes.c_int64(0), ctypes.c_int64(0)
    _check(lib().tatrg_sketch_shape(int(which), int(direction), int(chi), int(r),
                                    ctypes.byref(rows), ctypes.byref(cols)))
    return rows.value, cols.value


def get_spectrum(which) -> np.ndarray:
    w = SPECTRA[which] if isinstance(which, str) else int(which)
    out = np.empty(8192)
    n = lib().tatrg_get_spectrum(w, out.ctypes.data, out.size)
    if n < 0:
        _check(n)
    return out[:n].copy()


ROUTE_PLAIN_SWAP, ROUTE_HOUSEHOLDER_QR, ROUTE_DENSE_SQUEEZER, ROUTE_SEQUENTIAL_ISO, ROUTE_TMA_PRODUCER = 1, 2, 4, 8, 16
ROUTE_UNFUSED_SQUEEZER = 32


def set_routes(mask=0):
    """Forces the robust routes of coarse_grain (mask of ROUTE_*); 0 restores the defaults."""
    _check(lib().tatrg_set_routes(int(mask)))


_EXCHANGE_T = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64,
                               ctypes.c_void_p)


class _DeviceDoubles:
    """n doubles at a raw device address, for torch.as_tensor (no copy)."""

    def __init__(self, ptr, n):
        self.__cuda_array_interface__ = {"shape": (int(n),), "typestr": "<f8", "data": (int(ptr), False), "version": 2}


def set_side_split(sides=3, exchange=None):
    """tatrg_set_side_split: sides = 1 contracts Phi only, 2 Psi only, 3 both (default).  `exchange(phi, psi)` is a
    Python callable that gets the two new tensors as flat torch views of the library's buffers, with the library's
    stream current, and completes the half this process did not compute (two GPUs); with sides = 3
    it only observes the two finished, not yet normalised tensors."""
    import torch
    if int(sides) == 3 and exchange is None:
        _check(lib().tatrg_set_side_split(3, None, None))
        _keep.pop("exchange", None)
        return

    def trampoline(_user, phi_ptr, psi_ptr, n, stream_ptr):
        try:
            stream = torch.cuda.ExternalStream(stream_ptr) if stream_ptr else torch.cuda.default_stream()
            with torch.cuda.stream(stream):
                phi = torch.as_tensor(_DeviceDoubles(phi_ptr, n), device="cuda")
                psi = torch.as_tensor(_DeviceDoubles(psi_ptr, n), device="cuda")
                exchange(phi, psi)
            return 0
        except BaseException as e:      # an exception must not unwind through the C frames
            _keep["exchange_error"] = e
            return 1

    if exchange is None:
        raise TatrgError("set_side_split: computing one half needs an exchange callable")
    fn = _EXCHANGE_T(trampoline)
    _check(lib().tatrg_set_side_split(int(sides), ctypes.cast(fn, ctypes.c_void_p), None))
    _keep["exchange"] = fn


def exchange_halves(phi, psi, rank, group=None):
    """The one exchange of a split step: rank 0 of the two-process group owns Phi, rank 1 Psi; each sends its half
    to the other and receives the other's, as one batch of point-to-point operations (NCCL: both directions of
    the NVLink at once; ordered on the current stream).  Works on any pair of equally shaped tensors (gloo on CPU
    in the tests)."""
    import torch.distributed as dist
    if dist.get_world_size(group) != 2:
        raise TatrgError("the Phi / Psi split needs a group of exactly two processes")
    peer = dist.get_global_rank(group, 1 - rank) if group is not None else 1 - rank
    mine, other = (phi, psi) if rank == 0 else (psi, phi)
    ops = [dist.P2POp(dist.isend, mine, peer, group), dist.P2POp(dist.irecv, other, peer, group)]
    for w in dist.batch_isend_irecv(ops):
        w.wait()


def enable_phi_psi_split(group=None):
    """Splits every following coarse_grain / coarse_grain_atrg step over the two processes (one GPU each) of
    `group` (default: the world): this process contracts the half its group rank owns and exchange_halves
    completes the other over NCCL.  Both processes must run the same calls from the same state with the same seeds."""
    import torch.distributed as dist
    rank = dist.get_rank(group)
    if dist.get_world_size(group) != 2:
        raise TatrgError("the Phi / Psi split needs a group of exactly two processes")
    set_side_split(1 << rank, lambda phi, psi: exchange_halves(phi, psi, rank, group))


def disable_phi_psi_split():
    set_side_split(3)


def keep_isometries(on=True):
    _check(lib().tatrg_keep_isometries(int(bool(on))))


def get_isometry(which) -> np.ndarray:
    """U^which of the last step (which: 0..3 or 'A','X','Y','D'), shape [(p,q), k]; needs keep_isometries()."""
    w = "AXYD".index(which) if isinstance(which, str) else int(which)
    rows, cols = ctypes.c_int(0), ctypes.c_int(0)
    _check(lib().tatrg_get_isometry(w, None, 0, ctypes.byref(rows), ctypes.byref(cols)))
    out = np.empty((rows.value, cols.value))
    _check(lib().tatrg_get_isometry(w, out.ctypes.data, out.size, ctypes.byref(rows), ctypes.byref(cols)))
    return out


def get_gaps() -> np.ndarray:
    out = np.empty(4)
    _check(lib().tatrg_get_gaps(out.ctypes.data))
    return out


def get_dims():
    out = np.zeros(6, dtype=np.int32)
    _check(lib().tatrg_get_dims(out.ctypes.data))
    return tuple(int(v) for v in out)


def get_tensors():
    d = get_dims()
    shape = d[:5]
    n = int(np.prod(shape))
    phi, psi = np.empty(n), np.empty(n)
    _check(lib().tatrg_get_tensors(phi.ctypes.data, psi.ctypes.data, n))
    return phi.reshape(shape), psi.reshape(shape)


def order_parameter(leg: int = 4) -> float:
    return float(lib().tatrg_order_parameter(int(leg)))


def critical_temperature(chi: int, r: int, q: int, seed: int, T_lo: float, T_hi: float, n_steps: int = 12,
                         iters: int = 12, h: float = 0.0, leg: int = 4) -> float:
    """T_c by bisection on the order parameter X^(m) (Fig. 7): X -> 2 in the ordered
    phase (two degenerate ground states), X -> 1 in the disordered one; the bracket [T_lo, T_hi] is halved
    `iters` times on X(T) >< 1.5 after n_steps coarse-graining steps (directions cycling 1..4).  Host loop
    over the three calls of the path; every temperature is an independent run (replicas across GPUs).
    At h = 0 nothing protects the Z2 symmetry numerically: after ~16-20 steps rounding selects one of the two
    ordered states and X drops to 1 on the ordered side too, so X is read on its plateau (n_steps = 12-16)."""
    lo, hi = float(T_lo), float(T_hi)
    for _ in range(iters):
        T = 0.5 * (lo + hi)
        init_ising_tensor(1.0 / T, h)
        for m in range(n_steps):
            coarse_grain(m % 4 + 1, chi, r, q, seed)
        if order_parameter(leg) > 1.5:
            lo = T          # still ordered: T_c is above
        else:
            hi = T
    return 0.5 * (lo + hi)


def stage_ms() -> dict:
    out = np.zeros(16)
    n = lib().tatrg_get_stage_ms(out.ctypes.data, out.size)
    return {lib().tatrg_stage_name(i).decode(): float(out[i]) for i in range(n)}


def h2d():
    """(milliseconds on the copy stream, bytes) of the last step's host -> device input upload."""
    ms, nb = ctypes.c_double(0.0), ctypes.c_size_t(0)
    _check(lib().tatrg_get_h2d(ctypes.byref(ms), ctypes.byref(nb)))
    return ms.value, nb.value


def set_profile(on):
    """0 / False: off; 1 / True: time the 128x128-tile launches; 2: every tensor-GEMM launch."""
    _check(lib().tatrg_set_profile(int(on)))


def gemm_profile() -> dict:
    """{stage: {"ms": [small, big], "flops": [..], "launches": [..]}} of the last profiled step."""
    out = np.zeros(96)
    n = lib().tatrg_get_gemm_profile(out.ctypes.data, out.size)
    res = {}
    for i in range(n // 6):
        name = lib().tatrg_stage_name(i).decode()
        a = out[6 * i:6 * i + 6]
        res[name] = {"ms": [float(a[0]), float(a[3])], "flops": [float(a[1]), float(a[4])],
                     "launches": [int(a[2]), int(a[5])]}
    return res


def launch_count(reset=False) -> int:
    return int(lib().tatrg_launch_count(int(reset)))


def gemm_flops(reset=False) -> float:
    return float(lib().tatrg_gemm_flops(int(reset)))


def probe_fp64_peak(mode: int, iters: int = 4096) -> float:
    _require_cuda()
    v = float(lib().tatrg_probe_fp64_peak(int(mode), int(iters)))
    if v < 0:
        raise TatrgError(lib().tatrg_last_error().decode())
    return v


# ------------------------------------------------------------------ stand-alone kernels
def make_map(levels):
    """levels: list of (size, stride), fastest first, at most 4.  -> 7 int64."""
    assert 0 < len(levels) <= 4
    n = [0, 0, 0]
    s = [0, 0, 0, 0]
    for i, (size, stride) in enumerate(levels):
        s[i] = int(stride)
        if i < 3 and i + 1 < len(levels):
            n[i] = int(size)
    return n + s


def tensor_gemm(A, B, C, M, N, K, maps, batch=1, alpha=1.0, accumulate=False, tri_b=False):
    """maps: dict with keys am, ak, bk, bn, cm, cn (and optionally ab, bb, cb), each a list of
    (size, stride) levels.  A, B, C: torch CUDA float64 tensors.  tri_b: B[k][n] = 0 for k > n is promised
    (bit 1 of the C entry's `accumulate` argument)."""
    _require_cuda()
    flat = []
    for key in ("am", "ak", "bk", "bn", "cm", "cn", "ab", "bb", "cb"):
        flat += make_map(maps.get(key, [(1, 0)]))
    arr = np.asarray(flat, dtype=np.int64)
    _check(lib().tatrg_tensor_gemm(A.data_ptr(), B.data_ptr(), C.data_ptr(), int(M), int(N), int(K),
                                   int(batch), arr.ctypes.data, float(alpha), (1 if accumulate else 0) | (2 if tri_b else 0)))


def fill_gauss(out, seed: int, step: int, which: int):
    """out (CUDA float64 tensor) <- the seeded N(0,1) stream (seed, step, which), generated on the device."""
    _require_cuda()
    _check(lib().tatrg_fill_gauss(out.data_ptr(), out.numel(), int(seed), int(step), int(which)))


def qr_pos(Y, R):
    """In place: Y (m x n row-major CUDA tensor) <- Q; R (n x n) <- R with R_ii >= 0."""
    _require_cuda()
    m, n = Y.shape
    _check(lib().tatrg_qr_pos(Y.data_ptr(), int(m), int(n), R.data_ptr()))


def cholesky(A, Linv=None, shift_rel=0.0) -> bool:
    """In place: A (n x n row-major CUDA tensor, lower triangle read) <- lower Cholesky factor;
    Linv (optional, n x n) <- L^-1.  False if A was not numerically positive definite."""
    _require_cuda()
    n = A.shape[0]
    rc = lib().tatrg_cholesky(A.data_ptr(), int(n), float(shift_rel), Linv.data_ptr() if Linv is not None else None)
    if rc < 0:
        _check(rc)
    return rc == 0


def cholqr(Y, R=None, passes=2, shift_rel=0.0) -> bool:
    """In place Cholesky-QR of the tall m x n block Y (n <= 64): Y <- Q, R (optional) <- R."""
    _require_cuda()
    m, n = Y.shape
    rc = lib().tatrg_cholqr(Y.data_ptr(), int(m), int(n), int(passes), float(shift_rel),
                            R.data_ptr() if R is not None else None)
    if rc < 0:
        _check(rc)
    return rc == 0


def subspace_iteration(F, start, Q, Qt, iters, grid=16, R=None, minmax=None) -> bool:
    """Fused subspace iteration of a squeezer on the n x n matrix F with the n x 64 start block (sq_iter.cu)."""
    _require_cuda()
    n = F.shape[0]
    rc = lib().tatrg_subspace_iteration(F.data_ptr(), int(n), start.data_ptr(), Q.data_ptr(), Qt.data_ptr(), int(iters),
                                        int(grid), R.data_ptr() if R is not None else None,
                                        minmax.data_ptr() if minmax is not None else None)
    if rc < 0:
        _check(rc)
    return rc == 0


def jacobi_svd(G, V, s):
    """G: torch tensor holding a column-major m x n matrix as shape (n, m) row-major (row j = column j).
    In place G <- U diag(s); V shape (n, n), row k = k-th right singular vector."""
    _require_cuda()
    n, m = G.shape
    _check(lib().tatrg_jacobi_svd(G.data_ptr(), int(m), int(n), V.data_ptr(), s.data_ptr()))


def sumsq(x, out):
    _check(lib().tatrg_sumsq(x.data_ptr(), x.numel(), out.data_ptr()))


SUMSQ_STATIC_MAX_N = 1 << 32


def sumsq_static(x, out, n=None):
    """sumsq without workspace or allocation (static device scratch of the library); n defaults to x.numel()."""
    _check(lib().tatrg_sumsq_static(x.data_ptr(), x.numel() if n is None else int(n), out.data_ptr()))


def dot(x, y, out):
    _check(lib().tatrg_dot(x.data_ptr(), y.data_ptr(), x.numel(), out.data_ptr()))


def scale_by_rsqrt(x, ss):
    _check(lib().tatrg_scale_by_rsqrt(x.data_ptr(), x.numel(), ss.data_ptr()))


def destroy():
    lib().tatrg_destroy()
    _keep.clear()
