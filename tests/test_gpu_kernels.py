"""GPU kernel checks through the C-ABI: every stand-alone kernel of libtatrg against the plain
definition of what it computes (numpy FP64 on the host), on sizes that span several tiles and a
ragged tail, plus the degenerate cases (rank-deficient QR, zero columns, odd sizes)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def tt():
    import torch
    import paper_2412_14104_b200 as t
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    t.set_workspace(nbytes=1 << 30)
    t.set_stream()
    yield t
    t.destroy()


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("M,N,K", [(128, 128, 64), (200, 136, 77), (1, 1, 1), (7, 300, 5), (513, 65, 1030),
                                   (64, 64, 20000)])
def test_tensor_gemm_plain(tt, M, N, K):
    rng = np.random.default_rng(M * 7 + N * 3 + K)
    A, B = rng.standard_normal((M, K)), rng.standard_normal((K, N))
    import torch
    dA, dB = _dev(A), _dev(B)
    dC = torch.zeros(M, N, dtype=torch.float64, device="cuda")
    maps = dict(am=[(M, K)], ak=[(K, 1)], bk=[(K, N)], bn=[(N, 1)], cm=[(M, N)], cn=[(N, 1)])
    tt.tensor_gemm(dA, dB, dC, M, N, K, maps, alpha=0.5)
    torch.cuda.synchronize()
    ref = 0.5 * (A @ B)
    np.testing.assert_allclose(dC.cpu().numpy(), ref, rtol=0, atol=1e-12 * np.sqrt(K) * 4)
    # transposed operands (m-contiguous A, k-contiguous B) and accumulate
    dAt, dBt = _dev(A.T), _dev(B.T)
    maps = dict(am=[(M, 1)], ak=[(K, M)], bk=[(K, 1)], bn=[(N, K)], cm=[(M, N)], cn=[(N, 1)])
    tt.tensor_gemm(dAt, dBt, dC, M, N, K, maps, alpha=1.0, accumulate=True)
    torch.cuda.synchronize()
    np.testing.assert_allclose(dC.cpu().numpy(), 1.5 * (A @ B), rtol=0, atol=1e-12 * np.sqrt(K) * 8)


def test_tensor_gemm_permuted_legs_batched(tt):
    """C[b,x,w,l,g] = sum_{a,u} EM[b,x,a,u,w] F[a,l,u,g] * s : the shape of Eq. 13's inner product
     with composite row / column / summed indices and a batch leg."""
    import torch
    rng = np.random.default_rng(5)
    nb, nx, na, nu, nw, nl, ng = 3, 5, 6, 4, 7, 9, 6
    EM = rng.standard_normal((nb, nx, na, nu, nw))
    F = rng.standard_normal((na, nl, nu, ng))
    ref = np.ascontiguousarray(np.einsum("bxauw,alug->bxwlg", EM, F))
    dEM, dF = _dev(EM), _dev(F)
    dC = torch.empty(ref.shape, dtype=torch.float64, device="cuda")
    se, sf, sc = [s // 8 for s in EM.strides], [s // 8 for s in F.strides], [s // 8 for s in ref.strides]
    maps = dict(am=[(nw, se[4]), (nx, se[1])], ak=[(nu, se[3]), (na, se[2])],
                bk=[(nu, sf[2]), (na, sf[0])], bn=[(ng, sf[3]), (nl, sf[1])],
                cm=[(nw, sc[2]), (nx, sc[1])], cn=[(ng, sc[4]), (nl, sc[3])],
                ab=[(nb, se[0])], bb=[(nb, 0)], cb=[(nb, sc[0])])
    tt.tensor_gemm(dEM, dF, dC, nx * nw, nl * ng, na * nu, maps, batch=nb)
    torch.cuda.synchronize()
    np.testing.assert_allclose(dC.cpu().numpy(), ref, rtol=0, atol=1e-12)


@pytest.mark.parametrize("m,n", [(16, 2), (256, 64), (257, 33), (5000, 12), (70000, 64), (1000, 1), (64, 64)])
def test_qr_pos(tt, m, n):
    import torch
    rng = np.random.default_rng(m + n)
    Y = rng.standard_normal((m, n))
    dY = _dev(Y)
    dR = torch.empty(n, n, dtype=torch.float64, device="cuda")
    tt.qr_pos(dY, dR)
    torch.cuda.synchronize()
    Q, R = dY.cpu().numpy(), dR.cpu().numpy()
    assert np.all(np.diag(R) >= 0) and np.allclose(R, np.triu(R))
    assert np.abs(Q.T @ Q - np.eye(n)).max() < 1e-13
    assert np.abs(Q @ R - Y).max() < 1e-12 * np.abs(Y).max() * np.sqrt(m)
    # uniqueness: LAPACK's QR with the signs moved to R_ii > 0
    Ql, Rl = np.linalg.qr(Y)
    d = np.sign(np.diag(Rl))
    assert np.abs(Q - Ql * d).max() < 1e-10


def test_qr_pos_rank_deficient(tt):
    import torch
    rng = np.random.default_rng(3)
    m, n, rk = 3000, 24, 9
    Y = rng.standard_normal((m, rk)) @ rng.standard_normal((rk, n))
    Y[:, 5] = 0.0
    dY = _dev(Y)
    dR = torch.empty(n, n, dtype=torch.float64, device="cuda")
    tt.qr_pos(dY, dR)
    Q, R = dY.cpu().numpy(), dR.cpu().numpy()
    assert np.abs(Q.T @ Q - np.eye(n)).max() < 1e-12
    assert np.abs(Q @ R - Y).max() < 1e-11 * np.abs(Y).max()


@pytest.mark.parametrize("m,n", [(64, 64), (12, 12), (33, 7), (300, 129), (1, 1), (40, 64)])
def test_jacobi_svd(tt, m, n):
    import torch
    rng = np.random.default_rng(m * 3 + n)
    G = rng.standard_normal((m, n)) * np.logspace(0, -6, n)
    dG = _dev(G.T)                       # row j = column j
    dV = torch.empty(n, n, dtype=torch.float64, device="cuda")
    ds = torch.empty(n, dtype=torch.float64, device="cuda")
    tt.jacobi_svd(dG, dV, ds)
    Us, V, s = dG.cpu().numpy().T, dV.cpu().numpy().T, ds.cpu().numpy()
    sl = np.linalg.svd(G, compute_uv=False)
    k = min(m, n)
    assert np.abs(s[:k] - sl).max() < 1e-13 * sl[0]
    assert np.all(np.diff(s) <= 0)
    assert np.abs(V.T @ V - np.eye(n)).max() < 1e-13
    assert np.abs(G @ V - Us).max() < 1e-13 * sl[0]
    Un = Us[:, :k] / s[:k]
    assert np.abs(Un.T @ Un - np.eye(k)).max() < 1e-9   # tiny singular values: columns less orthogonal


def test_jacobi_symmetric_psd_eig(tt):
    import torch
    rng = np.random.default_rng(11)
    n, rk = 96, 40
    B = rng.standard_normal((n, rk)) * np.logspace(0, -5, rk)
    S = B @ B.T
    dG = _dev(S)
    dV = torch.empty(n, n, dtype=torch.float64, device="cuda")
    ds = torch.empty(n, dtype=torch.float64, device="cuda")
    tt.jacobi_svd(dG, dV, ds)
    lam, V = ds.cpu().numpy(), dV.cpu().numpy().T
    ll = np.linalg.eigvalsh(S)[::-1]
    assert np.abs(lam - np.maximum(ll, 0)).max() < 1e-13 * ll[0]
    assert np.abs(S @ V[:, :rk] - V[:, :rk] * lam[:rk]).max() < 1e-12 * ll[0]


@pytest.mark.parametrize("n", [1, 31, 4096, 1 << 20, (1 << 22) + 3])
def test_norm_and_trace_reductions(tt, n):
    import torch
    rng = np.random.default_rng(n)
    x, y = rng.standard_normal(n), rng.standard_normal(n)
    dx, dy = _dev(x), _dev(y)
    out = torch.empty(2, dtype=torch.float64, device="cuda")
    tt.sumsq(dx, out[0:1])
    tt.dot(dx, dy, out[1:2])
    o = out.cpu().numpy()
    assert abs(o[0] - np.sum(x * x)) < 1e-13 * n
    assert abs(o[1] - np.sum(x * y)) < 1e-13 * n
    tt.scale_by_rsqrt(dx, out[0:1])
    np.testing.assert_allclose(dx.cpu().numpy(), x / np.linalg.norm(x), rtol=1e-14, atol=0)


@pytest.mark.parametrize("n", [1, 7, 64, 65, 200, 320, 1024])
def test_cholesky_and_triangular_inverse(tt, n):
    """Blocked Cholesky (register-tiled 64x64 diagonal kernel + tensor-GEMM panels) and the
    block-doubling triangular inverse against numpy on a well-conditioned SPD matrix."""
    import torch
    rng = np.random.default_rng(n)
    B = rng.standard_normal((n, n + 5))
    A = B @ B.T + 0.5 * n * np.eye(n)
    dA = _dev(A)
    dLi = torch.empty(n, n, dtype=torch.float64, device="cuda")
    assert tt.cholesky(dA, dLi)
    L, Li = dA.cpu().numpy(), dLi.cpu().numpy()
    Lr = np.linalg.cholesky(A)
    assert np.abs(np.triu(L, 1)).max() == 0.0 and np.abs(np.triu(Li, 1)).max() == 0.0
    assert np.abs(L - Lr).max() < 1e-12 * np.abs(Lr).max()
    assert np.abs(Li @ Lr - np.eye(n)).max() < 1e-12


def test_cholesky_flags_indefinite(tt):
    import torch
    A = np.eye(100)
    A[70, 70] = -1.0
    assert not tt.cholesky(_dev(A))
    # the relative diagonal shift makes a semidefinite matrix factorisable
    v = np.ones((100, 1))
    assert tt.cholesky(_dev(v @ v.T), shift_rel=1e-10)


@pytest.mark.parametrize("m,n,passes", [(1024, 64, 2), (4096, 33, 2), (50000, 64, 2), (2048, 16, 3)])
def test_cholqr(tt, m, n, passes):
    """Asynchronous Cholesky-QR against LAPACK's QR (unique with R_ii > 0) on a block of
    condition number ~1e3."""
    import torch
    rng = np.random.default_rng(m + n)
    Y = rng.standard_normal((m, n)) * np.logspace(0, -3, n)
    dY = _dev(Y)
    dR = torch.empty(n, n, dtype=torch.float64, device="cuda")
    assert tt.cholqr(dY, dR, passes=passes)
    Q, R = dY.cpu().numpy(), dR.cpu().numpy()
    assert np.abs(Q.T @ Q - np.eye(n)).max() < 1e-13
    assert np.abs(Q @ R - Y).max() < 1e-12 * np.abs(Y).max() * np.sqrt(m)
    Ql, Rl = np.linalg.qr(Y)
    d = np.sign(np.diag(Rl))
    assert np.abs(Q - Ql * d).max() < 1e-9


def test_cholqr_single_shifted_pass_spans_the_block(tt):
    """One shifted pass (what the subspace iterations use between Ritz steps): not orthonormal to
    rounding, but the same column space and a well-conditioned basis."""
    rng = np.random.default_rng(5)
    Y = rng.standard_normal((1024, 64)) * np.logspace(0, -5, 64)
    dY = _dev(Y)
    assert tt.cholqr(dY, None, passes=1, shift_rel=1e-13)
    Q = dY.cpu().numpy()
    assert np.abs(Q.T @ Q - np.eye(64)).max() < 1e-2
    Qr, _ = np.linalg.qr(Y)
    assert np.abs(Q - Qr @ (Qr.T @ Q)).max() < 1e-9


@pytest.mark.parametrize("n,grid,iters", [(1024, 16, 6), (1024, 8, 6), (256, 32, 8), (289, 7, 8), (400, 64, 8), (1000, 9, 6)])
def test_subspace_iteration_fused(tt, n, grid, iters):
    """The squeezer's subspace iteration as one resident grid (sq_iter.cu; Eq. 12, DESIGN.md
    "Squeezers") against LAPACK: on a matrix whose singular values fall off as 10^(-i/16) (s_64 = 1e-4 s_1: the block
    stays well inside what two Cholesky-QR passes can orthonormalise), `iters` iterations with a block of 64 give
    orthonormal Q, Qt, the factorisation F^T Q = Qt R, and in R the leading 32 singular values of F to 1e-12
    (neglected part (s_65/s_32)^(2 iters + 1) = 1e-27 at 6 iterations).  Sizes: several row blocks per CTA, one
    row block per CTA, n odd (scalar operand loads), n not a multiple of 8 (ragged last block)."""
    import torch
    rng = np.random.default_rng(n + grid)
    Ul, _ = np.linalg.qr(rng.standard_normal((n, n)))
    Vr, _ = np.linalg.qr(rng.standard_normal((n, n)))
    sv = 10.0 ** (-np.arange(n) / 16.0)
    sv[100:] = sv[100] * 10.0 ** (-np.arange(n - 100) / 400.0)     # a long, nearly flat tail below 1e-6
    F = (Ul * sv) @ Vr.T
    start = rng.standard_normal((n, 64))
    dF, dS = _dev(F), _dev(start)
    dQ = torch.zeros(n, 64, dtype=torch.float64, device="cuda")
    dQt = torch.zeros(n, 64, dtype=torch.float64, device="cuda")
    dR = torch.zeros(64, 64, dtype=torch.float64, device="cuda")
    dmm = torch.zeros(4, dtype=torch.float64, device="cuda")
    assert tt.subspace_iteration(dF, dS, dQ, dQt, iters, grid=grid, R=dR, minmax=dmm)
    Q, Qt, R, mm = dQ.cpu().numpy(), dQt.cpu().numpy(), dR.cpu().numpy(), dmm.cpu().numpy()
    assert np.abs(Q.T @ Q - np.eye(64)).max() < 1e-13
    assert np.abs(Qt.T @ Qt - np.eye(64)).max() < 1e-13
    assert np.abs(np.tril(R, -1)).max() == 0.0
    assert np.abs(F.T @ Q - Qt @ R).max() < 1e-14
    s_it = np.linalg.svd(R, compute_uv=False)
    assert np.abs(s_it[:32] - sv[:32]).max() < 1e-12, np.abs(s_it[:32] - sv[:32]).max()
    assert 0 < mm[0] <= mm[1] and 0 < mm[2] <= mm[3]
    # the span of Q holds the leading left singular vectors
    P = Ul[:, :32] - Q @ (Q.T @ Ul[:, :32])
    assert np.abs(P * sv[:32]).max() < 1e-12


@pytest.mark.parametrize("M,N,K", [(1000, 64, 300), (4096, 40, 1024), (130, 64, 20000), (40, 3000, 256),
                                   (1024, 1024, 32768), (200, 200, 9000)])
def test_tensor_gemm_tile_variants(tt, M, N, K):
    """Shapes that select the 128x64 tile, the operand swap for short-and-wide outputs, and the
    128x128 tile with split-K."""
    import torch
    rng = np.random.default_rng(M + N + K)
    A, B = rng.standard_normal((M, K)), rng.standard_normal((K, N))
    dA, dB = _dev(A), _dev(B)
    dC = torch.empty(M, N, dtype=torch.float64, device="cuda")
    maps = dict(am=[(M, K)], ak=[(K, 1)], bk=[(K, N)], bn=[(N, 1)], cm=[(M, N)], cn=[(N, 1)])
    tt.tensor_gemm(dA, dB, dC, M, N, K, maps)
    torch.cuda.synchronize()
    np.testing.assert_allclose(dC.cpu().numpy(), A @ B, rtol=0, atol=1e-11 * np.sqrt(K))


@pytest.mark.parametrize("M,N,K", [(20000, 32, 32), (16384, 64, 64), (70001, 17, 33), (33000, 6, 6),
                                   (32, 32, 50000), (64, 64, 16384), (13, 40, 70001), (6, 6, 20000)])
def test_tensor_gemm_tall_skinny_streaming(tt, M, N, K):
    """The HBM-bound tall-and-skinny shapes (ts.cu): rows x K times K x N with <= 64 columns, and the
    (M x rows)(rows x N) products behind the Gram matrices of the Cholesky-QR passes."""
    import torch
    rng = np.random.default_rng(M + 3 * N + 7 * K)
    A, B = rng.standard_normal((M, K)), rng.standard_normal((K, N))
    dA, dB = _dev(A), _dev(B)
    dC = torch.full((M, N), 7.0, dtype=torch.float64, device="cuda")
    maps = dict(am=[(M, K)], ak=[(K, 1)], bk=[(K, N)], bn=[(N, 1)], cm=[(M, N)], cn=[(N, 1)])
    tt.tensor_gemm(dA, dB, dC, M, N, K, maps)
    torch.cuda.synchronize()
    np.testing.assert_allclose(dC.cpu().numpy(), A @ B, rtol=0, atol=1e-11 * np.sqrt(K))
    # A^T as the left operand (its small index contiguous): C2 = A^T-layout product, plus accumulate
    if M <= 64:
        At = np.ascontiguousarray(A.T)                      # K x M, element (k, m) at k*M + m
        dAt = _dev(At)
        dC2 = torch.full((M, N), 1.0, dtype=torch.float64, device="cuda")
        maps2 = dict(am=[(M, 1)], ak=[(K, M)], bk=[(K, N)], bn=[(N, 1)], cm=[(M, N)], cn=[(N, 1)])
        tt.tensor_gemm(dAt, dB, dC2, M, N, K, maps2, alpha=0.5, accumulate=True)
        torch.cuda.synchronize()
        np.testing.assert_allclose(dC2.cpu().numpy(), 1.0 + 0.5 * (A @ B), rtol=0, atol=1e-11 * np.sqrt(K))


@pytest.mark.parametrize("n", [1, 2, 7, 100001])
def test_device_generator_equals_host_generator(tt, n):
    """The library's device implementation of the seeded Gaussian recipe against the shared host module
    (what the oracle draws from): same values up to last-bit differences of log / sincos."""
    import torch
    import seeded_inputs as si
    out = torch.empty(n, dtype=torch.float64, device="cuda")
    tt.fill_gauss(out, 20241216, 11, 3)
    ref = si.gauss(si.subseed(20241216, 11, 3), n)
    got = out.cpu().numpy()
    assert np.abs(got - ref).max() <= 4e-15
    if n > 1000:
        assert abs(got.mean()) < 0.02 and abs(got.std() - 1.0) < 0.02


def test_tensor_gemm_randomised_shapes_and_layouts(tt):
    """Seeded sweep over shapes (ragged tails, all three CTA tiles, split-K, short and long summed index) and
    operand layouts (either index of A, B contiguous; odd leading dimensions defeat the 16-byte copies)."""
    import torch
    rng = np.random.default_rng(20241104)
    sizes_mn = [1, 5, 17, 33, 64, 65, 96, 130, 257, 520, 1030]
    sizes_k = [1, 3, 16, 31, 33, 64, 100, 257, 1025, 4100]
    for case in range(60):
        M, N, K = int(rng.choice(sizes_mn)), int(rng.choice(sizes_mn)), int(rng.choice(sizes_k))
        if case % 10 == 0:
            M, N, K = int(rng.choice([2048, 3000])), int(rng.choice([40, 64, 200])), int(rng.choice([32, 64, 700]))
        a_kfast, b_kfast = bool(rng.integers(2)), bool(rng.integers(2))
        pad_a, pad_b = int(rng.integers(3)), int(rng.integers(3))
        A, B = rng.standard_normal((M, K)), rng.standard_normal((K, N))
        if a_kfast:                      # A stored [m][k] with leading dimension K + pad
            bufA = np.zeros((M, K + pad_a)); bufA[:, :K] = A
            am, ak = [(M, K + pad_a)], [(K, 1)]
        else:                            # A stored [k][m]
            bufA = np.zeros((K, M + pad_a)); bufA[:, :M] = A.T
            am, ak = [(M, 1)], [(K, M + pad_a)]
        if b_kfast:                      # B stored [n][k]
            bufB = np.zeros((N, K + pad_b)); bufB[:, :K] = B.T
            bk, bn = [(K, 1)], [(N, K + pad_b)]
        else:                            # B stored [k][n]
            bufB = np.zeros((K, N + pad_b)); bufB[:, :N] = B
            bk, bn = [(K, N + pad_b)], [(N, 1)]
        C0 = rng.standard_normal((M, N))
        acc = bool(rng.integers(2))
        alpha = float(rng.choice([1.0, -0.5]))
        dA, dB, dC = _dev(bufA), _dev(bufB), _dev(C0)
        maps = dict(am=am, ak=ak, bk=bk, bn=bn, cm=[(M, N)], cn=[(N, 1)])
        tt.tensor_gemm(dA, dB, dC, M, N, K, maps, alpha=alpha, accumulate=acc)
        torch.cuda.synchronize()
        ref = alpha * (A @ B) + (C0 if acc else 0.0)
        err = np.abs(dC.cpu().numpy() - ref).max()
        assert err <= 1e-11 * np.sqrt(K) * 4, (case, M, N, K, a_kfast, b_kfast, pad_a, pad_b, acc, err)


@pytest.mark.parametrize("a_kfast", [False, True])
@pytest.mark.parametrize("b_kfast", [False, True])
@pytest.mark.parametrize("pad", [0, 1])
def test_tensor_gemm_persistent_tile_all_layouts(tt, a_kfast, b_kfast, pad):
    """The persistent 128x128 tile (gemm_p.cu): every operand layout (either index contiguous: the four
    swizzled shared-memory tile formats), 16-byte and 8-byte copies (an odd leading dimension defeats the
    16-byte path), ragged M / N / K tails, more tiles than SMs (several tiles per CTA: the pipeline runs
    across tile boundaries), alpha and accumulation, 16-byte and scalar epilogue stores."""
    import torch
    rng = np.random.default_rng(7 + 2 * a_kfast + 4 * b_kfast + 8 * pad)
    for (M, N, K, batch) in ((1500, 1301 + pad, 100, 1), (2100, 2048, 77, 1), (520, 524, 70, 6), (1024, 1024, 4100, 1)):
        A, B = rng.standard_normal((batch, M, K)), rng.standard_normal((batch, K, N))
        if a_kfast:
            bufA = np.zeros((batch, M, K + pad)); bufA[:, :, :K] = A
            am, ak, ab = [(M, K + pad)], [(K, 1)], [(batch, M * (K + pad))]
        else:
            bufA = np.zeros((batch, K, M + pad)); bufA[:, :, :M] = A.transpose(0, 2, 1)
            am, ak, ab = [(M, 1)], [(K, M + pad)], [(batch, K * (M + pad))]
        if b_kfast:
            bufB = np.zeros((batch, N, K + pad)); bufB[:, :, :K] = B.transpose(0, 2, 1)
            bk, bn, bb = [(K, 1)], [(N, K + pad)], [(batch, N * (K + pad))]
        else:
            bufB = np.zeros((batch, K, N + pad)); bufB[:, :, :N] = B
            bk, bn, bb = [(K, N + pad)], [(N, 1)], [(batch, K * (N + pad))]
        C0 = rng.standard_normal((batch, M, N))
        dA, dB, dC = _dev(bufA), _dev(bufB), _dev(C0)
        maps = dict(am=am, ak=ak, bk=bk, bn=bn, cm=[(M, N)], cn=[(N, 1)], ab=ab, bb=bb, cb=[(batch, M * N)])
        tt.tensor_gemm(dA, dB, dC, M, N, K, maps, batch=batch, alpha=-0.5, accumulate=True)
        torch.cuda.synchronize()
        ref = -0.5 * np.einsum("bmk,bkn->bmn", A, B) + C0
        err = np.abs(dC.cpu().numpy() - ref).max()
        assert err <= 4e-11 * np.sqrt(K), (M, N, K, batch, err)


def test_tensor_gemm_tma_producer_matches(tt):
    """The TMA-fed producer of the persistent tile (gemm_tma.cu: cp.async.bulk.tensor + SWIZZLE_128B boxes,
    the stage refilled by the last warp to leave it) against numpy and against the cp.async producer, on plain
    row-major operands with ragged M / N / K tails, alpha and accumulation."""
    import torch
    import paper_2412_14104_b200 as t
    rng = np.random.default_rng(5)
    for (M, N, K) in ((1500, 1302, 100), (2100, 2048, 77), (4096, 1024, 1000)):
        A, B, C0 = rng.standard_normal((M, K)), rng.standard_normal((K, N)), rng.standard_normal((M, N))
        maps = dict(am=[(M, K)], ak=[(K, 1)], bk=[(K, N)], bn=[(N, 1)], cm=[(M, N)], cn=[(N, 1)])
        res = []
        for mask in (0, t.ROUTE_TMA_PRODUCER):
            tt.set_routes(mask)
            try:
                dA, dB, dC = _dev(A), _dev(B), _dev(C0)
                tt.tensor_gemm(dA, dB, dC, M, N, K, maps, alpha=-0.5, accumulate=True)
                torch.cuda.synchronize()
                res.append(dC.cpu().numpy())
            finally:
                tt.set_routes(0)
        ref = -0.5 * (A @ B) + C0
        assert np.abs(res[1] - ref).max() <= 4e-11 * np.sqrt(K), (M, N, K)
        assert np.abs(res[1] - res[0]).max() <= 1e-12 * np.sqrt(K), (M, N, K)


@pytest.mark.parametrize("b_kfast", [False, True])
def test_tensor_gemm_triangular_b_hint(tt, b_kfast):
    """tri_b (bit 1 of tatrg_tensor_gemm's `accumulate`): B[k][n] = 0 for k > n, as in Q1 = T L^-T of the bond
    swap's Cholesky-QR.  The persistent tile skips the k tiles of zeros and walks the column tiles in
    pairs of equal work; the result is the same bit for bit as without the hint, and equal to numpy's.  Cases: an
    even number of column tiles (hint taken) with ragged M, K < N, K > N, batch 2; an odd number of column tiles
    and a split-K shape (hint dropped)."""
    import torch
    rng = np.random.default_rng(11 + b_kfast)
    for (M, N, K, batch) in ((4100, 1024, 1024, 1), (3000, 768, 512, 2), (2500, 1000, 1200, 1), (4096, 640, 640, 1),
                             (256, 256, 20000, 1)):
        A = rng.standard_normal((batch, M, K))
        B = np.triu(rng.standard_normal((batch, K, N)))          # zero for k > n
        if b_kfast:
            bufB = np.ascontiguousarray(B.transpose(0, 2, 1))
            bk, bn = [(K, 1)], [(N, K)]
        else:
            bufB = B
            bk, bn = [(K, N)], [(N, 1)]
        C0 = rng.standard_normal((batch, M, N))
        maps = dict(am=[(M, K)], ak=[(K, 1)], bk=bk, bn=bn, cm=[(M, N)], cn=[(N, 1)],
                    ab=[(batch, M * K)], bb=[(batch, K * N)], cb=[(batch, M * N)])
        res = []
        for hint in (False, True):
            dA, dB, dC = _dev(A), _dev(bufB), _dev(C0)
            tt.tensor_gemm(dA, dB, dC, M, N, K, maps, batch=batch, alpha=0.75, accumulate=True, tri_b=hint)
            torch.cuda.synchronize()
            res.append(dC.cpu().numpy())
        ref = 0.75 * np.einsum("bmk,bkn->bmn", A, B) + C0
        assert np.abs(res[1] - ref).max() <= 4e-11 * np.sqrt(K), (M, N, K, batch)
        assert np.array_equal(res[0], res[1]), (M, N, K, batch)


@pytest.mark.parametrize("dims", [(8, 8, 8, 32, 32, 32, 32), (6, 10, 6, 24, 36, 30, 36), (4, 16, 8, 32, 30, 32, 36)])
def test_tensor_gemm_persistent_tile_composite_maps(tt, dims):
    """Step (ii) of Eq. 13 in miniature, P[x,k,w,l,g] = sum_{a,T} EM[x,k,a,T,w] F[a,l,T,g], through the
    persistent tile: rows, columns, the summed index and the output are all composites of two or three tensor legs.
    A power-of-two faster leg of the summed index takes the shift-and-mask evaluation of its map (gemm_p.cu:
    Loader::load), other sizes the mixed-radix divisions; the third case mixes both kinds of leg sizes."""
    import torch
    x, k, a, T, w, l, g = dims
    rng = np.random.default_rng(sum(dims))
    EM, F = rng.standard_normal((x, k, a, T, w)), rng.standard_normal((a, l, T, g))
    M, N, K = x * k * w, l * g, a * T
    maps = dict(am=[(w, 1), (k, a * T * w), (x, k * a * T * w)], ak=[(T, w), (a, T * w)],
                bk=[(T, g), (a, l * T * g)], bn=[(g, 1), (l, T * g)],
                cm=[(w, l * g), (k, w * l * g), (x, k * w * l * g)], cn=[(g, 1), (l, g)])
    dA, dB = _dev(EM), _dev(F)
    dC = torch.zeros(x * k * w * l * g, dtype=torch.float64, device="cuda")
    tt.tensor_gemm(dA, dB, dC, M, N, K, maps)
    torch.cuda.synchronize()
    ref = np.einsum("xkaTw,alTg->xkwlg", EM, F)
    err = np.abs(dC.cpu().numpy().reshape(ref.shape) - ref).max()
    assert err <= 4e-11 * np.sqrt(K), (dims, err)
