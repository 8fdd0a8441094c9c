"""CPU oracle for ATRG / Triad-ATRG coarse-graining of the 4D Ising tensor network.

TEST INFRASTRUCTURE ONLY.  Plain, slow numpy FP64 restatement of the method of
arXiv:2412.14104 (Sugimoto & Sasaki), written from /root/reference/PAPER.md and
the readings listed in DESIGN.md ("Readings").  It shares no code with the CUDA
path (paper_2412_14104_b200/) and must never be imported by it; only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import it.  All random inputs (sketches Omega, gauge references) are passed in
by the caller; this module draws no random numbers.

Notation (Eq. 1): coarse-graining along direction `0` of the
*rotated frame* merges the "upper" site n+0^ and the "lower" site n.  In the
rotated frame the legs are (0 | 1, 2 | 3): 0 = coarse-graining direction,
(1, 2) = the grouped transverse pair that gets the oversampled isometries
(the paper's legs 2, 3), 3 = the lone transverse leg (the paper's leg 4).
Tensors:
    Phi[i0,i1,i2,i3,g], Psi[j0,j1,j2,j3,g] with T = sum_g Phi Psi
    A[i0,i1,i2,i3,a], D[j0,j1,j2,j3,a], sigT[a]
    X[a,i1',i2',i3',g], Y[b,j1,j2,j3,g], sig[g]                      (Eq. 1)
    UA,UX,UY,UD[p,q,k]  (I,J,K,L of Eqs. 8-11), E,F,G,H (Eqs. 4-7)
    M[mu][(up,lo),k], N[mu][k,(up,lo)]  squeezers (Eq. 12)

Pins: tests/test_oracle_pins.py (Onsager, exact enumeration, high-T series,
isometry / projector invariants, brute-force einsum, Triad==ATRG at r*chi>=d2*d3,
RSVD == exact SVD at full width).  Table 2 of the paper: parity unpinned
(temperature, lattice size, q not stated).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

RANK_TOL = 1e-14      # reading G9: numerical rank / Gram eigenvalue cut, relative to the largest
CLUSTER_TOL = 1e-8    # reading G12: singular values closer than this (relative to s_1) form a cluster


# --------------------------------------------------------------------------- helpers
def qr_pos(Y):
    """Thin QR with R_ii >= 0 (unique for full column rank) -- 'qr+' of reading O9."""
    Q, R = np.linalg.qr(Y)
    d = np.sign(np.diag(R)).copy()
    d[d == 0] = 1.0
    return Q * d, d[:, None] * R


def num_rank(s, cap=None, tol=RANK_TOL):
    """Number of values of the descending array s above tol*s[0], capped."""
    if len(s) == 0 or s[0] <= 0:
        return 0
    k = int(np.sum(s > tol * s[0]))
    return k if cap is None else min(cap, k)


def clusters(s, tol=CLUSTER_TOL):
    """Consecutive index ranges [c0,c1) of the descending array s whose neighbouring
    gaps are all <= tol*s[0] (reading G12)."""
    out, c0 = [], 0
    for i in range(1, len(s)):
        if s[i - 1] - s[i] > tol * s[0]:
            out.append((c0, i))
            c0 = i
    out.append((c0, len(s)))
    return out


def min_rel_gap(s, cut):
    """(s[cut-1]-s[cut])/s[0] if a value exists beyond the cut, else inf (logged, reading G12)."""
    if cut <= 0 or cut >= len(s):
        return np.inf
    return float((s[cut - 1] - s[cut]) / s[0])


def sym_eig_desc(S):
    lam, V = np.linalg.eigh(0.5 * (S + S.T))
    return lam[::-1].copy(), V[:, ::-1].copy()


# --------------------------------------------------------------------------- state
@dataclass
class State:
    phi: np.ndarray            # (d1,d2,d3,d4,g) standard frame
    psi: np.ndarray
    log_acc: float             # sum_m 2^-m ln c_m   (reading O8)
    step: int = 0
    beta: float = 0.0
    h: float = 0.0
    history: list = field(default_factory=list)

    @property
    def dims(self):
        return tuple(self.phi.shape)


def init_ising_tensor(beta, h=0.0, active=(1, 1, 1, 1)):
    """Initial tensor, Eqs. 16-17 with reading G1 (square roots restored,
    so that (W W^T)_{ab} = exp(beta s_a s_b)) and G2 (field weight exp(beta h s_a) on the
    site sum, H = -sum s s' - h sum s).  `active[mu]=0` replaces leg pair mu by a dummy leg
    of dimension 1: the same code then runs the d<4 model (pin P1 uses d=2).
    T[i,j] = sum_a Phi0[i,a] Psi0[j,a]."""
    if not (beta > 0 and np.isfinite(beta)):
        raise ValueError("beta must be finite and > 0")
    s = np.array([1.0, -1.0])
    W = np.empty((2, 2))
    W[:, 0] = np.sqrt(np.cosh(beta))
    W[:, 1] = s * np.sqrt(np.sinh(beta))
    dims = [2 if a else 1 for a in active]
    phi = np.ones(dims + [2])
    for mu in range(4):
        if active[mu]:
            shp = [1, 1, 1, 1, 2]
            shp[mu] = 2
            phi = phi * W.T.reshape(shp)           # W[a, i_mu] -> axes (i_mu, a)
    psi = phi * np.exp(beta * h * s).reshape(1, 1, 1, 1, 2)
    st = State(phi=phi, psi=psi, log_acc=0.0, step=0, beta=beta, h=h)
    _normalise(st)
    return st


def _normalise(st):
    """Reading O8/G11: c_m = |Phi|_F |Psi|_F, both scaled to unit norm,
    log_acc += 2^-m ln c_m."""
    nphi = np.linalg.norm(st.phi)
    npsi = np.linalg.norm(st.psi)
    st.phi = st.phi / nphi
    st.psi = st.psi / npsi
    lnc = np.log(nphi) + np.log(npsi)
    st.log_acc += 2.0 ** (-st.step) * lnc
    return lnc


def tensor_trace(st):
    """tTr T = sum_i T_{i;i} = <Phi,Psi> (Eq. 15 closed periodically)."""
    return float(np.sum(st.phi * st.psi))


def log_Z_per_site(st):
    """ln Z / V = sum_{m<=n} 2^-m ln c_m + 2^-n ln tTr T^(n)  (reading O8)."""
    t = tensor_trace(st)
    if not t > 0:
        return float("nan")
    return st.log_acc + 2.0 ** (-st.step) * np.log(t)


def order_parameter_X(st, leg=3):
    """X^(m) = (Tr A)^2 / Tr(A^2), A_kl = sum T_{..k..;..l..} with the other three leg
    pairs traced (`leg` = which direction stays open, paper: the 4th)."""
    g = st.phi.shape[4]
    ph = np.moveaxis(st.phi, leg, 3)
    ps = np.moveaxis(st.psi, leg, 3)
    n = ph.shape[3]
    ph = ph.reshape(-1, n, g)
    ps = ps.reshape(-1, n, g)
    Amat = np.einsum("xkg,xlg->kl", ph, ps)
    return float(np.trace(Amat) ** 2 / np.trace(Amat @ Amat))


# --------------------------------------------------------------------------- frames
def frame_perm(direction):
    """Reading G8: rotated frame for coarse-graining direction `direction` (1..4):
    transverse directions ascending, first two grouped, last lone."""
    d = direction - 1
    t = [m for m in range(4) if m != d]
    return [d] + t


# --------------------------------------------------------------------------- O2
def canonicalise(phi, psi, ref_ad=None):
    """Reading O2 (PAPER.md:37 'A ... D are the isometries'): thin QR of Phi and Psi,
    SVD of R_Phi R_Psi^T, keep the numerical rank; A = Q_Phi u, D = Q_Psi v.
    Exact: T already has rank <= g.  Gauge fixed per reading G12 with the reference
    ref_ad(a) -> [(i0..i3), a] (a callable, asked for the actual rank a)."""
    shp = phi.shape[:4]
    g = phi.shape[4]
    Qp, Rp = qr_pos(phi.reshape(-1, g))
    Qs, Rs = qr_pos(psi.reshape(-1, g))
    u, sT, vt = np.linalg.svd(Rp @ Rs.T)
    a = num_rank(sT)
    A = Qp @ u[:, :a]
    D = Qs @ vt[:a].T
    sT = sT[:a].copy()
    if ref_ad is not None:
        P = A.T @ ref_ad(a)
        for c0, c1 in clusters(sT):
            Qw, _ = qr_pos(P[c0:c1, c0:c1])
            A[:, c0:c1] = A[:, c0:c1] @ Qw
            D[:, c0:c1] = D[:, c0:c1] @ Qw
    return A.reshape(shp + (a,)), sT, D.reshape(shp + (a,))


# --------------------------------------------------------------------------- O9 / O3
def rsvd(apply, apply_t, omega, q, keep):
    """Reading O9 (RSVD named at PAPER.md:25, :106; subspace iteration after
    Halko-Martinsson-Tropp).  Returns left[:, :k], s[:k], right[:, :k], and the full
    width-l spectrum, k = min(keep, numerical rank)."""
    Q, _ = qr_pos(apply(omega))
    for _ in range(q):
        Qt, _ = qr_pos(apply_t(Q))
        Q, _ = qr_pos(apply(Qt))
    Bt = apply_t(Q)                      # B^T = Op^T Q   (n x l)
    Qb, Rb = qr_pos(Bt)                  # B^T = Q_B R_B
    u, s, vt = np.linalg.svd(Rb.T)       # R_B^T = u s v^T  =>  B = u s (Q_B v)^T
    k = num_rank(s, keep)
    return Q @ u[:, :k], s[:k].copy(), Qb @ vt[:k].T, s


def bond_swap(A, sT, D, chi, r, q, omega):
    """Reading O3 (Table 1 row 1): upper site T = A sigT D^T, lower site the
    same tensor.  B[al; c,J] = sigT[al] D[(c,J),al] (upper, c = its j0 leg),
    C[(c,I'); be] = A[(c,I'),be] sigT[be] (lower, c = its i0 leg);
    M[(al,I'),(be,J)] = sum_c B C, never formed.  RSVD of width l = min(r chi, dim),
    truncated to min(chi, rank).  omega[(be,J), l]."""
    n0, n1, n2, n3, a = A.shape
    nT = n1 * n2 * n3
    dim = a * nT
    ell = min(r * chi, dim)
    assert omega.shape == (dim, ell), (omega.shape, dim, ell)
    Dm = (D * sT).reshape(n0, nT, a)          # [c, J, al]
    Am = (A * sT).reshape(n0, nT, a)          # [c, I', be]

    def apply(w):                              # M w : [(be,J), l] -> [(al,I'), l]
        l = w.shape[1]
        Z = np.einsum("cJa,bJl->cabl", Dm, w.reshape(a, nT, l), optimize=True)
        return np.einsum("cIb,cabl->aIl", Am, Z, optimize=True).reshape(dim, l)

    def apply_t(w):                            # M^T w : [(al,I'), l] -> [(be,J), l]
        l = w.shape[1]
        Z = np.einsum("cIb,aIl->cbal", Am, w.reshape(a, nT, l), optimize=True)
        return np.einsum("cJa,cbal->bJl", Dm, Z, optimize=True).reshape(dim, l)

    left, s, right, s_full = rsvd(apply, apply_t, omega, q, chi)
    g = len(s)
    X = left.reshape(a, n1, n2, n3, g)
    Y = right.reshape(a, n1, n2, n3, g)
    return X, s, Y, s_full


# --------------------------------------------------------------------------- O4
def _pair_op(T5, pair_axes):
    """Matricise the 5-leg tensor T5 as (pair legs) x (rest)."""
    rest = [ax for ax in range(5) if ax not in pair_axes]
    P = np.transpose(T5, list(pair_axes) + rest)
    return P.reshape(T5.shape[pair_axes[0]] * T5.shape[pair_axes[1]], -1)


def isometry(K, Kw, k, q, omega, iso_mode):
    """Reading O4 with G6b: top-k eigenspace of the symmetric PSD operator S = K Kw^T on the
    (leg1, leg2) pair space (Eq. 3), where K Kw^T is A X sig sig X^T A^T etc.
    reduced by the canonical form.  iso_mode='exact': dense eigendecomposition (the paper's
    Eq. 3).  iso_mode='rsvd' (north star): Gaussian sketch omega[(p,q), k] in the leg space,
    Q = qr+(S omega), q times Q = qr+(S Q), Ritz step H = Q^T S Q = u L u^T, U = Q u.
    Returns U[(p,q), k] and the spectrum sqrt(L) (the paper's S^A)."""
    npair = K.shape[0]
    if k >= npair:                              # r chi >= d2 d3: U = identity
        return np.eye(npair), np.zeros(0)
    if iso_mode == "exact":
        lam, V = sym_eig_desc(K @ Kw.T)
        return V[:, :k].copy(), np.sqrt(np.maximum(lam[:k], 0.0))
    assert omega.shape == (npair, k), (omega.shape, npair, k)

    def S(w):
        return K @ (Kw.T @ w)

    Q, _ = qr_pos(S(omega))
    for _ in range(q):
        Q, _ = qr_pos(S(Q))
    lam, u = sym_eig_desc(Q.T @ S(Q))
    return Q @ u, np.sqrt(np.maximum(lam, 0.0))


def make_isometries(A, X, sig, Y, D, chi, r, q, omegas, iso_mode="rsvd"):
    """U^A, U^X, U^Y, U^D.  Canonical form (PAPER.md:41 'we only need to
    consider the SVD of A X sigma'): the Gram over everything but the pair legs reduces to
      U^X: (X sig)(X sig)^T,             U^Y: (Y sig)(Y sig)^T,
      U^A: A R_X A^T, R_X = sum X sig^2 X,  U^D: D R_Y D^T, R_Y = sum Y sig^2 Y."""
    n1, n2 = A.shape[1], A.shape[2]
    k = min(r * chi, n1 * n2)
    a = A.shape[4]
    Xs = X * sig
    Ys = Y * sig
    RX = np.einsum("aIg,bIg->ab", Xs.reshape(a, -1, len(sig)), Xs.reshape(a, -1, len(sig)))
    RY = np.einsum("aIg,bIg->ab", Ys.reshape(a, -1, len(sig)), Ys.reshape(a, -1, len(sig)))
    out, spec = {}, {}
    KX = _pair_op(Xs, (1, 2))
    out["X"], spec["X"] = isometry(KX, KX, k, q, omegas.get("X"), iso_mode)
    KY = _pair_op(Ys, (1, 2))
    out["Y"], spec["Y"] = isometry(KY, KY, k, q, omegas.get("Y"), iso_mode)
    KA = _pair_op(A, (1, 2))
    KAw = _pair_op(A @ RX, (1, 2))
    out["A"], spec["A"] = isometry(KA, KAw, k, q, omegas.get("A"), iso_mode)
    KD = _pair_op(D, (1, 2))
    KDw = _pair_op(D @ RY, (1, 2))
    out["D"], spec["D"] = isometry(KD, KDw, k, q, omegas.get("D"), iso_mode)
    U = {t: out[t].reshape(n1, n2, -1) for t in out}
    return U, spec


# --------------------------------------------------------------------------- O5
def triad_tensors(A, X, sig, Y, D, U):
    """Eqs. 4-7, real case; sigma goes into F only (Eq. 5)."""
    E = np.einsum("xpqta,pqk->xkta", A, U["A"], optimize=True)        # E[i0,kA,i3,al]
    F = np.einsum("apqtg,pqk->aktg", X, U["X"], optimize=True) * sig  # F[al,kX,i3',g]
    G = np.einsum("bpqtg,pqk->bktg", Y, U["Y"], optimize=True)        # G[be,kY,j3,g]
    H = np.einsum("xpqtb,pqk->xktb", D, U["D"], optimize=True)        # H[j0',kD,j3',be]
    return E, F, G, H


# --------------------------------------------------------------------------- O6
def triad_grams(E, F, G, H, U):
    """Gram matrices of Gamma^triad (Eq. 12, reading G10) on the + double
    leg (G^L) and the - double leg (G^R) for the three transverse directions, all of
    E..L included.  The traced legs of the isometries U give deltas (U^T U = 1).
    Index order of every Gram: [(upper, lower), (upper-bar, lower-bar)]."""
    UA, UX, UY, UD = U["A"], U["X"], U["Y"], U["D"]
    HH0 = np.einsum("xktb,xktc->bc", H, H, optimize=True)
    Sm = np.einsum("bktg,cktd,bc->gd", G, G, HH0, optimize=True)     # - half reduced to g x g
    EE0 = np.einsum("xkta,xktb->ab", E, E, optimize=True)
    Sp = np.einsum("aktg,bktd,ab->gd", F, F, EE0, optimize=True)     # + half reduced to g x g
    GL, GR = {}, {}
    # lone leg (rotated leg 3; the paper's mu=4)
    EE3 = np.einsum("xkta,xkub->taub", E, E, optimize=True)
    FF3 = np.einsum("aktg,gd,bkud->atbu", F, Sm, F, optimize=True)
    GL[3] = np.einsum("taub,asbv->tsuv", EE3, FF3, optimize=True)
    GG3 = np.einsum("bktg,gd,ckud->btcu", G, Sp, G, optimize=True)
    HH3 = np.einsum("xktb,xkuc->tbuc", H, H, optimize=True)
    GR[3] = np.einsum("btcu,sbvc->tsuv", GG3, HH3, optimize=True)
    # grouped legs (rotated legs 1, 2; the paper's mu=2,3)
    EEk = np.einsum("xkta,xltb->kalb", E, E, optimize=True)
    FFk = np.einsum("aktg,gd,bltd->kalb", F, Sm, F, optimize=True)
    GGk = np.einsum("bktg,gd,cltd->kblc", G, Sp, G, optimize=True)
    HHk = np.einsum("xktb,xltc->kblc", H, H, optimize=True)
    for mu, (uu, ww) in ((1, ("pqk,rql->pkrl", "pqk,rql->pkrl")),
                         (2, ("qpk,qrl->pkrl", "qpk,qrl->pkrl"))):
        UUA = np.einsum(uu, UA, UA, optimize=True)
        UUX = np.einsum(uu, UX, UX, optimize=True)
        T1 = np.einsum("pkrl,kalb->prab", UUA, EEk, optimize=True)
        T2 = np.einsum("pkrl,kalb->prab", UUX, FFk, optimize=True)
        GL[mu] = np.einsum("prab,qsab->pqrs", T1, T2, optimize=True)
        UUY = np.einsum(ww, UY, UY, optimize=True)
        UUD = np.einsum(ww, UD, UD, optimize=True)
        T3 = np.einsum("pkrl,kblc->prbc", UUY, GGk, optimize=True)
        T4 = np.einsum("pkrl,kblc->prbc", UUD, HHk, optimize=True)
        GR[mu] = np.einsum("prbc,qsbc->pqrs", T3, T4, optimize=True)
    for mu in (1, 2, 3):
        n = GL[mu].shape[0] * GL[mu].shape[1]
        GL[mu] = GL[mu].reshape(n, n)
        GR[mu] = GR[mu].reshape(n, n)
    return GL, GR


def atrg_grams(A, X, sig, Y, D):
    """Original ATRG squeezer Grams: G^L from A X sigma, G^R from sigma Y D only (canonical
    form drops the other half; Table 1 'Squeezer step O(chi^7)')."""
    a = A.shape[4]
    Xs = X * sig
    Ys = Y * sig
    GL, GR = {}, {}
    for mu in (1, 2, 3):
        oth = [m for m in (1, 2, 3) if m != mu]
        AA = np.einsum(A, [0, 1, 2, 3, 4], A, [0] + [m if m != mu else 5 for m in (1, 2, 3)] + [6],
                       [mu, 4, 5, 6], optimize=True)                  # [i_mu, al, ibar_mu, albar]
        XX = np.einsum(Xs, [4, 1, 2, 3, 7], Xs, [6] + [m if m != mu else 5 for m in (1, 2, 3)] + [7],
                       [4, mu, 6, 5], optimize=True)                  # [al, i_mu', albar, ibar_mu']
        GL[mu] = np.einsum("taub,asbv->tsuv", AA, XX, optimize=True)
        YY = np.einsum(Ys, [4, 1, 2, 3, 7], Ys, [6] + [m if m != mu else 5 for m in (1, 2, 3)] + [7],
                       [4, mu, 6, 5], optimize=True)                  # [be, j_mu, bebar, jbar_mu]
        DD = np.einsum(D, [0, 1, 2, 3, 4], D, [0] + [m if m != mu else 5 for m in (1, 2, 3)] + [6],
                       [mu, 4, 5, 6], optimize=True)                  # [j_mu', be, jbar_mu', bebar]
        GR[mu] = np.einsum("btcu,sbvc->tsuv", YY, DD, optimize=True)
        n = GL[mu].shape[0] * GL[mu].shape[1]
        GL[mu] = GL[mu].reshape(n, n)
        GR[mu] = GR[mu].reshape(n, n)
        del oth
    return GL, GR


def squeezer(GLm, GRm, chi, ref=None):
    """Reading O6/G10 (after Ref. [13]): G^L = R1^T R1, G^R = R2 R2^T from
    eigendecompositions (eigenvalues <= 1e-14 max dropped), SVD R1 R2 = U s V^T, keep
    chi' = min(chi, rank); M = R2 V s^-1/2, N = s^-1/2 U^T R1 (so N M = 1).  Gauge fixed per
    reading G12 with the reference ref(k) -> [(up,lo), k] (a callable)."""
    lamL, VL = sym_eig_desc(GLm)
    kl = num_rank(lamL)
    R1 = np.sqrt(lamL[:kl])[:, None] * VL[:, :kl].T
    lamR, VR = sym_eig_desc(GRm)
    kr = num_rank(lamR)
    R2 = VR[:, :kr] * np.sqrt(lamR[:kr])
    u, s, vt = np.linalg.svd(R1 @ R2)
    k = num_rank(s, chi)
    gap = min_rel_gap(s, k)
    isq = 1.0 / np.sqrt(s[:k])
    M = (R2 @ vt[:k].T) * isq
    N = isq[:, None] * (u[:, :k].T @ R1)
    if ref is not None:
        P = N @ ref(k)
        for c0, c1 in clusters(s[:k]):
            Qw, _ = qr_pos(P[c0:c1, c0:c1])
            M[:, c0:c1] = M[:, c0:c1] @ Qw
            N[c0:c1] = Qw.T @ N[c0:c1]
    return M, N, s[:k].copy(), gap


# --------------------------------------------------------------------------- O7
def contract_triad(E, F, G, H, U, Ms, Ns):
    """Eqs. 13-14 verbatim, real case."""
    n1, n2 = U["A"].shape[0], U["A"].shape[1]
    n3 = E.shape[2]
    M1 = Ms[1].reshape(n1, n1, -1)
    M2 = Ms[2].reshape(n2, n2, -1)
    M3 = Ms[3].reshape(n3, n3, -1)
    N1 = Ns[1].reshape(-1, n1, n1)
    N2 = Ns[2].reshape(-1, n2, n2)
    N3 = Ns[3].reshape(-1, n3, n3)
    Q = np.einsum("pqk,rsl,prm,qsn->klmn", U["A"], U["X"], M1, M2, optimize=True)
    EM = np.einsum("xkta,tuw->xkauw", E, M3, optimize=True)
    P = np.einsum("xkauw,alug->xkwlg", EM, F, optimize=True)
    phi = np.einsum("xkwlg,klmn->xmnwg", P, Q, optimize=True)
    Qp = np.einsum("pqk,rsl,mpr,nqs->klmn", U["Y"], U["D"], N1, N2, optimize=True)
    HN = np.einsum("xlub,wtu->xlbtw", H, N3, optimize=True)
    Pp = np.einsum("xlbtw,bktg->xlwkg", HN, G, optimize=True)
    psi = np.einsum("xlwkg,klmn->xmnwg", Pp, Qp, optimize=True)
    return phi, psi


def contract_atrg(A, X, sig, Y, D, Ms, Ns):
    """Plain ATRG contraction without triads, O(chi^9) (Table 1 :113):
    Phi = sum A (X sigma) M1 M2 M3, Psi = sum Y D N1 N2 N3; sigma stays on the Phi side as in
    the triad form (it sits in F, Eq. 5).

    The two five-operand sums
        Phi[x,m,n,w,g] = sum A[x,p,q,t,a] (X sigma)[a,r,s,u,g] M1[p,r,m] M2[q,s,n] M3[t,u,w]
        Psi[x,m,n,w,g] = sum Y[b,p,q,t,g] D[x,r,s,u,b] N1[m,p,r] N2[n,q,s] N3[w,t,u]
    are evaluated pairwise in the order of Table 1's cost count (squeezer of the first pair leg,
    then the O(chi^9) product with the second site over (bond, pair leg), then the other two
    squeezers), one value of the pass-through leg x at a time: x is a free index of both sums, and
    the chi^7-sized intermediate of the whole tensor would not fit host memory at chi = 24
    (BASELINE.json config 4).  Pinned by the 14-leg brute force of test_P7."""
    n0, n1, n2, n3 = A.shape[0], A.shape[1], A.shape[2], A.shape[3]
    M1 = Ms[1].reshape(n1, n1, -1)
    M2 = Ms[2].reshape(n2, n2, -1)
    M3 = Ms[3].reshape(n3, n3, -1)
    N1 = Ns[1].reshape(-1, n1, n1)
    N2 = Ns[2].reshape(-1, n2, n2)
    N3 = Ns[3].reshape(-1, n3, n3)
    Xs = X * sig
    g = len(sig)
    phi = np.empty((n0, M1.shape[2], M2.shape[2], M3.shape[2], g))
    psi = np.empty((n0, N1.shape[0], N2.shape[0], N3.shape[0], g))
    for x in range(n0):
        t = np.einsum("pqta,prm->qtarm", A[x], M1, optimize=True)
        t = np.einsum("qtarm,arsug->qtmsug", t, Xs, optimize=True)       # the O(chi^9) product
        t = np.einsum("qtmsug,qsn->tmnug", t, M2, optimize=True)
        phi[x] = np.einsum("tmnug,tuw->mnwg", t, M3, optimize=True)
        t = np.einsum("rsub,mpr->subpm", D[x], N1, optimize=True)
        t = np.einsum("subpm,bpqtg->sumqtg", t, Y, optimize=True)        # the O(chi^9) product
        t = np.einsum("sumqtg,nqs->umntg", t, N2, optimize=True)
        psi[x] = np.einsum("umntg,wtu->mnwg", t, N3, optimize=True)
    return phi, psi


# --------------------------------------------------------------------------- one step
def coarse_grain(st, direction, chi, r, q, inputs, mode="triad", iso_mode="rsvd"):
    """One coarse-graining step along `direction` (1..4): readings O2-O8.
    `inputs(which, rows, cols)` returns the seeded Gaussian matrix for
    which in {'swap','A','X','Y','D','ref_ad','ref_sq1','ref_sq2','ref_sq3'}
    (row-major in the rotated frame); the bond-dependent ones are requested with the
    actual bond after canonicalisation.  Returns a record of spectra."""
    if direction not in (1, 2, 3, 4) or chi < 1 or r < 1 or q < 0:
        raise ValueError("bad arguments")
    perm = frame_perm(direction)
    phi = np.transpose(st.phi, perm + [4])
    psi = np.transpose(st.psi, perm + [4])
    n0, n1, n2, n3, _ = phi.shape
    rec = {"direction": direction, "dims_in": st.dims}
    # O2
    A, sT, D = canonicalise(phi, psi, lambda a_: inputs("ref_ad", n0 * n1 * n2 * n3, a_))
    a = len(sT)
    rec["sigmaT"] = sT
    # O3
    dim = a * n1 * n2 * n3
    ell = min(r * chi, dim)
    X, sig, Y, s_full = bond_swap(A, sT, D, chi, r, q, inputs("swap", dim, ell))
    rec["sigma_swap"] = sig
    rec["gap_swap"] = min_rel_gap(s_full, len(sig))
    # O4-O7
    if mode == "triad":
        k = min(r * chi, n1 * n2)
        om = {}
        if k < n1 * n2 and iso_mode == "rsvd":
            om = {t: inputs(t, n1 * n2, k) for t in ("A", "X", "Y", "D")}
        U, spec = make_isometries(A, X, sig, Y, D, chi, r, q, om, iso_mode)
        for t in "AXYD":
            rec["S" + t] = spec[t]
        rec["U"] = U                      # record only (tests compare the projectors U U^T)
        E, F, G, H = triad_tensors(A, X, sig, Y, D, U)
        GL, GR = triad_grams(E, F, G, H, U)
    elif mode == "atrg":
        GL, GR = atrg_grams(A, X, sig, Y, D)
    else:
        raise ValueError(mode)
    Ms, Ns = {}, {}
    for mu in (1, 2, 3):
        nn = (n1, n2, n3)[mu - 1]
        Ms[mu], Ns[mu], s_mu, gap = squeezer(
            GL[mu], GR[mu], chi, lambda k_, mu=mu, nn=nn: inputs("ref_sq%d" % mu, nn * nn, k_))
        rec["s%d" % mu] = s_mu
        rec["gap_s%d" % mu] = gap
    if mode == "triad":
        phi2, psi2 = contract_triad(E, F, G, H, U, Ms, Ns)
    else:
        phi2, psi2 = contract_atrg(A, X, sig, Y, D, Ms, Ns)
    # back to the standard frame
    inv = list(np.argsort(perm)) + [4]
    st.phi = np.ascontiguousarray(np.transpose(phi2, inv))
    st.psi = np.ascontiguousarray(np.transpose(psi2, inv))
    st.step += 1
    rec["ln_c"] = _normalise(st)
    rec["dims_out"] = st.dims
    st.history.append(rec)
    return rec
