"""Independent references that pin the oracle (what the mathematics fixes, not the oracle).

* brute_force_lnZ: exact enumeration of the Ising partition function on a tiny periodic
  4D lattice with extents (L1..L4) (extent 1 = self bond, extent 2 = double bond), the
  closure the tensor trace builds (Eq. 15; SURVEY.md 8(c) pin P2).
* onsager_lnZ: Onsager's closed form for the square lattice (pin P1).
* ht_series_lnZ: high-temperature series on the d-dimensional hypercubic lattice to v^8 (pin P3).
"""
import itertools

import numpy as np


def brute_force_lnZ(beta, h, extents):
    """ln Z / V by summing over all 2^V spin configurations.
    H = -sum_<nn'> s s' - h sum s, weight exp(-beta H); every site owns one bond per
    direction to its +mu neighbour (periodic), so extent 1 gives a self bond (s*s = 1) and
    extent 2 gives two bonds between the same pair."""
    L = list(extents)
    V = int(np.prod(L))
    assert V <= 20
    coords = list(itertools.product(*[range(l) for l in L]))
    index = {c: i for i, c in enumerate(coords)}
    bonds = []
    for c in coords:
        for mu in range(len(L)):
            n = list(c)
            n[mu] = (n[mu] + 1) % L[mu]
            bonds.append((index[c], index[tuple(n)]))
    states = np.arange(2 ** V, dtype=np.int64)
    spins = 1 - 2 * ((states[:, None] >> np.arange(V)[None, :]) & 1)     # (2^V, V) of +-1
    energy = np.zeros(2 ** V)
    for (i, j) in bonds:
        energy += spins[:, i] * spins[:, j]
    mag = spins.sum(axis=1)
    logw = beta * energy + beta * h * mag
    m = logw.max()
    return float((m + np.log(np.sum(np.exp(logw - m)))) / V)


def onsager_lnZ(beta, n=4096):
    """ln Z / V = ln 2 + (1/(8 pi^2)) int int ln[cosh^2 2b - sinh 2b (cos t1 + cos t2)] dt1 dt2.
    Periodic integrand: the rectangle rule on an n x n grid converges geometrically away
    from criticality."""
    t = (np.arange(n) + 0.5) * (2 * np.pi / n)
    c = np.cos(t)
    arg = np.cosh(2 * beta) ** 2 - np.sinh(2 * beta) * (c[:, None] + c[None, :])
    return float(np.log(2.0) + 0.5 * np.mean(np.log(arg)))


def ht_series_lnZ(beta, d):
    """ln Z / V = ln 2 + d ln cosh b + d(d-1)/2 v^4 + d(d-1)(8d-13)/3 v^6
                  + d(d-1)(108 d^2 - 424 d + 425)/4 v^8 + O(v^10),  v = tanh b
    (Fisher-Gaunt general-d hypercubic series; d=2: 1, 2, 9/2; d=3: 3, 22, 187.5)."""
    v = np.tanh(beta)
    return float(np.log(2.0) + d * np.log(np.cosh(beta))
                 + 0.5 * d * (d - 1) * v ** 4
                 + d * (d - 1) * (8 * d - 13) / 3.0 * v ** 6
                 + d * (d - 1) * (108 * d * d - 424 * d + 425) / 4.0 * v ** 8)
