"""Seeded driver for the CPU oracle (TEST INFRASTRUCTURE ONLY).

Connects oracle/tatrg_oracle.py to the shared seeded input generator
(seeded_inputs/) with the sub-seed recipe of SURVEY.md 8(d): per-step Gaussian
sketches for the bond swap and the four isometries, step-independent gauge
references (reading G12).
"""
from __future__ import annotations

import seeded_inputs as si
from oracle import tatrg_oracle as orc

_WHICH = {"swap": si.WHICH_SWAP, "A": si.WHICH_A, "X": si.WHICH_X, "Y": si.WHICH_Y,
          "D": si.WHICH_D, "ref_ad": si.WHICH_REF_AD, "ref_sq1": si.WHICH_REF_SQ[0],
          "ref_sq2": si.WHICH_REF_SQ[1], "ref_sq3": si.WHICH_REF_SQ[2]}


def seeded_inputs_for(seed: int, step: int):
    """inputs(which, rows, cols) for oracle.coarse_grain at step index `step` (0-based).
    Sketches depend on (seed, step, which); gauge references on (seed, which) only."""
    def inputs(which, rows, cols):
        st = 0 if which.startswith("ref") else step
        return si.gauss_matrix(seed, st, _WHICH[which], rows, cols)
    return inputs


def run(beta, h, chi, r, q, n_steps, seed, mode="triad", iso_mode="rsvd",
        active=(1, 1, 1, 1), directions=None, callback=None):
    """init + n_steps coarse-graining steps cycling directions 1->4 (or `directions`)."""
    st = orc.init_ising_tensor(beta, h, active)
    for m in range(n_steps):
        d = directions[m % len(directions)] if directions else (m % 4) + 1
        orc.coarse_grain(st, d, chi, r, q, seeded_inputs_for(seed, m), mode, iso_mode)
        if callback:
            callback(st)
    return st
