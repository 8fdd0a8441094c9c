"""How far does the ORACLE move when its own inputs move by one unit in the last place?

Reading G13 compares the spectra of the CUDA path with the oracle's at 1e-9 of the largest
value.  Two correct FP64 implementations of the same step differ by rounding, and 40 coarse-graining
steps near criticality amplify that; this script measures the amplification on the oracle alone, so that
the tolerances of the parity tests rest on the method's conditioning, not on what the CUDA path happens
to reach.  It runs a config twice with the same seeds: once as it stands, once with every Gaussian
sketch element (bond swap and the four isometries) multiplied by (1 + u 2^-52), i.e. moved by u ulps
(u = 1 by default; u = 64 stands for the backward error of a different but backward-stable factorisation of
a 10^3..10^5-row block, which is tens of ulps), and records, per step and per spectrum,
max_i |s_i - s_i'| / s_1 and the relative change of ln Z/V.

Imports ONLY oracle/ and seeded_inputs/.  Writes tests/golden/oracle_sensitivity_<name>.json.

    python tests/golden/oracle_sensitivity.py c2 [ulps]
"""
from __future__ import annotations

import json
import os
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

RUNS = {
    "c1": dict(T=6.0, h=0.0, chi=6, r=2, q=2, seed=20241214, steps=8),
    "c2": dict(T=6.65, h=0.0, chi=16, r=2, q=2, seed=20241215, steps=40),
    # the first steps of the wide-route golden (tests/golden/oracle_w80.json): legs 2 -> 4 -> 16 -> 40, where the
    # pair operator K K_w^T still has exact rank deficiencies (no truncation has happened on those legs yet)
    "w80": dict(T=6.5, h=0.01, chi=40, r=2, q=3, seed=20241218, steps=4),
}
SPECTRA = ("sigmaT", "sigma_swap", "SA", "SX", "SY", "SD", "s1", "s2", "s3")
ULP = 2.0 ** -52


def main(name, ulps=1):
    from oracle import driver
    from oracle import tatrg_oracle as orc
    cfg = RUNS[name]
    beta = 1.0 / cfg["T"]
    a = orc.init_ising_tensor(beta, cfg["h"])
    b = orc.init_ising_tensor(beta, cfg["h"])
    out = {"name": name, "config": cfg, "perturbation": "every element of the five Gaussian sketches x (1 + %d * 2^-52)" % ulps,
           "steps": []}
    worst = {}
    for m in range(cfg["steps"]):
        d = m % 4 + 1
        base = driver.seeded_inputs_for(cfg["seed"], m)

        def moved(which, rows, cols, base=base):
            g = base(which, rows, cols)
            return g if which.startswith("ref") else g * (1.0 + ulps * ULP)
        ra = orc.coarse_grain(a, d, cfg["chi"], cfg["r"], cfg["q"], base)
        rb = orc.coarse_grain(b, d, cfg["chi"], cfg["r"], cfg["q"], moved)
        la, lb = orc.log_Z_per_site(a), orc.log_Z_per_site(b)
        rec = {"step": m, "lnz_rel": abs(lb / la - 1)}
        for k in SPECTRA:
            if k in ra and len(ra[k]):
                sa, sb = np.asarray(ra[k]), np.asarray(rb[k])
                rec[k] = float(np.abs(sa - sb).max() / sa[0]) if len(sa) == len(sb) else float("inf")
        for k, v in rec.items():
            if k != "step":
                worst[k] = max(worst.get(k, 0.0), v)
        out["steps"].append(rec)
        print(" ".join("%s %.1e" % (k, v) if k != "step" else "step %d" % (v + 1) for k, v in rec.items()), flush=True)
    out["worst"] = worst
    path = os.path.join(HERE, "oracle_sensitivity_%s%s.json" % (name, "" if ulps == 1 else "_%dulp" % ulps))
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
        f.write("\n")
    print("worst", {k: "%.2e" % v for k, v in worst.items()})
    print("wrote", path)


if __name__ == "__main__":
    main(sys.argv[1] if len(sys.argv) > 1 else "c2", int(sys.argv[2]) if len(sys.argv) > 2 else 1)
