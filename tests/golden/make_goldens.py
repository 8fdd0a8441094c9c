"""Writes the stored oracle results under tests/golden/ that the GPU parity tests compare against.

Imports ONLY `oracle/` and `seeded_inputs/` (the shared seeded input generator): no value in the
files it writes ever comes from the CUDA path.  Run on a CPU box:

    python tests/golden/make_goldens.py c3 c4 w80 [--threads N]

Each golden is one JSON text file `oracle_<name>.json` holding, for every step of the run, the
quantities the north star compares (BASELINE.json): ln Z/V after the step and the nine spectra of
the step (sigma^T of the canonical form, sigma of the bond swap, the isometry spectra S^A, S^X, S^Y,
S^D, the squeezer spectra s^(t1..t3)), plus dims, ln c_m, the order parameter X^(m)
 and the relative gaps at the truncation cuts (reading G12).  Floats are written
with `repr` (round-trip exact).

Runs (all cycling directions 1..4, seeds of bench.py:CONFIGS):
  c3   BASELINE.json configs[2], T=6.65 h=0 chi=32 r=2 q=2, steps 1..12: eight steady-state steps
       (all legs = chi on input from step 5 on) -- the launch configuration bench.py times.
  c4   BASELINE.json configs[3], plain ATRG (Table 1) chi=24 r=2 q=2, steps 1..6:
       two steps through the O(chi^9) product at its full size (13824 x 13824 x 576 per slice).
  w80  the parameters of BASELINE.json configs[4] (T=6.5, h=0.01, r=2, q=3) at chi=40, steps 1..6:
       internal lines r*chi = 80 > 64, i.e. the routes of the CUDA path that are wider than 64
       columns (128-column Cholesky-QR panels, multi-launch Jacobi core, sequential isometry route);
       chi=64 itself is out of the oracle's reach (about 80 GB and 4.6e14 flop per step).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

RUNS = {
    "c3": dict(T=6.65, h=0.0, chi=32, r=2, q=2, seed=20241216, mode="triad", steps=12),
    "c4": dict(T=6.65, h=0.0, chi=24, r=2, q=2, seed=20241217, mode="atrg", steps=6),
    "w80": dict(T=6.5, h=0.01, chi=40, r=2, q=3, seed=20241218, mode="triad", steps=6),
}
SPECTRA = ("sigmaT", "sigma_swap", "SA", "SX", "SY", "SD", "s1", "s2", "s3")


def make(name: str) -> str:
    from oracle import driver
    from oracle import tatrg_oracle as orc
    cfg = RUNS[name]
    beta = 1.0 / cfg["T"]
    st = orc.init_ising_tensor(beta, cfg["h"])
    out = {"name": name, "config": cfg, "lnz_init": repr(float(orc.log_Z_per_site(st))), "steps": []}
    path = os.path.join(HERE, "oracle_%s.json" % name)
    for m in range(cfg["steps"]):
        d = m % 4 + 1
        t0 = time.time()
        rec = orc.coarse_grain(st, d, cfg["chi"], cfg["r"], cfg["q"], driver.seeded_inputs_for(cfg["seed"], m),
                               mode=cfg["mode"])
        dt = time.time() - t0
        step = {"step": m, "direction": d, "dims_in": list(rec["dims_in"]), "dims_out": list(rec["dims_out"]),
                "lnz": repr(float(orc.log_Z_per_site(st))), "ln_c": repr(float(rec["ln_c"])),
                "order_parameter": repr(float(orc.order_parameter_X(st))),
                "gaps": {k: repr(float(rec[k])) for k in ("gap_swap", "gap_s1", "gap_s2", "gap_s3")},
                "spectra": {k: [repr(float(v)) for v in rec[k]] for k in SPECTRA if k in rec},
                "oracle_seconds": round(dt, 1)}
        out["steps"].append(step)
        print("%s step %d dir %d dims %s -> %s  lnZ/V %s  (%.1f s)" %
              (name, m + 1, d, rec["dims_in"], rec["dims_out"], step["lnz"], dt), flush=True)
        with open(path, "w") as f:          # rewritten after every step: a cut-off run keeps what it has
            json.dump(out, f, indent=1)
            f.write("\n")
    return path


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("names", nargs="+", choices=sorted(RUNS))
    ap.add_argument("--threads", type=int, default=0, help="BLAS threads (0 = library default)")
    args = ap.parse_args()
    if args.threads:
        for v in ("OMP_NUM_THREADS", "OPENBLAS_NUM_THREADS", "MKL_NUM_THREADS"):
            os.environ[v] = str(args.threads)
    for n in args.names:
        print("wrote", make(n), flush=True)


if __name__ == "__main__":
    main()
