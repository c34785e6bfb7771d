"""Writes the stored expected values under tests/golden/ from oracle/ ONLY (never from the CUDA path).

    python tests/golden/make_golden.py cfg1        # scalars of config 1 (fast)
    python tests/golden/make_golden.py cfg2        # dense LU solution of config 2 (n = 30720: ~15 GB, ~10-20 min)

cfg1_scalars.txt: C_ext, C_sca, ||s||_2 of BASELINE.json config 1 (PAPER.md Eqs. I21-I25 via oracle.driver).
cfg2_solution.npy: scattered coefficients s (1024, 30) complex128 of config 2 by dense LU.
"""
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import driver, fields  # noqa: E402
from paper_2107_09879_b200 import workloads as W  # noqa: E402  (input generator only)


def cfg1():
    w = W.config(1)
    out = driver.solve(w)
    cext, csca = fields.cross_sections(w["lmax"], w["k"], w["pos"], out["s"], out["p"])
    with open(os.path.join(HERE, "cfg1_scalars.txt"), "w") as f:
        f.write("# BASELINE.json config 1, written by tests/golden/make_golden.py cfg1 (oracle only)\n")
        f.write(f"C_ext={cext:.15e}\nC_sca={csca:.15e}\nnorm_s={np.linalg.norm(out['s']):.15e}\n")


def cfg2():
    w = W.config(2)
    t0 = time.time()
    out = driver.solve(w)
    np.save(os.path.join(HERE, "cfg2_solution.npy"), out["s"])
    M = out["M"]
    t, type_of, diag = driver.tmatrices(w)
    b = (t[type_of] * out["p"]).reshape(-1)
    res = np.linalg.norm(M @ out["s"].reshape(-1) - b) / np.linalg.norm(b)
    with open(os.path.join(HERE, "cfg2_solution.txt"), "w") as f:
        f.write("# BASELINE.json config 2 dense LU (oracle only): tests/golden/make_golden.py cfg2\n")
        f.write(f"norm_s={np.linalg.norm(out['s']):.15e}\nlu_rel_residual={res:.3e}\nseconds={time.time() - t0:.1f}\n")


if __name__ == "__main__":
    {"cfg1": cfg1, "cfg2": cfg2}[sys.argv[1]]()
