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
    """Dense LU of config 2 (n = 30720).  Same arithmetic as oracle.driver.solve / oracle.system (M = I - T A, LAPACK LU),
    written in place so that the 15 GB matrix exists once: A <- -T A (T diagonal: row scaling), diagonal += 1."""
    import scipy.linalg as sla
    from oracle import system
    w = W.config(2)
    t0 = time.time()
    t, type_of, diag = driver.tmatrices(w)
    assert diag
    p = driver.incident_coeffs(w)
    b = system.apply_T(t, type_of, p, diag).reshape(-1)
    M = system.assemble_A(w["lmax"], w["k"], w["pos"], list(w["win_ptr"]))
    M *= -t[type_of].reshape(-1)[:, None]
    M[np.diag_indices_from(M)] += 1.0
    t1 = time.time()
    lu, piv = sla.lu_factor(M, overwrite_a=True, check_finite=False)
    s = sla.lu_solve((lu, piv), b, check_finite=False)
    del lu
    t2 = time.time()
    np.save(os.path.join(HERE, "cfg2_solution.npy"), s.reshape(p.shape))
    # residual with the oracle's matrix-free operator (independent of the factorisation)
    from oracle import matvec as omv
    u = omv.matvec_rows(w["lmax"], w["k"], w["pos"], s.reshape(p.shape))
    r = b - (s - (t[type_of] * u).reshape(-1))
    res = np.linalg.norm(r) / np.linalg.norm(b)
    with open(os.path.join(HERE, "cfg2_solution.txt"), "w") as f:
        f.write("# BASELINE.json config 2 dense LU (oracle only): tests/golden/make_golden.py cfg2\n")
        f.write(f"norm_s={np.linalg.norm(s):.15e}\nlu_rel_residual={res:.3e}\nassemble_seconds={t1 - t0:.1f}\nlu_seconds={t2 - t1:.1f}\n")


if __name__ == "__main__":
    {"cfg1": cfg1, "cfg2": cfg2}[sys.argv[1]]()
