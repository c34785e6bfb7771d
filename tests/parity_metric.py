"""The error metric of the GPU parity tests (tests/test_gpu_*.py).

`rel(a, b)` returns the LARGER of
  * the relative L2 error  ||a - b||_2 / ||b||_2  (the metric north_star states for the solve), and
  * the worst block-wise maximum error  max_block ( max|a - b| / max|b| ):
      - coefficient arrays [..., L] (L = 2 lmax (lmax + 2), flat order R1): one block per (l, p), all m and all scatterers -
        |T_{l=3}| is ~1e-3 of |T_{l=1}|, so an L2 bound alone leaves the high-l entries of a solution checked to ~1e-6 only;
      - field arrays [n_pts, 3]: one block per detector point (far points carry little of the L2 norm),
so every `assert rel(...) <= tol` in the tests bounds both.  Arrays of any other shape are compared by L2 only.

`rel_solve(a, b)` is the metric for CONVERGED GMRES SOLUTIONS: the larger of the L2 error and the global max-norm error
max|a - b| / max|b|.  A norm-wise stopping rule (||b - M x||_2 <= tol ||b||_2, reading R13) bounds the error of a block only
in absolute terms: the part of b in the l = 6 block is ~1e-8 of ||b|| for Mie spheres, so GMRES has met a 1e-11 tolerance
once that block is reduced by 1e-3 - its RELATIVE error (7e-8 measured in test_lmax6_solve_small, absolute 7e-15) is a
property of the stopping rule, not of a kernel.  The per-block relative figure of every solve is still logged (third column).
With TM_PARITY_LOG=<file> every call appends "caller<TAB>l2<TAB>block" (used to record the achieved numbers).
"""
import inspect
import os

import numpy as np

_L_OF = {2 * l * (l + 2): l for l in range(1, 9)}


def l2(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(b))


def block_err(a, b):
    """Worst per-(l, p)-block (coefficients) or per-point (fields) max error relative to the block's max |b|; None if the
    shape carries no block structure."""
    a, b = np.asarray(a), np.asarray(b)
    if a.shape != b.shape or a.ndim < 2:
        return None
    last = a.shape[-1]
    if last in _L_OF:
        lmax = _L_OF[last]
        half = last // 2
        worst = 0.0
        for p in (0, 1):
            for l in range(1, lmax + 1):
                sl = slice(p * half + l * l - 1, p * half + l * l + 2 * l)          # m = -l..l of (l, p)
                scale = np.abs(b[..., sl]).max()
                if scale > 0:
                    worst = max(worst, float(np.abs(a[..., sl] - b[..., sl]).max() / scale))
        return worst
    if last == 3 and a.ndim == 2:
        scale = np.abs(b).max(axis=1)
        ok = scale > 0
        return float((np.abs(a - b).max(axis=1)[ok] / scale[ok]).max()) if ok.any() else 0.0
    return None


def rel(a, b):
    e2 = l2(a, b)
    eb = block_err(a, b)
    log = os.environ.get("TM_PARITY_LOG")
    if log:
        fr = inspect.stack()[1]
        with open(log, "a") as f:
            f.write(f"{os.path.basename(fr.filename)}:{fr.lineno}:{fr.function}\t{e2:.3e}\t{'-' if eb is None else format(eb, '.3e')}\n")
    return e2 if eb is None else max(e2, eb)


def rel_solve(a, b):
    a, b = np.asarray(a), np.asarray(b)
    e2 = l2(a, b)
    emax = float(np.abs(a - b).max() / np.abs(b).max())
    log = os.environ.get("TM_PARITY_LOG")
    if log:
        fr = inspect.stack()[1]
        eb = block_err(a, b)
        with open(log, "a") as f:
            f.write(f"{os.path.basename(fr.filename)}:{fr.lineno}:{fr.function}\t{e2:.3e}\t{'-' if eb is None else format(eb, '.3e')}\tsolve: max-norm {emax:.3e}\n")
    return max(e2, emax)
