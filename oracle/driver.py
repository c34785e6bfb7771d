"""Run the oracle on a workload dict (TEST INFRASTRUCTURE ONLY - see oracle/__init__.py).

Glue only: picks the T-matrices (oracle.tmatrix), incident coefficients (oracle.incident) and the
dense solve (oracle.system) for a workload produced by paper_2107_09879_b200.workloads (which is
passed in as a plain dict - this package does not import the product)."""
import numpy as np

from . import incident, system, tmatrix
from .modes import n_modes


def tmatrices(w):
    """-> (t, type_of, diag)."""
    if w["t_kind"] in ("mie_types", "mie_sites"):
        t = np.stack([tmatrix.mie_tmatrix_diag(w["lmax"], w["k"], r, w["eps_r"]) for r in w["radii"]])
        return t, np.asarray(w["type_of"]), True
    return np.asarray(w["t_full"]), np.asarray(w["type_of"]), False


def incident_coeffs(w):
    pos = w["pos"]
    if w["inc_kind"] == "plane":
        return incident.plane_wave_incident(w["lmax"], w["k"], pos, w["beta"], w["alpha"], w["A_beta"], w["A_alpha"])
    out = np.zeros((pos.shape[0], n_modes(w["lmax"])), dtype=complex)
    wp = w["win_ptr"]
    for iw in range(len(wp) - 1):
        sl = slice(wp[iw], wp[iw + 1])
        out[sl] = incident.gaussian_beam_incident(w["lmax"], w["k"], pos[sl], w["focus"][iw], w["w0"], w["Ax"], w["Ay"])
    return out


def solve(w, p_inc=None, adjoint_w=None):
    """Dense LU solve of the workload: returns dict(s=..., lam=... if adjoint_w given, M=...)."""
    t, type_of, diag = tmatrices(w)
    if p_inc is None:
        p_inc = incident_coeffs(w)
    M = system.assemble_M(w["lmax"], w["k"], w["pos"], t, type_of, diag, list(w["win_ptr"]))
    out = dict(M=M, p=p_inc, s=system.solve_forward(M, t, type_of, diag, p_inc))
    if adjoint_w is not None:
        out["lam"] = system.solve_adjoint(M, adjoint_w)
    return out
