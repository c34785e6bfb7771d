"""Thin ctypes binding over libtm.so (include/tm.h): argument marshalling only.

Every step of the path runs in the CUDA library; this module never computes.  It fails loudly when the
library is missing (there is no CPU fallback).  PyTorch is used only to allocate device memory / hand over
the current CUDA stream (``Solver(..., use_torch=True)``); numpy arrays are passed as host pointers.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "lib", "libtm.so")

TM_FP64, TM_FP32, TM_MIXED = 0, 1, 2
TM_PEAK_FP64_TENSOR = 3
TM_OK, TM_NOT_CONVERGED = 0, 1
TM_E_INVALID, TM_E_OVERLAP, TM_E_STATE, TM_E_CUDA, TM_E_NOMEM = -1, -2, -3, -4, -5
TM_INC_PLANE, TM_INC_GAUSS, TM_INC_COEFFS, TM_INC_JINC = 0, 1, 2, 3
TM_FIELD_E_SCA, TM_FIELD_H_SCA, TM_FIELD_E_INC = 0, 1, 2
TM_KERNEL_AUTO, TM_KERNEL_GENERAL, TM_KERNEL_COPLANAR, TM_KERNEL_SYM3D, TM_KERNEL_ROT3D = 0, 1, 2, 3, 4

EXPORTS = ["tm_create", "tm_set_tmatrices", "tm_set_incident", "tm_get_incident", "tm_solve", "tm_solve_adjoint",
           "tm_matvec", "tm_solve_multi", "tm_fields", "tm_workspace_bytes", "tm_set_workspace", "tm_set_kernel", "tm_get_kernel",
           "tm_kernel_time", "tm_pair_cost", "tm_measure_fma_peak", "tm_grad_tmatrix", "tm_grad_positions", "tm_mie_tmatrix_dR", "tm_mie_tmatrix",
           "tm_nullfield_tmatrix", "tm_nullfield_dtmatrix", "tm_ttable_interp",
           "tm_fields_static_setup", "tm_fields_static", "tm_fields_static_error",
           "tm_release_cached_memory", "tm_debug_guards", "tm_num_modes", "tm_last_error", "tm_destroy"]


class c64(ctypes.Structure):
    _fields_ = [("re", ctypes.c_double), ("im", ctypes.c_double)]


class PlaneDesc(ctypes.Structure):
    _fields_ = [("beta", ctypes.c_double), ("alpha", ctypes.c_double), ("A_beta", c64), ("A_alpha", c64)]


class GaussDesc(ctypes.Structure):
    _fields_ = [("focus", ctypes.c_void_p), ("w0", ctypes.c_double), ("Ax", c64), ("Ay", c64), ("n_beta", ctypes.c_int)]


class JincDesc(ctypes.Structure):
    _fields_ = [("n_src", ctypes.c_int), ("src_xyz", ctypes.c_void_p), ("amp", ctypes.c_void_p), ("src_ptr", ctypes.c_void_p),
                ("n_beta", ctypes.c_int), ("amp_is_sample", ctypes.c_int)]


class CoeffsDesc(ctypes.Structure):
    _fields_ = [("p", ctypes.c_void_p)]


class SolveOpts(ctypes.Structure):
    _fields_ = [("tol", ctypes.c_double), ("restart", ctypes.c_int), ("max_iter", ctypes.c_int), ("warm_start", ctypes.c_int)]


class SolveInfo(ctypes.Structure):
    _fields_ = [("iterations", ctypes.c_int), ("restarts", ctypes.c_int), ("converged", ctypes.c_int),
                ("matvecs", ctypes.c_int), ("rel_residual", ctypes.c_double), ("seconds", ctypes.c_double)]


class TmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libtm error {code}: {msg}")
        self.code = code


_lib = None


def lib():
    """Load libtm.so (hard error when it has not been built: run __graft_entry__.build())."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise ImportError(f"{_SO} not found: build it with `python -m paper_2107_09879_b200.build` "
                              "(the CUDA library is required; there is no CPU fallback)")
        L = ctypes.CDLL(_SO)
        vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        L.tm_create.argtypes = [ctypes.POINTER(vp), ci, vp, ci, vp, ci, cd, ci, vp]
        L.tm_set_tmatrices.argtypes = [vp, ci, ci, vp, vp, vp]
        L.tm_set_incident.argtypes = [vp, ci, vp]
        L.tm_get_incident.argtypes = [vp, vp]
        L.tm_solve.argtypes = [vp, ctypes.POINTER(SolveOpts), vp, vp]
        L.tm_solve_adjoint.argtypes = [vp, vp, ctypes.POINTER(SolveOpts), vp, vp]
        L.tm_matvec.argtypes = [vp, ci, vp, vp]
        L.tm_solve_multi.argtypes = [vp, ci, ci, vp, ctypes.POINTER(SolveOpts), vp, vp]
        L.tm_fields.argtypes = [vp, ci, vp, vp, ci, vp]
        L.tm_workspace_bytes.argtypes = [vp, ctypes.POINTER(SolveOpts)]
        L.tm_workspace_bytes.restype = ctypes.c_size_t
        L.tm_set_workspace.argtypes = [vp, vp, ctypes.c_size_t]
        L.tm_set_kernel.argtypes = [vp, ci]
        L.tm_get_kernel.argtypes = [vp]
        L.tm_kernel_time.argtypes = [vp, ci, ctypes.POINTER(cd), ctypes.POINTER(ctypes.c_longlong), ctypes.POINTER(ctypes.c_longlong)]
        L.tm_mie_tmatrix.argtypes = [ci, cd, cd, c64, vp]
        L.tm_grad_tmatrix.argtypes = [vp, vp, vp, vp, vp]
        L.tm_grad_positions.argtypes = [vp, vp, vp, vp, vp]
        L.tm_mie_tmatrix_dR.argtypes = [ci, cd, cd, c64, vp]
        L.tm_nullfield_tmatrix.argtypes = [ci, ci, cd, c64, ci, ci, vp, vp, vp, vp, vp, vp]
        L.tm_nullfield_dtmatrix.argtypes = [ci, ci, cd, c64, ci, ci, vp, vp, vp, vp, cd, vp, vp]
        L.tm_pair_cost.argtypes = [vp, ctypes.POINTER(cd), ctypes.POINTER(cd)]
        L.tm_measure_fma_peak.argtypes = [ci, ctypes.POINTER(cd), vp]
        L.tm_num_modes.argtypes = [ci]
        L.tm_last_error.argtypes = [vp]
        L.tm_last_error.restype = ctypes.c_char_p
        L.tm_destroy.argtypes = [vp]
        L.tm_destroy.restype = None
        L.tm_fields_static_setup.argtypes = []
        L.tm_fields_static.argtypes = [ci, cd, ci, vp, vp, ci, vp, ci, vp, vp]
        L.tm_fields_static_error.argtypes = []
        L.tm_fields_static_error.restype = ctypes.c_char_p
        L.tm_ttable_interp.argtypes = [ci, vp, ctypes.c_longlong, vp, ci, vp, vp, vp, vp]
        L.tm_debug_guards.argtypes = [ci, ctypes.POINTER(ctypes.c_longlong)]
        L.tm_debug_guards.restype = ctypes.c_longlong
        _lib = L
    return _lib


def _ptr(a):
    """Host numpy array or torch tensor (host or CUDA) -> raw pointer; None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags["C_CONTIGUOUS"]
        return a.ctypes.data
    return a.data_ptr()      # torch tensor


def _c64(z):
    z = complex(z)
    return c64(z.real, z.imag)


def mie_tmatrix(lmax, k_b, radius, eps_r):
    """Diagonal Mie T-matrix (tm_mie_tmatrix), shape (L,) complex128."""
    out = np.zeros(lib().tm_num_modes(lmax), dtype=np.complex128)
    rc = lib().tm_mie_tmatrix(lmax, float(k_b), float(radius), _c64(eps_r), out.ctypes.data)
    if rc != TM_OK:
        raise TmError(rc, "tm_mie_tmatrix: invalid arguments")
    return out


def mie_tmatrix_dR(lmax, k_b, radius, eps_r):
    """d(diag Mie T)/dR (tm_mie_tmatrix_dR), shape (L,) complex128."""
    out = np.zeros(lib().tm_num_modes(lmax), dtype=np.complex128)
    rc = lib().tm_mie_tmatrix_dR(lmax, float(k_b), float(radius), _c64(eps_r), out.ctypes.data)
    if rc != TM_OK:
        raise TmError(rc, "tm_mie_tmatrix_dR: invalid arguments")
    return out


def nullfield_tmatrix(lmax, k_b, eps_r, generatrices, stream=None, lmax_internal=0):
    """Null-field T-matrices of bodies of revolution (tm_nullfield_tmatrix).  `generatrices`: one (theta, r, dr, w) tuple
    or a list of them with equal node counts (workloads.generatrix_*).  Returns (L, L) or (n_shapes, L, L) complex128."""
    single = not isinstance(generatrices, list)
    gens = [generatrices] if single else generatrices
    arr = [np.ascontiguousarray(np.stack([np.asarray(g[i], dtype=np.float64) for g in gens])) for i in range(4)]
    n_shapes, n_nodes = arr[0].shape
    L = lib().tm_num_modes(lmax)
    out = np.zeros((n_shapes, L, L), dtype=np.complex128)
    rc = lib().tm_nullfield_tmatrix(int(lmax), int(lmax_internal), float(k_b), _c64(eps_r), n_shapes, n_nodes, arr[0].ctypes.data, arr[1].ctypes.data,
                                    arr[2].ctypes.data, arr[3].ctypes.data, out.ctypes.data,
                                    ctypes.c_void_p(stream) if stream else None)
    if rc != TM_OK:
        raise TmError(rc, "tm_nullfield_tmatrix failed")
    return out[0] if single else out


def nullfield_dtmatrix(lmax, k_b, eps_r, generatrix_fn, params, h, stream=None, lmax_internal=0):
    """dT/dp of null-field T-matrices (tm_nullfield_dtmatrix).  generatrix_fn(p) -> (theta, r, dr, w) for parameter value p;
    params: the parameter value of every shape.  Returns (n_shapes, L, L) complex128."""
    gens = [generatrix_fn(p + d) for p in params for d in (h, -h, 0.5 * h, -0.5 * h)]
    arr = [np.ascontiguousarray(np.stack([np.asarray(g[i], dtype=np.float64) for g in gens])) for i in range(4)]
    n_nodes = arr[0].shape[1]
    L = lib().tm_num_modes(lmax)
    out = np.zeros((len(params), L, L), dtype=np.complex128)
    rc = lib().tm_nullfield_dtmatrix(int(lmax), int(lmax_internal), float(k_b), _c64(eps_r), len(params), n_nodes, arr[0].ctypes.data, arr[1].ctypes.data,
                                     arr[2].ctypes.data, arr[3].ctypes.data, float(h), out.ctypes.data,
                                     ctypes.c_void_p(stream) if stream else None)
    if rc != TM_OK:
        raise TmError(rc, "tm_nullfield_dtmatrix failed")
    return out


def ttable_interp(p_tab, T_tab, p, deriv=True, out=None, dout=None, stream=None):
    """tm_ttable_interp: T_tab (n_tab, ...) at the nodes p_tab -> (T (n_out, ...), dT/dp (n_out, ...) or None) at the values p.
    numpy arrays or torch CUDA tensors (outputs are made where `p` lives)."""
    on_dev = not isinstance(p, np.ndarray)
    if isinstance(p_tab, np.ndarray):
        p_tab = np.ascontiguousarray(p_tab, dtype=np.float64)
    if isinstance(T_tab, np.ndarray):
        T_tab = np.ascontiguousarray(T_tab, dtype=np.complex128)
    if not on_dev:
        p = np.ascontiguousarray(p, dtype=np.float64)
    n_tab, n_out = int(T_tab.shape[0]), int(p.shape[0])
    shape = (n_out,) + tuple(T_tab.shape[1:])
    n_entry = 1
    for d in T_tab.shape[1:]:
        n_entry *= int(d)

    def make():
        if on_dev:
            import torch
            return torch.empty(shape, dtype=torch.complex128, device=p.device)
        return np.empty(shape, dtype=np.complex128)
    out = make() if out is None else out
    if deriv and dout is None:
        dout = make()
    rc = lib().tm_ttable_interp(n_tab, _ptr(p_tab), n_entry, _ptr(T_tab), n_out, _ptr(p), _ptr(out), _ptr(dout) if deriv else None,
                                ctypes.c_void_p(stream) if stream else None)
    if rc != TM_OK:
        raise TmError(rc, "tm_ttable_interp failed (TM_E_INVALID: a parameter outside the table, fewer than 4 nodes, nodes not increasing)")
    return out, (dout if deriv else None)


def measure_fma_peak(precision=TM_FP64, stream=None):
    """Measured register-resident FMA peak of the device in TFLOP/s (tm_measure_fma_peak)."""
    v = ctypes.c_double()
    rc = lib().tm_measure_fma_peak(int(precision), ctypes.byref(v), ctypes.c_void_p(stream) if stream else None)
    if rc != TM_OK:
        raise TmError(rc, "tm_measure_fma_peak failed (no CUDA device?)")
    return v.value


def fields_static_setup():
    """Resolve the static scratch array of tm_fields_static on the current device (once per device; e.g. before a graph capture)."""
    rc = lib().tm_fields_static_setup()
    if rc != TM_OK:
        raise TmError(rc, lib().tm_fields_static_error().decode())


def fields_static(lmax, k_b, pos, s, pts, which=TM_FIELD_E_SCA, out=None, stream=None):
    """tm_fields_static: scattered E (or Z_b H) at pts from coefficients s, allocation-free in the library.  pos (N,3) float64,
    s (N,L) complex128, pts (M,3) float64: torch CUDA tensors; out (M,3) complex128 CUDA tensor (created here when None - pass
    one in where the caller must not allocate either).  Enqueued on `stream` (raw cudaStream_t, default stream when None)
    WITHOUT synchronising.  Raises TmError for M > 65536 and other invalid arguments."""
    import torch
    if out is None:
        out = torch.empty((int(pts.shape[0]), 3), dtype=torch.complex128, device=pts.device)
    rc = lib().tm_fields_static(int(lmax), float(k_b), int(pos.shape[0]), _ptr(pos), _ptr(s), int(pts.shape[0]), _ptr(pts), int(which),
                                _ptr(out), ctypes.c_void_p(stream) if stream else None)
    if rc != TM_OK:
        raise TmError(rc, lib().tm_fields_static_error().decode())
    return out


def debug_guards(enable=-1):
    """tm_debug_guards: switch the sentinel margins of the library's internal device buffers on (1) / off (0) or query (-1);
    returns (damaged margins found so far, guarded blocks handed out)."""
    nb = ctypes.c_longlong()
    bad = lib().tm_debug_guards(int(enable), ctypes.byref(nb))
    if bad < 0:
        raise TmError(int(bad), "tm_debug_guards failed")
    return int(bad), int(nb.value)


def release_cached_memory():
    """Hand the library's cached, unused device memory back to the driver (tm_release_cached_memory)."""
    rc = lib().tm_release_cached_memory()
    if rc != TM_OK:
        raise TmError(rc, "tm_release_cached_memory failed")


class Solver:
    """One tm_ctx.  Arrays may be numpy (host) or torch CUDA tensors (device); complex data is complex128
    [n_scat, L] (torch.complex128 on the device)."""

    def __init__(self, pos, lmax, k_b, win_ptr=None, precision=TM_FP64, stream=None):
        self._h = ctypes.c_void_p()
        L = lib()
        self.pos = np.ascontiguousarray(pos, dtype=np.float64) if isinstance(pos, np.ndarray) else pos
        self.n_scat = int(self.pos.shape[0])
        self.lmax = int(lmax)
        self.L = L.tm_num_modes(self.lmax)
        wp = None
        self.n_win = 1
        if win_ptr is not None:
            wp = np.ascontiguousarray(win_ptr, dtype=np.int32)
            self.n_win = wp.size - 1
        rc = L.tm_create(ctypes.byref(self._h), self.n_scat, _ptr(self.pos), self.n_win, _ptr(wp), self.lmax, float(k_b),
                         int(precision), ctypes.c_void_p(stream) if stream else None)
        if rc != TM_OK:
            msg = L.tm_last_error(None).decode()
            self._h = ctypes.c_void_p()
            raise TmError(rc, msg)
        self._keep = []          # buffers the library keeps using (workspace)

    def _check(self, rc):
        if rc < 0:
            raise TmError(rc, lib().tm_last_error(self._h).decode())
        return rc

    def close(self):
        if self._h:
            lib().tm_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- setup
    def set_tmatrices(self, T, type_of, diag_only, r_enclosing=None):
        T = np.ascontiguousarray(T, dtype=np.complex128) if isinstance(T, np.ndarray) else T
        ty = np.ascontiguousarray(type_of, dtype=np.int32) if isinstance(type_of, np.ndarray) else type_of
        re = None if r_enclosing is None else np.ascontiguousarray(r_enclosing, dtype=np.float64)
        return self._check(lib().tm_set_tmatrices(self._h, int(T.shape[0]), 1 if diag_only else 0, _ptr(T), _ptr(ty), _ptr(re)))

    def set_incident_plane(self, beta, alpha, A_beta, A_alpha):
        d = PlaneDesc(float(beta), float(alpha), _c64(A_beta), _c64(A_alpha))
        return self._check(lib().tm_set_incident(self._h, TM_INC_PLANE, ctypes.addressof(d)))

    def set_incident_gauss(self, focus, w0, Ax, Ay, n_beta=0):
        f = np.ascontiguousarray(focus, dtype=np.float64).reshape(self.n_win, 3)
        d = GaussDesc(f.ctypes.data, float(w0), _c64(Ax), _c64(Ay), int(n_beta))
        return self._check(lib().tm_set_incident(self._h, TM_INC_GAUSS, ctypes.addressof(d)))

    def set_incident_jinc(self, src, amp, src_ptr=None, n_beta=0, samples=False):
        """Jinc sources (PAPER.md Eqs. II1-II17): src (S,3), amp (S,2) complex transverse amplitudes - or, with samples=True,
        the field samples on the lambda/2 grid (the library applies the Nyquist factor of reading R17) -, src_ptr (n_win+1,)."""
        src = np.ascontiguousarray(src, dtype=np.float64).reshape(-1, 3)
        amp = np.ascontiguousarray(amp, dtype=np.complex128).reshape(-1, 2)
        ptr = np.array([0, src.shape[0]], dtype=np.int32) if src_ptr is None else np.ascontiguousarray(src_ptr, dtype=np.int32)
        d = JincDesc(int(src.shape[0]), src.ctypes.data, amp.ctypes.data, ptr.ctypes.data, int(n_beta), 1 if samples else 0)
        return self._check(lib().tm_set_incident(self._h, TM_INC_JINC, ctypes.addressof(d)))

    def set_incident_coeffs(self, p):
        p = np.ascontiguousarray(p, dtype=np.complex128) if isinstance(p, np.ndarray) else p
        d = CoeffsDesc(_ptr(p))
        return self._check(lib().tm_set_incident(self._h, TM_INC_COEFFS, ctypes.addressof(d)))

    def get_incident(self, out=None):
        out = np.empty((self.n_scat, self.L), dtype=np.complex128) if out is None else out
        self._check(lib().tm_get_incident(self._h, _ptr(out)))
        return out

    def set_kernel(self, kernel):
        return self._check(lib().tm_set_kernel(self._h, int(kernel)))

    def get_kernel(self):
        return lib().tm_get_kernel(self._h)

    def workspace_bytes(self, restart):
        o = SolveOpts(1e-6, int(restart), 1, 0)
        return int(lib().tm_workspace_bytes(self._h, ctypes.byref(o)))

    def set_workspace(self, tensor):
        """tensor: torch CUDA uint8 tensor (kept alive by this object) or None."""
        self._keep = [tensor]
        if tensor is None:
            return self._check(lib().tm_set_workspace(self._h, None, 0))
        return self._check(lib().tm_set_workspace(self._h, tensor.data_ptr(), tensor.numel() * tensor.element_size()))

    # ---- compute
    def matvec(self, x, transpose=0, out=None):
        x = np.ascontiguousarray(x, dtype=np.complex128) if isinstance(x, np.ndarray) else x
        out = self._like(x) if out is None else out
        self._check(lib().tm_matvec(self._h, int(transpose), _ptr(x), _ptr(out)))
        return out

    def _like(self, x):
        if isinstance(x, np.ndarray):
            return np.empty((self.n_scat, self.L), dtype=np.complex128)
        import torch
        return torch.empty((self.n_scat, self.L), dtype=torch.complex128, device=x.device)

    def solve(self, tol, restart, max_iter, out=None, warm_start=False):
        """warm_start: `out` holds the initial guess on entry (tm_solve_opts.warm_start)."""
        if warm_start and out is None:
            raise ValueError("warm_start needs the initial guess in `out`")
        out = np.empty((self.n_scat, self.L), dtype=np.complex128) if out is None else out
        o = SolveOpts(float(tol), int(restart), int(max_iter), 1 if warm_start else 0)
        info = (SolveInfo * self.n_win)()
        rc = self._check(lib().tm_solve(self._h, ctypes.byref(o), _ptr(out), ctypes.addressof(info)))
        return out, list(info), rc

    def solve_adjoint(self, w, tol, restart, max_iter, out=None, warm_start=False):
        w = np.ascontiguousarray(w, dtype=np.complex128) if isinstance(w, np.ndarray) else w
        if warm_start and out is None:
            raise ValueError("warm_start needs the initial guess in `out`")
        out = self._like(w) if out is None else out
        o = SolveOpts(float(tol), int(restart), int(max_iter), 1 if warm_start else 0)
        info = (SolveInfo * self.n_win)()
        rc = self._check(lib().tm_solve_adjoint(self._h, _ptr(w), ctypes.byref(o), _ptr(out), ctypes.addressof(info)))
        return out, list(info), rc

    def solve_multi(self, rhs, tol, restart, max_iter, adjoint=False, out=None):
        """tm_solve_multi: rhs (n_rhs, n_scat, L) incident coefficients (or adjoint weights) -> (out (n_rhs, n_scat, L),
        info[n_rhs][n_win], rc)."""
        rhs = np.ascontiguousarray(rhs, dtype=np.complex128) if isinstance(rhs, np.ndarray) else rhs
        n_rhs = int(rhs.shape[0])
        if out is None:
            if isinstance(rhs, np.ndarray):
                out = np.empty((n_rhs, self.n_scat, self.L), dtype=np.complex128)
            else:
                import torch
                out = torch.empty((n_rhs, self.n_scat, self.L), dtype=torch.complex128, device=rhs.device)
        o = SolveOpts(float(tol), int(restart), int(max_iter), 0)
        info = (SolveInfo * (self.n_win * n_rhs))()
        rc = self._check(lib().tm_solve_multi(self._h, 1 if adjoint else 0, n_rhs, _ptr(rhs), ctypes.byref(o), _ptr(out),
                                              ctypes.addressof(info)))
        flat = list(info)
        return out, [flat[r * self.n_win:(r + 1) * self.n_win] for r in range(n_rhs)], rc

    def fields(self, pts, s, which=TM_FIELD_E_SCA, out=None):
        pts = np.ascontiguousarray(pts, dtype=np.float64) if isinstance(pts, np.ndarray) else pts
        s = np.ascontiguousarray(s, dtype=np.complex128) if isinstance(s, np.ndarray) else s      # None for TM_FIELD_E_INC
        n_pts = int(pts.shape[0])
        if out is None:
            if isinstance(pts, np.ndarray):
                out = np.empty((n_pts, 3), dtype=np.complex128)
            else:
                import torch
                out = torch.empty((n_pts, 3), dtype=torch.complex128, device=pts.device)
        self._check(lib().tm_fields(self._h, n_pts, _ptr(pts), _ptr(s), int(which), _ptr(out)))
        return out

    def pair_cost(self):
        """(fp_instructions, flop) per ordered pair of the active all-pairs kernel."""
        a, b = ctypes.c_double(), ctypes.c_double()
        self._check(lib().tm_pair_cost(self._h, ctypes.byref(a), ctypes.byref(b)))
        return a.value, b.value

    def grad_tmatrix(self, dT, lam, s, out=None):
        """out[j] = lambda_j^T dT_{type(j)} (p_j + (A s)_j)  (tm_grad_tmatrix; PAPER.md Eqs. IV8-IV9)."""
        dT = np.ascontiguousarray(dT, dtype=np.complex128) if isinstance(dT, np.ndarray) else dT
        lam = np.ascontiguousarray(lam, dtype=np.complex128) if isinstance(lam, np.ndarray) else lam
        s = np.ascontiguousarray(s, dtype=np.complex128) if isinstance(s, np.ndarray) else s
        out = np.empty(self.n_scat, dtype=np.complex128) if out is None else out
        self._check(lib().tm_grad_tmatrix(self._h, _ptr(dT), _ptr(lam), _ptr(s), _ptr(out)))
        return out

    def grad_positions(self, lam, s, dp=None, out=None):
        """out[j, alpha] = lambda^T T (dA/dx_{j,alpha}) s (+ mu_j^T dp[j, alpha])  (tm_grad_positions; PAPER.md Eqs. IV3-IV9)."""
        lam = np.ascontiguousarray(lam, dtype=np.complex128) if isinstance(lam, np.ndarray) else lam
        s = np.ascontiguousarray(s, dtype=np.complex128) if isinstance(s, np.ndarray) else s
        if dp is not None and isinstance(dp, np.ndarray):
            dp = np.ascontiguousarray(dp, dtype=np.complex128)
        out = np.empty((self.n_scat, 3), dtype=np.complex128) if out is None else out
        self._check(lib().tm_grad_positions(self._h, _ptr(lam), _ptr(s), _ptr(dp), _ptr(out)))
        return out

    def kernel_time(self, reset=False):
        """reset: True / 1 starts timing mode (events per all-pairs launch), -1 leaves it (tm_kernel_time)."""
        ms, n_ap, n_tot = ctypes.c_double(), ctypes.c_longlong(), ctypes.c_longlong()
        self._check(lib().tm_kernel_time(self._h, int(reset), ctypes.byref(ms), ctypes.byref(n_ap), ctypes.byref(n_tot)))
        return ms.value, n_ap.value, n_tot.value


def solver_for_workload(w, precision=TM_FP64, stream=None, kernel=TM_KERNEL_AUTO):
    """Build a Solver for a workloads.py dict: positions, windows, T (Mie via tm_mie_tmatrix or given full T) and
    the incident field.  Input marshalling only."""
    s = Solver(w["pos"], w["lmax"], w["k"], win_ptr=w["win_ptr"], precision=precision, stream=stream)
    if kernel != TM_KERNEL_AUTO:
        s.set_kernel(kernel)
    if w["t_kind"] in ("mie_types", "mie_sites"):
        T = np.stack([mie_tmatrix(w["lmax"], w["k"], r, w["eps_r"]) for r in w["radii"]])
        s.set_tmatrices(T, w["type_of"], True, r_enclosing=np.asarray(w["radii"], dtype=np.float64))
    else:
        s.set_tmatrices(w["t_full"], w["type_of"], False)
    if w["inc_kind"] == "plane":
        s.set_incident_plane(w["beta"], w["alpha"], w["A_beta"], w["A_alpha"])
    else:
        s.set_incident_gauss(w["focus"], w["w0"], w["Ax"], w["Ay"])
    return s
