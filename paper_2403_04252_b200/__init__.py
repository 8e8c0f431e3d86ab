"""Thin ctypes binding over libwpccc.so, the C-ABI CUDA library of include/wpccc.h.

Argument marshalling only: every step of the hot path (direct-coupling GEMM, transfer quadrature, factorisation,
RK4 sweep, probabilities) runs in the CUDA kernels of ``csrc/``.  PyTorch supplies device memory and the stream.
There is no CPU fallback: importing works without a GPU (so that the symbol table can be checked), but every
compute call raises ``WpcccError`` when the library cannot run on a CUDA device, and importing raises
``ImportError`` when ``libwpccc.so`` has not been built (``python paper_2403_04252_b200/build.py`` or ``__graft_entry__.build()``).

The function names mirror the C entry points: ``setup_basis`` (wpccc_setup_basis), ``matrix_elements``,
``propagate``, ``probabilities``, ``fp64_peak``, ``last_timing``, ``last_units``.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libwpccc.so")
HEADER_PATH = os.path.join(os.path.dirname(_HERE), "include", "wpccc.h")

if not os.path.exists(LIB_PATH):
    raise ImportError("paper_2403_04252_b200: %s is missing -- build it with `python paper_2403_04252_b200/build.py` "
                      "(there is no CPU fallback)" % LIB_PATH)
_lib = C.CDLL(LIB_PATH)

FAMILIES = ("direct_gemm", "direct_assemble", "transfer_tables", "transfer_contraction", "rotation", "factor", "sweep", "other")


class WpcccError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("wpccc error %d: %s" % (code, msg))
        self.code = code


class _Centre(C.Structure):
    _fields_ = [("Z", C.c_double), ("n_rad", C.c_int), ("l", C.POINTER(C.c_int)), ("eps", C.POINTER(C.c_double)),
                ("kind", C.POINTER(C.c_int)), ("nq", C.POINTER(C.c_int)), ("u", C.POINTER(C.c_double)),
                ("g", C.POINTER(C.c_double))]


class _Quad(C.Structure):
    _fields_ = [("n_rho", C.c_int), ("n_phi", C.c_int), ("n_z", C.c_int), ("rho_max", C.c_double), ("z_pad", C.c_double),
                ("phi_rule", C.c_int), ("kind", C.c_int), ("eta_scale", C.c_double)]


_dp, _ip, _vp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_void_p
_lib.wpccc_basis_bytes.restype = C.c_size_t
_lib.wpccc_basis_bytes.argtypes = [C.c_int, C.POINTER(_Centre), C.c_int, C.c_int, C.POINTER(_Quad)]
_lib.wpccc_setup_basis.restype = C.c_int
_lib.wpccc_setup_basis.argtypes = [C.POINTER(_vp), C.c_int, C.POINTER(_Centre), C.c_double, C.c_int, C.c_double, _dp, C.c_int,
                                   C.POINTER(_Quad), _vp, C.c_size_t, _vp]
_lib.wpccc_setup_basis_grid.restype = C.c_int
_lib.wpccc_setup_basis_grid.argtypes = [C.POINTER(_vp), C.c_int, C.POINTER(_Centre), C.c_double, C.c_int, _dp, _dp, C.c_int,
                                        C.POINTER(_Quad), _vp, C.c_size_t, _vp]
_lib.wpccc_free_basis.restype = None
_lib.wpccc_free_basis.argtypes = [_vp]
for _n in ("wpccc_n_states",):
    getattr(_lib, _n).restype = C.c_int
    getattr(_lib, _n).argtypes = [_vp]
for _n in ("wpccc_n_states_centre", "wpccc_n_rad_centre", "wpccc_n_radial_entries"):
    getattr(_lib, _n).restype = C.c_int
    getattr(_lib, _n).argtypes = [_vp, C.c_int]
_lib.wpccc_radial_entry.restype = C.c_int
_lib.wpccc_radial_entry.argtypes = [_vp, C.c_int, C.c_int, _ip, _ip, _ip]
_lib.wpccc_workspace_bytes.restype = C.c_size_t
_lib.wpccc_workspace_bytes.argtypes = [_vp, C.c_int, C.c_int, C.c_int]
_lib.wpccc_matrix_elements.restype = C.c_int
_lib.wpccc_matrix_elements.argtypes = [_vp, C.c_int, _dp, _dp, _dp, C.c_int, _vp, _vp, _vp, _vp, C.c_size_t, _vp]
_lib.wpccc_propagate.restype = C.c_int
_lib.wpccc_propagate.argtypes = [_vp, C.c_int, _dp, _dp, C.c_double, C.c_double, C.c_int, C.c_int, _vp, _vp, _vp, C.c_size_t, _vp]
_lib.wpccc_propagate_grid.restype = C.c_int
_lib.wpccc_propagate_grid.argtypes = [_vp, C.c_int, _dp, _dp, C.c_int, _dp, C.c_int, _vp, _vp, _vp, C.c_size_t, _vp]
_lib.wpccc_last_status.restype = C.c_int
_lib.wpccc_last_status.argtypes = [_vp, C.c_int, _ip]
_lib.wpccc_set_option.restype = C.c_int
_lib.wpccc_set_option.argtypes = [_vp, C.c_char_p, C.c_longlong]
_lib.wpccc_coupling_matrix_ws_bytes.restype = C.c_size_t
_lib.wpccc_coupling_matrix_ws_bytes.argtypes = [_vp, C.c_int]
_lib.wpccc_coupling_matrix.restype = C.c_int
_lib.wpccc_coupling_matrix.argtypes = [_vp, C.c_int, _dp, _dp, _dp, C.c_int, _vp, _vp, C.c_size_t, _vp]
_lib.wpccc_probabilities.restype = C.c_int
_lib.wpccc_probabilities.argtypes = [_vp, C.c_int, _vp, _dp, _ip, C.c_int, C.c_int, _vp, _vp, _vp, _vp, _vp, _vp]
_lib.wpccc_cross_sections_static.restype = C.c_int
_lib.wpccc_cross_sections_static.argtypes = [C.c_int, C.c_int, _vp, _dp, _ip, C.c_int, _vp, _vp]
_lib.wpccc_last_timing.restype = C.c_int
_lib.wpccc_last_timing.argtypes = [_vp, _dp, C.POINTER(C.c_longlong)]
_lib.wpccc_last_units.restype = C.c_int
_lib.wpccc_last_units.argtypes = [_vp, C.POINTER(C.c_longlong)]
_lib.wpccc_fp64_peak.restype = C.c_double
_lib.wpccc_fp64_peak.argtypes = [C.c_int, _vp]
_lib.wpccc_direct_table_bytes.restype = C.c_size_t
_lib.wpccc_direct_table_bytes.argtypes = [_vp]
_lib.wpccc_enable_direct_tables.restype = C.c_int
_lib.wpccc_enable_direct_tables.argtypes = [_vp, _vp, C.c_size_t, _vp]
_lib.wpccc_last_error.restype = C.c_char_p
_lib.wpccc_version.restype = C.c_char_p

EXPORTS = ("wpccc_basis_bytes", "wpccc_setup_basis", "wpccc_setup_basis_grid", "wpccc_free_basis", "wpccc_n_states", "wpccc_n_states_centre",
           "wpccc_n_rad_centre", "wpccc_n_radial_entries", "wpccc_radial_entry", "wpccc_workspace_bytes",
           "wpccc_matrix_elements", "wpccc_propagate", "wpccc_propagate_grid", "wpccc_last_status", "wpccc_set_option", "wpccc_coupling_matrix_ws_bytes", "wpccc_coupling_matrix", "wpccc_probabilities", "wpccc_cross_sections_static", "wpccc_last_timing", "wpccc_last_units", "wpccc_fp64_peak",
           "wpccc_direct_table_bytes", "wpccc_enable_direct_tables", "wpccc_last_error", "wpccc_version")


def version() -> str:
    return _lib.wpccc_version().decode()


def _check(rc):
    if rc != 0:
        raise WpcccError(rc, _lib.wpccc_last_error().decode())


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _ptr(a, t=C.c_double):
    return a.ctypes.data_as(C.POINTER(t))


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise WpcccError(-3, "no CUDA device: the WP-CCC hot path has no CPU fallback")
    return torch


def _stream(torch):
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _marshal(prob):
    """Problem (wpccc_inputs.Problem-like: centres[], Z_proj, Nr, h, w, lambda_max, quad) -> C structs (+ keep-alive list)."""
    keep, cs = [], (_Centre * len(prob.centres))()
    for i, c in enumerate(prob.centres):
        l, eps, kind, nq = _i32(c.l), _f64(c.eps), _i32(c.kind), _i32(c.nq)
        u = _f64(c.u)
        g = _f64(c.g) if c.g is not None else None
        keep += [l, eps, kind, nq, u, g]
        cs[i].Z, cs[i].n_rad = float(c.Z), len(l)
        cs[i].l, cs[i].eps, cs[i].kind, cs[i].nq = _ptr(l, C.c_int), _ptr(eps), _ptr(kind, C.c_int), _ptr(nq, C.c_int)
        cs[i].u = _ptr(u)
        cs[i].g = _ptr(g) if g is not None else None
    quad = None
    if prob.quad is not None:
        q = prob.quad
        quad = _Quad(int(q["n_rho"]), int(q["n_phi"]), int(q["n_z"]), float(q["rho_max"]), float(q["z_pad"]), int(q.get("phi_rule", 0)),
                     int(q.get("kind", 0)), float(q.get("eta_scale", 1.0)))
    return cs, quad, keep


class Basis:
    """Handle returned by setup_basis: owns the device arena (a torch uint8 tensor) and the wpccc_basis pointer."""

    def __init__(self, prob):
        torch = _torch()
        cs, quad, keep = _marshal(prob)
        qp = C.byref(quad) if quad is not None else None
        nbytes = _lib.wpccc_basis_bytes(len(prob.centres), cs, int(prob.Nr), int(prob.lambda_max), qp)
        if nbytes == 0:
            raise WpcccError(-1, _lib.wpccc_last_error().decode() or "invalid basis description")
        self.arena = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
        base = (self.arena.data_ptr() + 255) & ~255
        w = _f64(prob.w)
        h = C.c_void_p()
        rgrid = getattr(prob, "rgrid", None)             # non-uniform radial grid [Nr+1] (wpccc_setup_basis_grid), else uniform k h
        if rgrid is not None:
            rg = _f64(rgrid)
            _check(_lib.wpccc_setup_basis_grid(C.byref(h), len(prob.centres), cs, float(prob.Z_proj), int(prob.Nr), _ptr(rg), _ptr(w),
                                               int(prob.lambda_max), qp, C.c_void_p(base), nbytes, _stream(torch)))
        else:
            _check(_lib.wpccc_setup_basis(C.byref(h), len(prob.centres), cs, float(prob.Z_proj), int(prob.Nr), float(prob.h), _ptr(w),
                                          int(prob.lambda_max), qp, C.c_void_p(base), nbytes, _stream(torch)))
        self._h = h
        self.n_centres = len(prob.centres)
        self.n_tot = _lib.wpccc_n_states(h)
        self.n_states = [_lib.wpccc_n_states_centre(h, c) for c in range(self.n_centres)]
        self.n_rad = [_lib.wpccc_n_rad_centre(h, c) for c in range(self.n_centres)]
        self.n_entries = [_lib.wpccc_n_radial_entries(h, c) for c in range(self.n_centres)]

    def close(self):
        if getattr(self, "_h", None):
            _lib.wpccc_free_basis(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_option(self, key: str, value: int):
        """wpccc_set_option: choose between CUDA routes ("mirror_pairs", "solve_route", "inverse_kernel", ...; see wpccc.h)."""
        _check(_lib.wpccc_set_option(self._h, key.encode(), int(value)))

    def enable_direct_tables(self, on: bool = True):
        """wpccc_enable_direct_tables: evaluate the radial sums of eq. (7) from prefix/suffix tables
        instead of the DMMA GEMM; the table tensor is owned by this handle.  on=False switches back to the GEMM."""
        torch = _torch()
        if not on:
            _check(_lib.wpccc_enable_direct_tables(self._h, None, 0, _stream(torch)))
            self._dtab = None
            return
        nbytes = _lib.wpccc_direct_table_bytes(self._h)
        self._dtab = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
        base = (self._dtab.data_ptr() + 255) & ~255
        _check(_lib.wpccc_enable_direct_tables(self._h, C.c_void_p(base), nbytes, _stream(torch)))

    def radial_entries(self, c):
        """[(a', a, lambda)] of the radial entries F^c_lambda(a', a) in output order."""
        out, a1, a, lam = [], C.c_int(), C.c_int(), C.c_int()
        for e in range(self.n_entries[c]):
            _check(_lib.wpccc_radial_entry(self._h, c, e, C.byref(a1), C.byref(a), C.byref(lam)))
            out.append((a1.value, a.value, lam.value))
        return out

    def workspace(self, nbytes):
        """The call workspace: ONE torch tensor per process, shared by every handle and grown on demand (a handle is
        single-caller and every compute call has finished with the workspace when it returns)."""
        global _WS
        torch = _torch()
        if _WS is None or _WS.numel() < nbytes + 256:
            _WS = None
            _WS = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
        return C.c_void_p((_WS.data_ptr() + 255) & ~255), _WS.numel() - 256


_WS = None


def release_workspace():
    """Drops the shared call workspace (tens of GB for the large configurations)."""
    global _WS
    _WS = None


def setup_basis(prob) -> Basis:
    """wpccc_setup_basis: stage the basis and the position-independent tables in HBM."""
    return Basis(prob)


def matrix_elements(basis: Basis, b, z, v, phases: bool = True, want_S: bool = True, want_H: bool = True, want_F: bool = False,
                    ws_bytes: int | None = None):
    """wpccc_matrix_elements: (S, H[, F]) as torch tensors on the device; S, H complex128 [n_pos, N, N]."""
    torch = _torch()
    b, z, v = _f64(np.atleast_1d(b)), _f64(np.atleast_1d(z)), _f64(np.atleast_1d(v))
    n, N = len(b), basis.n_tot
    S = torch.empty((n, N, N), dtype=torch.complex128, device="cuda") if want_S else None
    H = torch.empty((n, N, N), dtype=torch.complex128, device="cuda") if want_H else None
    F = torch.empty((n, sum(basis.n_entries)), dtype=torch.float64, device="cuda") if want_F else None
    need = _lib.wpccc_workspace_bytes(basis._h, max(n, 1), 0, 0) if ws_bytes is None else ws_bytes
    ws, cap = basis.workspace(need)
    p = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
    _check(_lib.wpccc_matrix_elements(basis._h, n, _ptr(b), _ptr(z), _ptr(v), (1 if phases else 0) | (2 if want_F else 0),
                                      p(S), p(H), p(F), ws, min(cap, need), _stream(torch)))
    return (S, H, F) if want_F else (S, H)


def coupling_matrix(basis: Basis, b, z, v, phases: bool = True):
    """wpccc_coupling_matrix: the explicit M = -(i/v) S^{-1} H of eq. (4) [n_pos, N, N] complex128 on the device."""
    torch = _torch()
    b, z, v = _f64(np.atleast_1d(b)), _f64(np.atleast_1d(z)), _f64(np.atleast_1d(v))
    n, N = len(b), basis.n_tot
    M = torch.empty((n, N, N), dtype=torch.complex128, device="cuda")
    need = _lib.wpccc_coupling_matrix_ws_bytes(basis._h, max(n, 1))
    ws, cap = basis.workspace(need)
    _check(_lib.wpccc_coupling_matrix(basis._h, n, _ptr(b), _ptr(z), _ptr(v), 1 if phases else 0, C.c_void_p(M.data_ptr()), ws, min(cap, need),
                                      _stream(torch)))
    return M


def _propagate_common(basis, b, v, n_steps, init_state, track_norm, ws_bytes, C0, drift0, allow_singular, call):
    torch = _torch()
    b, v = _f64(np.atleast_1d(b)), _f64(np.atleast_1d(v))
    n, N = len(b), basis.n_tot
    if C0 is not None:                         # continue from given amplitudes (WPCCC_INIT_FROM_DC): updated in place
        if tuple(C0.shape) != (n, N) or C0.dtype != torch.complex128 or not C0.is_cuda or not C0.is_contiguous():
            raise ValueError("C0 must be a contiguous complex128 CUDA tensor [n_traj, N]")
        Cc, init_state = C0, -1
    else:
        Cc = torch.empty((n, N), dtype=torch.complex128, device="cuda")
    drift = None
    if track_norm:
        drift = drift0 if drift0 is not None else torch.zeros(n, dtype=torch.float64, device="cuda")
    need = _lib.wpccc_workspace_bytes(basis._h, max(n, 1), int(n_steps), 1) if ws_bytes is None else ws_bytes
    ws, cap = basis.workspace(need)
    rc = call(n, _ptr(b), _ptr(v), int(init_state), C.c_void_p(Cc.data_ptr()), C.c_void_p(drift.data_ptr()) if track_norm else None, ws,
              min(cap, need), _stream(torch))
    if not (allow_singular and rc == -4):
        _check(rc)
    return (Cc, drift) if track_norm else Cc


def propagate(basis: Basis, b, v, z_min: float, z_max: float, n_steps: int, init_state: int = 0, track_norm: bool = False,
              ws_bytes: int | None = None, C0=None, drift0=None, allow_singular: bool = False):
    """wpccc_propagate: amplitudes c(z_max) [n_traj, N] complex128 on the device (and the norm drift if asked).
    C0: continue from these amplitudes (updated in place).  allow_singular: do not raise on WPCCC_ESINGULAR (the flagged
    trajectories are NaN; see last_status)."""
    return _propagate_common(basis, b, v, n_steps, init_state, track_norm, ws_bytes, C0, drift0, allow_singular,
                             lambda n, bp, vp, ini, cp, dp, ws, nb, st: _lib.wpccc_propagate(
                                 basis._h, n, bp, vp, float(z_min), float(z_max), int(n_steps), ini, cp, dp, ws, nb, st))


def propagate_grid(basis: Basis, b, v, zgrid, init_state: int = 0, track_norm: bool = False, ws_bytes: int | None = None, C0=None,
                   drift0=None, allow_singular: bool = False):
    """wpccc_propagate_grid: the same on an explicit step grid zgrid[0] < ... < zgrid[n] (e.g. the paper's geometric grid)."""
    zg = _f64(zgrid)
    return _propagate_common(basis, b, v, len(zg) - 1, init_state, track_norm, ws_bytes, C0, drift0, allow_singular,
                             lambda n, bp, vp, ini, cp, dp, ws, nb, st: _lib.wpccc_propagate_grid(
                                 basis._h, n, bp, vp, len(zg), _ptr(zg), ini, cp, dp, ws, nb, st))


def last_status(basis: Basis, n_traj: int):
    """wpccc_last_status: per trajectory (code, half_step_index) of the first position whose overlap system could not be
    factorised in the last propagate call (code 1 zero pivot, 2 |S_PT| >= 1, 3 not positive definite), or None."""
    st = (C.c_int * max(n_traj, 1))()
    _check(_lib.wpccc_last_status(basis._h, n_traj, st))
    return [None if st[t] == 0 else (st[t] >> 28, (st[t] & 0x0fffffff) - 1) for t in range(n_traj)]


def probabilities(basis: Basis, Cc, b=None, vgroup=None, n_vgroups: int = 0, init_state: int = 0):
    """wpccc_probabilities: dict of device tensors P_state, P_nl, P_class (and sigma_nl, sigma_class with b, vgroup)."""
    torch = _torch()
    n, N = Cc.shape
    nrt = sum(basis.n_rad)
    out = dict(P_state=torch.empty((n, N), dtype=torch.float64, device="cuda"), P_nl=torch.empty((n, nrt), dtype=torch.float64, device="cuda"),
               P_class=torch.empty((n, 5), dtype=torch.float64, device="cuda"))
    bb = vg = None
    if b is not None and vgroup is not None and n_vgroups > 0:
        bb, vg = _f64(b), _i32(vgroup)
        out["sigma_nl"] = torch.empty((n_vgroups, nrt), dtype=torch.float64, device="cuda")
        out["sigma_class"] = torch.empty((n_vgroups, 5), dtype=torch.float64, device="cuda")
    p = lambda k: C.c_void_p(out[k].data_ptr()) if k in out else None
    Cc = Cc.contiguous()
    _check(_lib.wpccc_probabilities(basis._h, n, C.c_void_p(Cc.data_ptr()), _ptr(bb) if bb is not None else None,
                                    _ptr(vg, C.c_int) if vg is not None else None, int(n_vgroups), int(init_state), p("P_state"), p("P_nl"),
                                    p("P_class"), p("sigma_nl"), p("sigma_class"), _stream(torch)))
    return out


STATIC_MAX_TRAJ, STATIC_MAX_VGROUPS = 16384, 1024     # WPCCC_STATIC_MAX_TRAJ / _VGROUPS of wpccc.h


def cross_sections_static(P, b, vgroup, n_vgroups: int):
    """wpccc_cross_sections_static: sigma [n_vgroups][n_cols] of a probability table P [n_traj][n_cols] (device, float64) with
    the index scratch in the library's static device array: no allocation inside the call (the output tensor is the caller's)."""
    torch = _torch()
    n, ncol = P.shape
    P = P.contiguous()
    sigma = torch.empty((int(n_vgroups), ncol), dtype=torch.float64, device="cuda")
    cross_sections_static_into(P, b, vgroup, n_vgroups, sigma)
    return sigma


def cross_sections_static_into(P, b, vgroup, n_vgroups: int, sigma):
    """The same with the output tensor passed in (nothing at all is allocated on the device)."""
    torch = _torch()
    n, ncol = P.shape
    bb, vg = _f64(b), _i32(vgroup)
    _check(_lib.wpccc_cross_sections_static(int(n), int(ncol), C.c_void_p(P.data_ptr()), _ptr(bb), _ptr(vg, C.c_int), int(n_vgroups),
                                            C.c_void_p(sigma.data_ptr()), _stream(torch)))


def last_timing(basis: Basis):
    """wpccc_last_timing: {family: (milliseconds, launches)} of the last propagate / matrix_elements call."""
    ms = (C.c_double * 8)()
    ln = (C.c_longlong * 8)()
    _lib.wpccc_last_timing(basis._h, ms, ln)
    return {f: (ms[i], ln[i]) for i, f in enumerate(FAMILIES)}


def last_units(basis: Basis):
    """wpccc_last_units: {family: positions processed} of the last propagate / matrix_elements call (0: not counted)."""
    un = (C.c_longlong * 8)()
    _lib.wpccc_last_units(basis._h, un)
    return {f: un[i] for i, f in enumerate(FAMILIES)}


def fp64_peak(kind: int) -> float:
    """wpccc_fp64_peak: measured FP64 TFLOP/s of the DFMA (kind 0) or DMMA m8n8k4 (kind 1) pipe."""
    torch = _torch()
    r = _lib.wpccc_fp64_peak(int(kind), _stream(torch))
    if r < 0:
        raise WpcccError(int(r), _lib.wpccc_last_error().decode())
    return r
