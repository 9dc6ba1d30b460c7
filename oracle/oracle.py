"""ctypes wrapper around oracle/mgrhd_oracle.cpp (TEST INFRASTRUCTURE, not product code).

Argument marshalling only: every number comes out of the C++ file.  numpy float64
host arrays in, updated in place.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mgrhd_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None

HIST = 64


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no fast-math, no FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True)
    return _LIB


class _CModel(ctypes.Structure):
    _fields_ = [
        ("Nq", ctypes.c_int),
        ("edges", ctypes.POINTER(ctypes.c_double)),
        ("a_rad", ctypes.c_double),
        ("k_B", ctypes.c_double),
        ("h_planck", ctypes.c_double),
        ("mean_mass", ctypes.c_double),
        ("gamma", ctypes.c_double),
        ("kappa_lo", ctypes.POINTER(ctypes.c_double)),
        ("alpha", ctypes.POINTER(ctypes.c_double)),
        ("closure", ctypes.c_int),
        ("newton_tol", ctypes.c_double),
        ("newton_maxit", ctypes.c_int),
        ("outer_maxit", ctypes.c_int),
        ("outer_tol", ctypes.c_double),
        ("outer_stop", ctypes.c_int),
        ("outer_rel_tol", ctypes.c_double),
        ("spectrum", ctypes.c_int),
        ("opacity_kind", ctypes.c_int),
        ("T_ref", ctypes.c_double),
        ("p_T", ctypes.c_double),
        ("NT", ctypes.c_int),
        ("lnT0", ctypes.c_double),
        ("dlnT", ctypes.c_double),
        ("lnk_edge", ctypes.POINTER(ctypes.c_double)),
        ("outer_mode", ctypes.c_int),
    ]


class _CStats(ctypes.Structure):
    _fields_ = [
        ("n_newton_unconverged", ctypes.c_longlong),
        ("n_outer_unconverged", ctypes.c_longlong),
        ("n_T_nonpositive_steps", ctypes.c_longlong),
        ("n_chiF_guard", ctypes.c_longlong),
        ("n_denominator_nonpositive", ctypes.c_longlong),
        ("n_lu_singular", ctypes.c_longlong),
        ("newton_evals_total", ctypes.c_longlong),
        ("outer_trips_total", ctypes.c_longlong),
        ("newton_hist", ctypes.c_longlong * HIST),
        ("outer_hist", ctypes.c_longlong * HIST),
    ]


def _load():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        d, dp, ip = ctypes.c_double, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
        for name in ("oracle_planck_Y", "oracle_planck_Z", "oracle_planck_Xi"):
            getattr(L, name).restype = d
            getattr(L, name).argtypes = [d]
        L.oracle_planck_dY.restype = d
        L.oracle_planck_dY.argtypes = [d, d]
        L.oracle_chi_mean.restype = d
        L.oracle_chi_mean.argtypes = [d, d, d, d]
        L.oracle_chi_flux.restype = d
        L.oracle_chi_flux.argtypes = [d] * 8 + [ip]
        L.oracle_vP.restype = None
        L.oracle_vP.argtypes = [ctypes.c_int, d, dp, dp, d, dp]
        L.oracle_lu_solve.restype = ctypes.c_int
        L.oracle_lu_solve.argtypes = [ctypes.c_int, dp, dp]
        L.oracle_arrowhead_solve.restype = None
        L.oracle_arrowhead_solve.argtypes = [ctypes.c_int, d, dp, dp, dp, dp, dp]
        L.oracle_source_update.restype = ctypes.c_int
        L.oracle_source_update.argtypes = (
            [ctypes.POINTER(_CModel), ctypes.c_longlong] + [dp] * 11 + [d, d, d, ctypes.POINTER(_CStats)]
        )
        L.oracle_transport_add.restype = ctypes.c_int
        L.oracle_transport_add.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_longlong, d, d, d, d, ctypes.c_int] + [dp] * 8
        L.oracle_imex_step_1d.restype = ctypes.c_int
        L.oracle_imex_step_1d.argtypes = ([ctypes.POINTER(_CModel), ctypes.c_longlong, d, d, d, d, ctypes.c_int] + [dp] * 10
                                          + [ctypes.POINTER(_CStats)])
        L.oracle_free_slopes.restype = None
        L.oracle_free_slopes.argtypes = [ctypes.c_int, dp, dp, dp]
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _arr(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def planck_Y(x: float) -> float:
    return _load().oracle_planck_Y(float(x))


def planck_Z(x: float) -> float:
    return _load().oracle_planck_Z(float(x))


def planck_Xi(x: float) -> float:
    return _load().oracle_planck_Xi(float(x))


def planck_dY(xlo: float, xhi: float) -> float:
    return _load().oracle_planck_dY(float(xlo), float(xhi))


def chi_mean(chi_lo, lnr, a_chi, a_Q) -> float:
    return _load().oracle_chi_mean(float(chi_lo), float(lnr), float(a_chi), float(a_Q))


def chi_flux(chiB, chiE, alpha, chi_lo, Bt, Db, D, aT4):
    g = ctypes.c_int(0)
    v = _load().oracle_chi_flux(*(float(t) for t in (chiB, chiE, alpha, chi_lo, Bt, Db, D, aT4)), ctypes.byref(g))
    return v, g.value


def vP(closure, E, F, v, c):
    F = _arr(F)
    v = _arr(v)
    out = np.zeros(3)
    _load().oracle_vP(int(closure), float(E), _p(F), _p(v), float(c), _p(out))
    return out


def free_slopes(edges, Q) -> np.ndarray:
    """Appendix A (Eq. A1-A2): alpha_{Q,g} from the group integrals Q[Nq]."""
    e, q = _arr(edges), _arr(Q)
    out = np.empty(q.shape[0])
    _load().oracle_free_slopes(q.shape[0], _p(e), _p(q), _p(out))
    return out


def lu_solve(A, b):
    A = _arr(A).copy()
    b = _arr(b).copy()
    n = b.shape[0]
    assert A.shape == (n, n)
    rc = _load().oracle_lu_solve(n, _p(A), _p(b))
    if rc != 0:
        raise ZeroDivisionError("singular matrix")
    return b


def arrowhead_solve(J00, J0g, Jg0, Jgg, rhs):
    J0g, Jg0, Jgg, rhs = (_arr(t) for t in (J0g, Jg0, Jgg, rhs))
    Nq = J0g.shape[0]
    dx = np.zeros(Nq + 1)
    _load().oracle_arrowhead_solve(Nq, float(J00), _p(J0g), _p(Jg0), _p(Jgg), _p(rhs), _p(dx))
    return dx


@dataclass
class OracleModel:
    """Mirror of oracle_model in mgrhd_oracle.cpp (group structure, units, opacity table, controls)."""

    edges: np.ndarray
    kappa_lo: np.ndarray
    alpha: np.ndarray
    a_rad: float = 1.0
    k_B: float = 1.0
    h_planck: float = 1.0
    mean_mass: float = 1.0
    gamma: float = 5.0 / 3.0
    closure: int = 0
    newton_tol: float = 1e-13
    newton_maxit: int = 50
    outer_maxit: int = 50
    outer_tol: float = 1e-13
    outer_stop: int = 1
    outer_rel_tol: float = 1e-12
    spectrum: int = 0            # 0 fixed slope alpha_Q = -1; 1 free slope (Appendix A)
    opacity_kind: int = 0        # 0 table; 1 kappa_lo (T/T_ref)^p_T; 2 ln kappa at the edges tabulated in ln T (Eq. 20)
    T_ref: float = 1.0
    p_T: float = 0.0
    lnT0: float = 0.0
    dlnT: float = 1.0
    lnk_edge: np.ndarray | None = None   # [Nq+1, NT] for opacity_kind 2
    outer_mode: int = 0          # 0 lagged velocity (paper); 1 implicit in v ("variant L")
    _keep: list = field(default_factory=list, repr=False)

    def _c(self) -> _CModel:
        e, k, a = _arr(self.edges), _arr(self.kappa_lo), _arr(self.alpha)
        assert e.shape[0] == k.shape[0] + 1 == a.shape[0] + 1
        t = None if self.lnk_edge is None else _arr(self.lnk_edge)
        if t is not None:
            assert t.ndim == 2 and t.shape[0] == e.shape[0]
        self._keep = [e, k, a, t]
        return _CModel(
            k.shape[0], _p(e), self.a_rad, self.k_B, self.h_planck, self.mean_mass, self.gamma, _p(k), _p(a),
            self.closure, self.newton_tol, self.newton_maxit, self.outer_maxit, self.outer_tol,
            self.outer_stop, self.outer_rel_tol, self.spectrum, self.opacity_kind, self.T_ref, self.p_T,
            0 if t is None else t.shape[1], self.lnT0, self.dlnT, None if t is None else _p(t), self.outer_mode,
        )


def source_update(model: OracleModel, state: dict, dt: float, c: float, c_hat: float) -> dict:
    """Run the oracle in place on a host state dict.

    state: rho[n], mom[3,n], Egas[n], Erad[Nq,n], Frad[3,Nq,n], kappa_scale[n] or None --
    C-contiguous float64 numpy arrays (mom, Egas, Erad, Frad are overwritten).
    Returns the stats as a dict.
    """
    cm = model._c()
    Nq = cm.Nq
    n = state["rho"].shape[0]
    for key, shape in (("rho", (n,)), ("mom", (3, n)), ("Egas", (n,)), ("Erad", (Nq, n)), ("Frad", (3, Nq, n))):
        a = state[key]
        assert a.dtype == np.float64 and a.flags.c_contiguous and a.shape == shape, key
    ks = state.get("kappa_scale")
    if ks is not None:
        assert ks.dtype == np.float64 and ks.flags.c_contiguous and ks.shape == (n,)
    sr = state.get("Srad")
    if sr is not None:
        assert sr.dtype == np.float64 and sr.flags.c_contiguous and sr.shape == (Nq, n)
    st = _CStats()
    rc = _load().oracle_source_update(
        ctypes.byref(cm), n, _p(state["rho"]),
        _p(state["mom"][0]), _p(state["mom"][1]), _p(state["mom"][2]), _p(state["Egas"]), _p(state["Erad"]),
        _p(state["Frad"][0]), _p(state["Frad"][1]), _p(state["Frad"][2]),
        _p(ks) if ks is not None else None, _p(sr) if sr is not None else None,
        float(dt), float(c), float(c_hat), ctypes.byref(st),
    )
    if rc != 0:
        raise ValueError(f"oracle_source_update: argument error {rc}")
    out = {k: getattr(st, k) for k, _ in _CStats._fields_ if not k.endswith("_hist")}
    out["newton_hist"] = np.array(st.newton_hist[:], dtype=np.int64)
    out["outer_hist"] = np.array(st.outer_hist[:], dtype=np.int64)
    return out


def transport_add(src: dict, dst: dict, closure: int, dx: float, wdt: float, c: float, c_hat: float, bc: int = 0) -> None:
    """dst[Erad, Frad] += wdt * T(src) (Eq. 34 in 1-D, reading S22); src, dst: state dicts ([Nq, nx] arrays)."""
    Nq, nx = src["Erad"].shape
    for st in (src, dst):
        assert st["Erad"].flags.c_contiguous and st["Frad"].flags.c_contiguous
    rc = _load().oracle_transport_add(Nq, closure, nx, float(dx), float(wdt), float(c), float(c_hat), bc,
                                      _p(src["Erad"]), _p(src["Frad"][0]), _p(src["Frad"][1]), _p(src["Frad"][2]),
                                      _p(dst["Erad"]), _p(dst["Frad"][0]), _p(dst["Frad"][1]), _p(dst["Frad"][2]))
    if rc != 0:
        raise ValueError(f"oracle_transport_add: argument error {rc}")


def imex_step_1d(model: OracleModel, state: dict, dx: float, dt: float, c: float, c_hat: float, bc: int = 0) -> dict:
    """One two-stage IMEX step (Eq. 35-36) of a 1-D state, in place.  Returns the summed source-update stats."""
    cm = model._c()
    nx = state["rho"].shape[0]
    ks = state.get("kappa_scale")
    st = _CStats()
    rc = _load().oracle_imex_step_1d(
        ctypes.byref(cm), nx, float(dx), float(dt), float(c), float(c_hat), bc, _p(state["rho"]),
        _p(state["mom"][0]), _p(state["mom"][1]), _p(state["mom"][2]), _p(state["Egas"]), _p(state["Erad"]),
        _p(state["Frad"][0]), _p(state["Frad"][1]), _p(state["Frad"][2]), _p(ks) if ks is not None else None,
        ctypes.byref(st))
    if rc != 0:
        raise ValueError(f"oracle_imex_step_1d: argument error {rc}")
    return {k: getattr(st, k) for k, _ in _CStats._fields_ if not k.endswith("_hist")}
