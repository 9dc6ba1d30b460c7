"""Thin ctypes binding of the C ABI in include/mgrhd.h -- argument marshalling only.

Every step of the update runs in the CUDA kernels of libmgrhd.so; nothing here computes and
there is no CPU fallback: if the library is missing or CUDA is unusable the calls raise.
Names mirror the C entry points (mgrhd_init -> Context(...), mgrhd_source_update ->
Context.source_update, ...).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmgrhd.so")
MAX_GROUPS = 64
HIST = 64

EXPORTS = (
    "mgrhd_init", "mgrhd_source_update", "mgrhd_source_update_host", "mgrhd_source_update_static", "mgrhd_conserved_totals",
    "mgrhd_transport_add", "mgrhd_imex_step_1d",
    "mgrhd_get_stats", "mgrhd_reset_stats", "mgrhd_set_flop_counting", "mgrhd_launch_count", "mgrhd_planck_edge_functions", "mgrhd_measure_dfma_peak",
    "mgrhd_last_error", "mgrhd_free",
)

_dp = ctypes.POINTER(ctypes.c_double)


class Units(ctypes.Structure):
    _fields_ = [("a_rad", ctypes.c_double), ("k_B", ctypes.c_double), ("h_planck", ctypes.c_double),
                ("mean_mass", ctypes.c_double), ("gamma", ctypes.c_double)]


class OpacityModel(ctypes.Structure):
    _fields_ = [("kappa_lo", _dp), ("alpha", _dp), ("closure", ctypes.c_int), ("spectrum", ctypes.c_int),
                ("newton_tol", ctypes.c_double), ("newton_maxit", ctypes.c_int), ("outer_maxit", ctypes.c_int),
                ("outer_tol", ctypes.c_double), ("outer_stop", ctypes.c_int), ("outer_rel_tol", ctypes.c_double),
                ("opacity_kind", ctypes.c_int), ("T_ref", ctypes.c_double), ("p_T", ctypes.c_double),
                ("NT", ctypes.c_int), ("lnT0", ctypes.c_double), ("dlnT", ctypes.c_double), ("lnk_edge", _dp),
                ("outer_mode", ctypes.c_int)]


class State(ctypes.Structure):
    _fields_ = [("rho", ctypes.c_void_p), ("mom", ctypes.c_void_p * 3), ("Egas", ctypes.c_void_p),
                ("Erad", ctypes.c_void_p), ("Frad", ctypes.c_void_p * 3), ("kappa_scale", ctypes.c_void_p),
                ("Srad", ctypes.c_void_p)]


class Stats(ctypes.Structure):
    _fields_ = [("n_cells", ctypes.c_longlong), ("n_newton_unconverged", ctypes.c_longlong),
                ("n_outer_unconverged", ctypes.c_longlong), ("n_T_nonpositive_steps", ctypes.c_longlong),
                ("n_chiF_guard", ctypes.c_longlong), ("n_denominator_nonpositive", ctypes.c_longlong),
                ("newton_evals_total", ctypes.c_longlong), ("outer_trips_total", ctypes.c_longlong), ("flops", ctypes.c_longlong),
                ("newton_hist", ctypes.c_longlong * HIST), ("outer_hist", ctypes.c_longlong * HIST)]


class MgrhdError(RuntimeError):
    pass


_lib = None


def load_library() -> ctypes.CDLL:
    """dlopen libmgrhd.so (built by paper_2407_18304_b200.build) and declare the prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise MgrhdError(f"{LIB_PATH} not built: run `python -m paper_2407_18304_b200.build` "
                         "(there is no CPU fallback)")
    L = ctypes.CDLL(LIB_PATH)
    vp, ll, d, i = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_double, ctypes.c_int
    L.mgrhd_init.restype = i
    L.mgrhd_init.argtypes = [ctypes.POINTER(vp), _dp, i, ctypes.POINTER(Units), ctypes.POINTER(OpacityModel)]
    L.mgrhd_source_update.restype = i
    L.mgrhd_source_update.argtypes = [vp, ctypes.POINTER(State), ll, d, d, d, vp]
    L.mgrhd_source_update_static.restype = i
    L.mgrhd_source_update_static.argtypes = [_dp, i, ctypes.POINTER(Units), ctypes.POINTER(OpacityModel),
                                             ctypes.POINTER(State), ll, d, d, d, vp, ctypes.POINTER(Stats)]
    L.mgrhd_source_update_host.restype = i
    L.mgrhd_source_update_host.argtypes = [vp, ctypes.POINTER(State), ll, d, d, d]
    L.mgrhd_transport_add.restype = i
    L.mgrhd_transport_add.argtypes = [vp, ctypes.POINTER(State), ctypes.POINTER(State), ll, d, d, d, d, i, vp]
    L.mgrhd_imex_step_1d.restype = i
    L.mgrhd_imex_step_1d.argtypes = [vp, ctypes.POINTER(State), ctypes.POINTER(State), ll, d, d, d, d, i, vp]
    L.mgrhd_conserved_totals.restype = i
    L.mgrhd_conserved_totals.argtypes = [vp, ctypes.POINTER(State), ll, d, d, vp, vp, vp]
    L.mgrhd_get_stats.restype = i
    L.mgrhd_get_stats.argtypes = [vp, ctypes.POINTER(Stats)]
    L.mgrhd_reset_stats.restype = i
    L.mgrhd_reset_stats.argtypes = [vp]
    L.mgrhd_set_flop_counting.restype = i
    L.mgrhd_set_flop_counting.argtypes = [vp, i]
    L.mgrhd_launch_count.restype = ll
    L.mgrhd_launch_count.argtypes = [vp]
    L.mgrhd_planck_edge_functions.restype = i
    L.mgrhd_planck_edge_functions.argtypes = [vp, ll, vp, vp, vp, i, vp]
    L.mgrhd_measure_dfma_peak.restype = i
    L.mgrhd_measure_dfma_peak.argtypes = [ll, _dp]
    L.mgrhd_last_error.restype = ctypes.c_char_p
    L.mgrhd_last_error.argtypes = []
    L.mgrhd_free.restype = None
    L.mgrhd_free.argtypes = [vp]
    _lib = L
    return L


_ERR = {-1: "MGRHD_ERR_ARG", -2: "MGRHD_ERR_RANGE", -3: "MGRHD_ERR_EDGES", -4: "MGRHD_ERR_ALPHA",
        -5: "MGRHD_ERR_CUDA", -6: "MGRHD_ERR_SIZE"}


def _check(rc: int, what: str) -> None:
    if rc != 0:
        msg = load_library().mgrhd_last_error().decode() if rc in (-5, -6) else ""
        raise MgrhdError(f"{what}: {_ERR.get(rc, rc)} {msg}".strip())


def _ptr(t) -> int:
    """Address of a torch tensor (device or host) or numpy array; float64, contiguous."""
    if t is None:
        return 0
    if isinstance(t, np.ndarray):
        assert t.dtype == np.float64 and t.flags.c_contiguous
        return t.ctypes.data
    assert str(t.dtype) == "torch.float64" and t.is_contiguous()
    return t.data_ptr()


def _state_struct(state: dict, Nq: int, n: int) -> State:
    """state: rho[n] mom[3,n] Egas[n] Erad[Nq,n] Frad[3,Nq,n] kappa_scale[n]|None (workloads.py layout)."""
    for key, shape in (("rho", (n,)), ("mom", (3, n)), ("Egas", (n,)), ("Erad", (Nq, n)), ("Frad", (3, Nq, n))):
        assert tuple(state[key].shape) == shape, (key, tuple(state[key].shape), shape)
    s = State()
    s.rho = _ptr(state["rho"])
    s.Egas = _ptr(state["Egas"])
    s.Erad = _ptr(state["Erad"])
    s.kappa_scale = _ptr(state.get("kappa_scale"))
    if state.get("Srad") is not None:
        assert tuple(state["Srad"].shape) == (Nq, n), ("Srad", tuple(state["Srad"].shape))
    s.Srad = _ptr(state.get("Srad"))
    row = 8 * n
    m0, f0 = _ptr(state["mom"]), _ptr(state["Frad"])
    for k in range(3):
        s.mom[k] = m0 + k * row
        s.Frad[k] = f0 + k * Nq * row
    return s


class Context:
    """mgrhd_ctx: one group structure / unit system / opacity model on the current CUDA device."""

    def __init__(self, edges, kappa_lo, alpha, *, a_rad=1.0, k_B=1.0, h_planck=1.0, mean_mass=1.0,
                 gamma=5.0 / 3.0, closure=0, spectrum=0, newton_tol=1e-11, newton_maxit=50, outer_maxit=50,
                 outer_tol=1e-13, outer_stop=1, outer_rel_tol=1e-12, opacity_kind=0, T_ref=1.0, p_T=0.0,
                 lnT0=0.0, dlnT=1.0, lnk_edge=None, outer_mode=0):
        L = load_library()
        e = np.ascontiguousarray(edges, dtype=np.float64)
        self.Nq = int(e.shape[0]) - 1
        k = None if kappa_lo is None else np.ascontiguousarray(kappa_lo, dtype=np.float64)
        a = None if alpha is None else np.ascontiguousarray(alpha, dtype=np.float64)
        if (k is not None and k.shape[0] != self.Nq) or (a is not None and a.shape[0] != self.Nq):
            raise MgrhdError("edges must have Nq+1 entries and kappa_lo, alpha Nq")
        t = None if lnk_edge is None else np.ascontiguousarray(lnk_edge, dtype=np.float64)
        if t is not None and (t.ndim != 2 or t.shape[0] != self.Nq + 1):
            raise MgrhdError("lnk_edge must be [Nq+1, NT]")
        u = Units(a_rad, k_B, h_planck, mean_mass, gamma)
        null = ctypes.cast(None, _dp)
        m = OpacityModel(null if k is None else k.ctypes.data_as(_dp), null if a is None else a.ctypes.data_as(_dp),
                         closure, spectrum, newton_tol, newton_maxit, outer_maxit, outer_tol, outer_stop, outer_rel_tol,
                         opacity_kind, T_ref, p_T, 0 if t is None else t.shape[1], lnT0, dlnT,
                         null if t is None else t.ctypes.data_as(_dp), outer_mode)
        h = ctypes.c_void_p()
        _check(L.mgrhd_init(ctypes.byref(h), e.ctypes.data_as(_dp), self.Nq, ctypes.byref(u), ctypes.byref(m)),
               "mgrhd_init")
        self._h = h
        self._L = L

    @classmethod
    def from_workload(cls, wl, **kw) -> "Context":
        args = dict(a_rad=wl.a_rad, k_B=wl.k_B, h_planck=wl.h_planck,
                    mean_mass=wl.mean_mass, gamma=wl.gamma, closure=wl.closure, newton_tol=wl.newton_tol,
                    newton_maxit=wl.newton_maxit, outer_maxit=wl.outer_maxit, outer_tol=wl.outer_tol,
                    outer_stop=wl.outer_stop, outer_rel_tol=wl.outer_rel_tol)
        for key in ("spectrum", "opacity_kind", "T_ref", "p_T", "lnT0", "dlnT", "lnk_edge", "outer_mode"):   # optional model fields
            if hasattr(wl, key):
                args[key] = getattr(wl, key)
        args.update(kw)
        return cls(wl.edges, wl.kappa_lo, wl.alpha, **args)

    def source_update(self, state: dict, dt: float, c: float, c_hat: float, stream=None) -> None:
        """mgrhd_source_update on DEVICE tensors, in place, stream-ordered (default: torch's current stream)."""
        n = int(state["rho"].shape[0])
        assert state["rho"].is_cuda, "mgrhd_source_update takes device tensors (use source_update_host)"
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        s = _state_struct(state, self.Nq, n)
        _check(self._L.mgrhd_source_update(self._h, ctypes.byref(s), n, dt, c, c_hat, ctypes.c_void_p(stream)),
               "mgrhd_source_update")

    def source_update_host(self, state: dict, dt: float, c: float, c_hat: float) -> None:
        """mgrhd_source_update_host on HOST tensors / numpy arrays, in place, synchronous."""
        n = int(state["rho"].shape[0])
        s = _state_struct(state, self.Nq, n)
        _check(self._L.mgrhd_source_update_host(self._h, ctypes.byref(s), n, dt, c, c_hat),
               "mgrhd_source_update_host")

    def transport_add(self, src: dict, dst: dict, dx: float, w_dt: float, c: float, c_hat: float, bc: int = 0,
                      stream=None) -> None:
        """mgrhd_transport_add: dst[Erad, Frad] += w_dt * T(src) along a 1-D row of DEVICE tensors."""
        n = int(src["rho"].shape[0])
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        a, b = _state_struct(src, self.Nq, n), _state_struct(dst, self.Nq, n)
        _check(self._L.mgrhd_transport_add(self._h, ctypes.byref(a), ctypes.byref(b), n, dx, w_dt, c, c_hat, bc,
                                           ctypes.c_void_p(stream)), "mgrhd_transport_add")

    def imex_step_1d(self, state: dict, work: dict, dx: float, dt: float, c: float, c_hat: float, bc: int = 0,
                     stream=None) -> None:
        """mgrhd_imex_step_1d: one two-stage IMEX step (Eq. 35-36) of a 1-D row, in place; `work` is scratch."""
        n = int(state["rho"].shape[0])
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        a, b = _state_struct(state, self.Nq, n), _state_struct(work, self.Nq, n)
        _check(self._L.mgrhd_imex_step_1d(self._h, ctypes.byref(a), ctypes.byref(b), n, dx, dt, c, c_hat, bc,
                                          ctypes.c_void_p(stream)), "mgrhd_imex_step_1d")

    def conserved_totals(self, state: dict, c: float, c_hat: float, out_energy, out_momentum, stream=None) -> None:
        n = int(state["rho"].shape[0])
        if stream is None:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        s = _state_struct(state, self.Nq, n)
        assert tuple(out_energy.shape) == (n,) and tuple(out_momentum.shape) == (3, n)
        _check(self._L.mgrhd_conserved_totals(self._h, ctypes.byref(s), n, c, c_hat, _ptr(out_energy),
                                              _ptr(out_momentum), ctypes.c_void_p(stream)),
               "mgrhd_conserved_totals")

    def get_stats(self) -> dict:
        st = Stats()
        _check(self._L.mgrhd_get_stats(self._h, ctypes.byref(st)), "mgrhd_get_stats")
        out = {k: getattr(st, k) for k, _ in Stats._fields_ if not k.endswith("_hist")}
        out["newton_hist"] = np.array(st.newton_hist[:], dtype=np.int64)
        out["outer_hist"] = np.array(st.outer_hist[:], dtype=np.int64)
        return out

    def reset_stats(self) -> None:
        _check(self._L.mgrhd_reset_stats(self._h), "mgrhd_reset_stats")

    def set_flop_counting(self, on: bool) -> None:
        _check(self._L.mgrhd_set_flop_counting(self._h, 1 if on else 0), "mgrhd_set_flop_counting")

    def launch_count(self) -> int:
        return int(self._L.mgrhd_launch_count(self._h))

    def free(self) -> None:
        if getattr(self, "_h", None):
            self._L.mgrhd_free(self._h)
            self._h = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def measure_dfma_peak(iters: int = 1 << 20) -> float:
    """FP64 FMA/s of the current device (mgrhd_measure_dfma_peak)."""
    out = ctypes.c_double(0.0)
    _check(load_library().mgrhd_measure_dfma_peak(iters, ctypes.byref(out)), "mgrhd_measure_dfma_peak")
    return out.value


STATIC_SCRATCH_BYTES = 12 << 20


def source_update_static(wl, state: dict, dt: float, c: float, c_hat: float, stream=None, want_stats=False):
    """mgrhd_source_update_static: the update of DEVICE tensors in place with no context and no device allocation
    (scratch and counters in static device arrays of the library; see include/mgrhd.h for the limits and the
    sharing rule).  wl: anything with the attributes Context.from_workload reads.  Returns the call's counters
    when want_stats (which synchronises the stream), else None."""
    L = load_library()
    e = np.ascontiguousarray(wl.edges, dtype=np.float64)
    Nq = int(e.shape[0]) - 1
    k = np.ascontiguousarray(wl.kappa_lo, dtype=np.float64)
    a = np.ascontiguousarray(wl.alpha, dtype=np.float64)
    if k.shape[0] != Nq or a.shape[0] != Nq:
        raise MgrhdError("edges must have Nq+1 entries and kappa_lo, alpha Nq")
    u = Units(wl.a_rad, wl.k_B, wl.h_planck, wl.mean_mass, wl.gamma)
    m = OpacityModel(k.ctypes.data_as(_dp), a.ctypes.data_as(_dp), wl.closure, getattr(wl, "spectrum", 0), wl.newton_tol,
                     wl.newton_maxit, wl.outer_maxit, wl.outer_tol, wl.outer_stop, wl.outer_rel_tol,
                     getattr(wl, "opacity_kind", 0), getattr(wl, "T_ref", 1.0), getattr(wl, "p_T", 0.0), 0, 0.0, 1.0,
                     ctypes.cast(None, _dp), getattr(wl, "outer_mode", 0))
    n = int(state["rho"].shape[0])
    assert state["rho"].is_cuda, "mgrhd_source_update_static takes device tensors"
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    s = _state_struct(state, Nq, n)
    st = Stats()
    _check(L.mgrhd_source_update_static(e.ctypes.data_as(_dp), Nq, ctypes.byref(u), ctypes.byref(m), ctypes.byref(s), n,
                                        dt, c, c_hat, ctypes.c_void_p(stream), ctypes.byref(st) if want_stats else None),
           "mgrhd_source_update_static")
    if not want_stats:
        return None
    out = {key: getattr(st, key) for key, _ in Stats._fields_ if not key.endswith("_hist")}
    out["newton_hist"] = np.array(st.newton_hist[:], dtype=np.int64)
    out["outer_hist"] = np.array(st.outer_hist[:], dtype=np.int64)
    return out


def planck_edge_functions(x, form=0):
    """mgrhd_planck_edge_functions on a CUDA float64 tensor x; returns (yz, xi, is_y) tensors.  form 0: per-interval
    rows (Nq <= 32), 1: three branches (Nq <= 64, general kernel)."""
    import torch

    assert x.is_cuda and x.dtype == torch.float64 and x.is_contiguous()
    yz, xi = torch.empty_like(x), torch.empty_like(x)
    is_y = torch.empty(x.shape, dtype=torch.int32, device=x.device)
    _check(load_library().mgrhd_planck_edge_functions(x.data_ptr(), x.numel(), yz.data_ptr(), xi.data_ptr(),
                                                      is_y.data_ptr(), form, ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)),
           "mgrhd_planck_edge_functions")
    return yz, xi, is_y
