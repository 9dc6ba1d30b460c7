"""Seeded synthetic inputs for the five BASELINE.json workloads.

This module serves BOTH the oracle tests and the CUDA path and therefore holds none of
the method's arithmetic: it only draws numbers.  Random draws come from one counter-based
64-bit hash of (seed, field, cell, group), so any cell range of any workload can be
generated independently, on the CPU or directly in GPU memory (torch ops only).

The "Planck-shaped" group energies E_g(T_r) are produced by a fixed 32-node Gauss-Legendre
rule applied to the *definition* int x^3/(e^x-1) dx in ln x (accuracy ~1e-6; it only
shapes the input and is no claim about the method's B_g).  The oracle is always fed a host
copy of the very buffers the GPU updates, so CPU/GPU libm differences never enter parity.

State layout (structure of arrays, float64, cell index fastest):
  rho[n]  mom[3][n]  Egas[n]  Erad[Nq][n]  Frad[3][Nq][n]  kappa_scale[n] | None
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
import torch

_M64 = (1 << 64) - 1


def _s64(v: int) -> int:
    v &= _M64
    return v - (1 << 64) if v >= (1 << 63) else v


_C1 = _s64(0xBF58476D1CE4E5B9)
_C2 = _s64(0x94D049BB133111EB)
_GOLD = _s64(0x9E3779B97F4A7C15)
_K_CELL = _s64(0xD6E8FEB86659FD93)
_K_GROUP = _s64(0xA0761D6478BD642F)
_K_FIELD = _s64(0xE7037ED1A0B428DB)
_K_SEED = _s64(0x8EBC6AF09C88C6E3)


def _lsr(x: torch.Tensor, k: int) -> torch.Tensor:
    return (x >> k) & ((1 << (64 - k)) - 1)


def _mix(z: torch.Tensor) -> torch.Tensor:
    z = (z ^ _lsr(z, 30)) * _C1
    z = (z ^ _lsr(z, 27)) * _C2
    return z ^ _lsr(z, 31)


def uniform01(seed: int, fld: int, cell: torch.Tensor, group: int = 0) -> torch.Tensor:
    """U(0,1) float64, a pure function of (seed, fld, cell, group). cell: int64 tensor."""
    const = _s64(group * (_K_GROUP & _M64) + fld * (_K_FIELD & _M64) + seed * (_K_SEED & _M64) + (_GOLD & _M64))
    z = _mix(_mix(cell * _K_CELL + const) + _GOLD)
    return (_lsr(z, 11).to(torch.float64) + 0.5) * (2.0 ** -53)


def normal01(seed: int, fld: int, cell: torch.Tensor, group: int = 0) -> torch.Tensor:
    u1 = uniform01(seed, fld, cell, group)
    u2 = uniform01(seed, fld + 1000, cell, group)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos(2.0 * math.pi * u2)


def _scalar_uniforms(seed: int, fld: int, count: int) -> np.ndarray:
    idx = torch.arange(count, dtype=torch.int64)
    return uniform01(seed, fld, idx).numpy()


# field ids
F_RHO, F_T, F_VMU, F_VPHI, F_VMAG, F_TR, F_ENOISE, F_FMU, F_FPHI, F_FMAG, F_KAPPA0, F_TAB_K, F_TAB_A, F_DT = range(14)

_GL_T, _GL_W = np.polynomial.legendre.leggauss(32)


def planck_shaped_group_energy(a_rad: float, Tr: torch.Tensor, xlo: torch.Tensor, xhi: torch.Tensor) -> torch.Tensor:
    """a_rad Tr^4 (15/pi^4) int_xlo^xhi x^3/(e^x-1) dx by a fixed Gauss-Legendre rule in ln x."""
    b = torch.minimum(xhi, torch.clamp(xlo, min=1.0) + 45.0)
    a = torch.where(xlo > 0, xlo, 1e-4 * torch.clamp(b, max=1.0))
    la, lb = torch.log(a), torch.log(b)
    half = 0.5 * (lb - la)
    t = torch.as_tensor(_GL_T, dtype=torch.float64, device=Tr.device)[:, None]
    w = torch.as_tensor(_GL_W, dtype=torch.float64, device=Tr.device)[:, None]
    x = torch.exp(la[None, :] + half[None, :] * (t + 1.0))
    integrand = x ** 4 / torch.expm1(x)
    integral = (w * integrand).sum(0) * half
    return a_rad * Tr ** 4 * (15.0 / math.pi ** 4) * integral


@dataclass
class Workload:
    """One BASELINE.json config: group structure, units, opacity table, controls, and the state recipe."""

    name: str
    index: int                      # 1..5 as in BASELINE.json / SURVEY 8(d)
    ncells: int
    Nq: int
    edges: np.ndarray               # [Nq+1], h nu / k_B units (h = k_B = 1)
    kappa_lo: np.ndarray            # [Nq]
    alpha: np.ndarray               # [Nq]
    seed: int
    a_rad: float
    c: float
    c_hat: float
    dt: float
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
    ncalls: int = 1
    extra: dict = field(default_factory=dict)

    @property
    def Cv_over_rho(self) -> float:
        return self.k_B / ((self.gamma - 1.0) * self.mean_mass)

    def dt_of_call(self, i: int) -> float:
        """Config 5 varies dt per call: dt_i = dt0 * 10^U[-.5,.5]; other configs use dt."""
        if self.index != 5:
            return self.dt
        u = float(_scalar_uniforms(self.seed, F_DT, i + 1)[i])
        return self.dt * 10.0 ** (u - 0.5)

    def state_bytes(self, ncells: int | None = None) -> int:
        n = self.ncells if ncells is None else ncells
        return 8 * n * (5 + 4 * self.Nq + (1 if self.index != 1 else 0))

    # ------------------------------------------------------------------
    def make_state(self, device="cpu", cell_start: int = 0, ncells: int | None = None,
                   chunk: int = 1 << 20) -> dict:
        """Generate cells [cell_start, cell_start+ncells) of this workload on `device`."""
        n = self.ncells if ncells is None else ncells
        dev = torch.device(device)
        f64 = dict(dtype=torch.float64, device=dev)
        st = {
            "rho": torch.empty(n, **f64),
            "mom": torch.empty(3, n, **f64),
            "Egas": torch.empty(n, **f64),
            "Erad": torch.empty(self.Nq, n, **f64),
            "Frad": torch.empty(3, self.Nq, n, **f64),
            "kappa_scale": None if self.index == 1 else torch.empty(n, **f64),
        }
        for lo in range(0, n, chunk):
            hi = min(n, lo + chunk)
            cell = torch.arange(cell_start + lo, cell_start + hi, dtype=torch.int64, device=dev)
            self._fill(st, slice(lo, hi), cell)
        return st

    def _fill(self, st: dict, sl: slice, cell: torch.Tensor) -> None:
        s, i = self.seed, self.index
        U = lambda fld, g=0: uniform01(s, fld, cell, g)  # noqa: E731
        N = lambda fld, g=0: normal01(s, fld, cell, g)   # noqa: E731
        c = self.c
        # gas
        if i == 1:
            rho = 0.5 + 1.5 * U(F_RHO)
            T = 0.5 + 1.5 * U(F_T)
            beta = torch.zeros_like(rho)
        elif i == 2:
            rho = torch.exp(0.5 * N(F_RHO))
            T = 0.3 + 2.7 * U(F_T)
            beta = 1e-3 * U(F_VMAG)
        elif i == 3:
            rho = 1.0 + 9.0 * U(F_RHO)
            T = 0.5 + 4.5 * U(F_T)
            beta = 1e-2 * U(F_VMAG)
        else:
            rho = torch.exp(N(F_RHO))
            T = 10.0 ** torch.clamp(0.5 * N(F_T), -1.0, 1.0)
            beta = 1e-2 * U(F_VMAG)
        mu = 2.0 * U(F_VMU) - 1.0
        phi = 2.0 * math.pi * U(F_VPHI)
        sin = torch.sqrt(torch.clamp(1.0 - mu * mu, min=0.0))
        vmag = beta * c
        v = torch.stack([vmag * sin * torch.cos(phi), vmag * sin * torch.sin(phi), vmag * mu])
        st["rho"][sl] = rho
        st["mom"][:, sl] = rho[None, :] * v
        st["Egas"][sl] = self.Cv_over_rho * rho * T + 0.5 * rho * (v * v).sum(0)
        # per-cell opacity scale
        if i == 2:
            st["kappa_scale"][sl] = 0.1 + 9.9 * U(F_KAPPA0)
        elif i == 3:
            st["kappa_scale"][sl] = 10.0 ** (4.0 + 2.0 * U(F_KAPPA0)) / (c * rho * self.dt)
        elif i == 4:
            st["kappa_scale"][sl] = 10.0 / (c * rho * self.dt)
        elif i == 5:
            st["kappa_scale"][sl] = 10.0 ** (-2.0 + 8.0 * U(F_KAPPA0)) / (c * rho * self.dt)
        # radiation
        if i == 1:
            Tr = 0.5 + 1.5 * U(F_TR)
        else:
            Tr = T * (1.0 + 0.3 * (2.0 * U(F_TR) - 1.0))
        fmax = {1: 0.0, 2: 0.5, 3: 0.1, 4: 0.9, 5: 0.9}[i]
        edges = torch.as_tensor(self.edges, dtype=torch.float64, device=cell.device)
        for g in range(self.Nq):
            xlo = self.h_planck * edges[g] / (self.k_B * Tr)
            xhi = self.h_planck * edges[g + 1] / (self.k_B * Tr)
            Eg = planck_shaped_group_energy(self.a_rad, Tr, xlo, xhi)
            if i == 1:
                Eg = Eg * (1.0 + 0.1 * (2.0 * U(F_ENOISE, g) - 1.0))
            st["Erad"][g, sl] = Eg
            if fmax == 0.0:
                st["Frad"][:, g, sl] = 0.0
                continue
            fm = fmax * U(F_FMAG, g) * c * Eg
            mu = 2.0 * U(F_FMU, g) - 1.0
            phi = 2.0 * math.pi * U(F_FPHI, g)
            sin = torch.sqrt(torch.clamp(1.0 - mu * mu, min=0.0))
            st["Frad"][0, g, sl] = fm * sin * torch.cos(phi)
            st["Frad"][1, g, sl] = fm * sin * torch.sin(phi)
            st["Frad"][2, g, sl] = fm * mu


def workload(index: int, ncells: int | None = None) -> Workload:
    """The five BASELINE.json configs (1-based index); `ncells` overrides the size for tests."""
    scaled = dict(a_rad=1e-3, c=1e3)   # configs 2-5, SURVEY 8(d) "Unit systems"
    if index == 1:
        k = 0.1 + 9.9 * _scalar_uniforms(0, F_TAB_K, 4)
        return Workload("static_relaxation_16c_Nq4", 1, ncells or 16 ** 3, 4,
                        np.array([0.0, 1e-2, 1.0, 1e2, np.inf]), k, np.zeros(4), seed=0,
                        a_rad=1.0, c=1.0, c_hat=1.0, dt=1.0 / (1.0 * 1.25 * float(k.mean())))
    if index == 2:
        e = np.logspace(-2, 2, 9)
        return Workload("moving_gas_64c_Nq8", 2, ncells or 64 ** 3, 8, e, e[:-1] ** -2.0, np.full(8, -2.0),
                        seed=1, c_hat=scaled["c"], dt=1.0 / scaled["c"], **scaled)
    if index == 3:
        e = np.logspace(-3, 3, 17)
        return Workload("thick_diffusion_128c_Nq16", 3, ncells or 128 ** 3, 16, e, e[:-1] ** -3.0, np.full(16, -3.0),
                        seed=2, c_hat=0.1 * scaled["c"], dt=1.0 / scaled["c"], **scaled)
    if index == 4:
        e = np.logspace(-3, 3, 33)
        k = 10.0 ** (-3.0 + 3.0 * _scalar_uniforms(3, F_TAB_K, 32))
        a = -4.0 + 6.0 * _scalar_uniforms(3, F_TAB_A, 32)
        return Workload("variable_opacity_256c_Nq32", 4, ncells or 256 ** 3, 32, e, k, a,
                        seed=3, c_hat=scaled["c"], dt=1.0 / scaled["c"], **scaled)
    if index == 5:
        e = np.logspace(-4, 4, 65)
        k = 10.0 ** (-3.0 + 3.0 * _scalar_uniforms(4, F_TAB_K, 64))
        a = -4.0 + 6.0 * _scalar_uniforms(4, F_TAB_A, 64)
        return Workload("sustained_256c_Nq64", 5, ncells or 256 ** 3, 64, e, k, a,
                        seed=4, c_hat=scaled["c"], dt=1.0 / scaled["c"], ncalls=100, **scaled)
    raise ValueError("workload index must be 1..5")


def to_numpy(state: dict) -> dict:
    """Host float64 C-contiguous copy of a state dict (what the oracle consumes)."""
    return {k: (None if v is None else np.ascontiguousarray(v.detach().cpu().numpy()).copy())
            for k, v in state.items()}


def clone_state(state: dict) -> dict:
    return {k: (None if v is None else v.clone()) for k, v in state.items()}
