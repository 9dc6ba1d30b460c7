"""Seeded inputs that make the guard branches of the update fire (readings S8, S9) --
drawn here with numpy only (no method arithmetic), used by the oracle pins (CPU) and by the GPU
parity tests so that both implementations execute the same branches on the same cells.

  s8ii_case:  wide groups in the Rayleigh-Jeans range with rising opacity (r = 10, alpha = 2) make Eq. 27
              negative (chi_F/chi_E = -7.9) and c_hat chi_F dt < -1, so the guard
              "1 + c_hat chi_F dt <= 0 -> chi_F = chi_E" fires in two of the four groups of every cell.
  s9_case:    radiation-dominated moving cells (E_rad >> E_gas): the gas momentum gained in the first outer
              trip carries more kinetic energy than the gas has in total, so T <= 0 at the start of the
              second trip: the "invalid state" guard stops the iteration and the cell keeps the first
              trip's result.  (The step-halving half of S9 cannot fire: see DESIGN.md section 2.)
"""
import numpy as np


class GuardCase:
    def __init__(self, edges, kappa_lo, alpha, state, dt, c, c_hat, a_rad):
        self.edges, self.kappa_lo, self.alpha = edges, kappa_lo, alpha
        self.state, self.dt, self.c, self.c_hat, self.a_rad = state, dt, c, c_hat, a_rad
        self.Nq = len(kappa_lo)
        self.k_B = self.h_planck = self.mean_mass = 1.0
        self.gamma = 5.0 / 3.0
        self.closure, self.newton_tol, self.newton_maxit, self.outer_maxit = 0, 1e-13, 50, 50
        self.outer_tol, self.outer_stop, self.outer_rel_tol = 1e-13, 1, 1e-12
        self.ncells = state["rho"].shape[0]


def _state(rho, T, v, Eg, F, ks):
    n = rho.shape[0]
    return {"rho": rho.copy(), "mom": np.ascontiguousarray(rho[None, :] * v),
            "Egas": 1.5 * rho * T + 0.5 * rho * (v * v).sum(0),
            "Erad": np.ascontiguousarray(Eg), "Frad": np.ascontiguousarray(F),
            "kappa_scale": np.full(n, ks) if np.isscalar(ks) else ks.copy()}


def s8ii_case(n=300, seed=7):
    rng = np.random.default_rng(seed)
    edges = np.array([1e-3, 1e-2, 1e-1, 1.0, 10.0])
    rho = rng.uniform(0.5, 2.0, n)
    T = rng.uniform(0.7, 1.5, n)
    v = rng.normal(size=(3, n)) * 2.0
    Eg = np.array([1e-9, 1e-7, 1e-4, 5e-4])[:, None] * rng.uniform(0.5, 1.5, (4, n))
    F = rng.normal(size=(3, 4, n)) * 0.1 * 1e3 * Eg[None]
    st = _state(rho, T, v, Eg, F, 50.0)
    return GuardCase(edges, np.ones(4), np.array([2.0, 2.0, 0.0, 0.0]), st, dt=1.0, c=1e3, c_hat=1e3, a_rad=1e-3)


def s9_case(n=400, seed=11):
    rng = np.random.default_rng(seed)
    edges = np.array([0.4, 0.85, 2.0])
    rho = 10 ** rng.uniform(-3.2, -2.6, n)
    T = rng.uniform(8.0, 12.0, n)
    v = rng.normal(size=(3, n)) * 0.15
    Eg = np.array([1.2e5, 0.8e5])[:, None] * rng.uniform(0.5, 1.5, (2, n))
    d = rng.normal(size=(3, 2, n))
    d /= np.sqrt((d * d).sum(0))
    F = d * rng.uniform(0.5, 1.0, (2, n))[None] * 1e3 * Eg[None]
    st = _state(rho, T, v, Eg, F, 1.0)
    return GuardCase(edges, np.array([12.6, 3.0]), np.array([-2.2, -1.0]), st, dt=5e-3, c=1e3, c_hat=1e3, a_rad=1e-3)
