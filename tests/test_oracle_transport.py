"""Pins for the oracle's 1-D explicit transport and two-stage IMEX step (Eq. 33-36;
SURVEY 8(f) NEXT-3) -- CPU only.  The paper defers the spatial discretisation to Paper II, so the scheme is
reading S22 of DESIGN.md (piecewise constant, local Lax-Friedrichs with signal speed c_hat); what can be
pinned independently is pinned here: exact conservation, uniform states, the closed forms the scheme reduces
to for a beam (upwinding at c_hat) and for small isotropic perturbations, the literal stage equations of
Eq. 35-36, and the steady state of a uniform moving medium (section 4.2.1's setup without hydro).
"""
import math

import mpmath as mp
import numpy as np
import pytest

from test_oracle_update import _brute_force_residual, one_cell_state


def rad_state(E, F):
    Nq, nx = E.shape
    return {"Erad": np.array(E, dtype=np.float64, order="C", copy=True), "Frad": np.array(F, dtype=np.float64, order="C", copy=True)}


def copy(st):
    return {k: (None if v is None else v.copy()) for k, v in st.items()}


@pytest.mark.parametrize("lam,chat_over_c", [(1.0, 1.0), (0.4, 1.0), (0.7, 0.25)])
def test_beam_is_upwinded_at_the_reduced_speed_of_light(oracle_lib, lam, chat_over_c):
    """|F| = cE along +x (f = 1, chi = 1, P^xx = E): f(u) = (c_hat E, c c_hat E) and the Lax-Friedrichs flux with
    signal speed c_hat is exactly the upwind flux c_hat E_{i-1}: E_i^new = E_i - lam (E_i - E_{i-1})."""
    rng = np.random.default_rng(0)
    nx, Nq, c, dx = 37, 3, 3.0, 0.5
    chat = chat_over_c * c
    dt = lam * dx / chat
    E = rng.uniform(0.1, 2.0, (Nq, nx))
    F = np.zeros((3, Nq, nx))
    F[0] = c * E
    src, dst = rad_state(E, F), rad_state(E, F)
    oracle_lib.transport_add(src, dst, 0, dx, dt, c, chat, bc=0)
    ref = E - lam * (E - np.roll(E, 1, axis=1))
    assert np.allclose(dst["Erad"], ref, rtol=1e-14, atol=0)
    assert np.allclose(dst["Frad"][0], c * ref, rtol=1e-14, atol=0)
    assert np.all(dst["Frad"][1:] == 0.0)
    if lam == 1.0:      # CFL 1: the profile moves by exactly one cell
        assert np.allclose(dst["Erad"], np.roll(E, 1, axis=1), rtol=1e-13, atol=0)


def test_oblique_beam_closed_form(oracle_lib):
    """Beam at 60 degrees to x: n = (1/2, sqrt(3)/2, 0), P^xx = E/4, P^xy = E sqrt(3)/4.  Central flux plus the
    c_hat/2 dissipation: E_i^new = E_i - (lam/2) n_x (E_{i+1} - E_{i-1}) + (lam/2)(E_{i+1} - 2 E_i + E_{i-1})."""
    rng = np.random.default_rng(1)
    nx, c, dx, lam = 29, 2.0, 1.0, 0.6
    nxv, nyv = 0.5, math.sqrt(3.0) / 2
    E = rng.uniform(0.5, 1.5, (1, nx))
    F = np.zeros((3, 1, nx))
    F[0], F[1] = c * E * nxv, c * E * nyv
    src, dst = rad_state(E, F), rad_state(E, F)
    oracle_lib.transport_add(src, dst, 0, dx, lam * dx / c, c, c, bc=0)
    Ep, Em = np.roll(E, -1, axis=1), np.roll(E, 1, axis=1)
    lap = Ep - 2 * E + Em
    assert np.allclose(dst["Erad"], E - 0.5 * lam * nxv * (Ep - Em) + 0.5 * lam * lap, rtol=1e-13)
    assert np.allclose(dst["Frad"][0], c * (E * nxv - 0.5 * lam * nxv * nxv * (Ep - Em) + 0.5 * lam * nxv * lap), rtol=1e-13)
    assert np.allclose(dst["Frad"][1], c * (E * nyv - 0.5 * lam * nxv * nyv * (Ep - Em) + 0.5 * lam * nyv * lap), rtol=1e-13)


def test_isotropic_perturbation_eddington(oracle_lib):
    """Eddington closure, F = 0: only the dissipation acts on E, and F^x picks up -c c_hat dt (E_{i+1}-E_{i-1})/(6 dx)."""
    nx, c, chat, dx, dt = 32, 5.0, 2.0, 0.25, 0.03
    x = np.arange(nx)
    E = (1.0 + 0.1 * np.cos(2 * np.pi * 3 * x / nx))[None, :] * np.array([[1.0], [0.3]])
    F = np.zeros((3, 2, nx))
    src, dst = rad_state(E, F), rad_state(E, F)
    oracle_lib.transport_add(src, dst, 1, dx, dt, c, chat, bc=0)
    Ep, Em = np.roll(E, -1, axis=1), np.roll(E, 1, axis=1)
    assert np.allclose(dst["Erad"], E + 0.5 * chat * dt / dx * (Ep - 2 * E + Em), rtol=1e-14)
    assert np.allclose(dst["Frad"][0], -c * chat * dt / (6 * dx) * (Ep - Em), rtol=1e-12, atol=1e-16)


@pytest.mark.parametrize("closure", [0, 1])
def test_conservation_uniform_states_and_boundaries(oracle_lib, closure):
    rng = np.random.default_rng(2)
    nx, Nq, c, chat, dx, dt = 41, 4, 10.0, 4.0, 0.1, 0.01
    E = rng.uniform(0.1, 1.0, (Nq, nx))
    d = rng.normal(size=(3, Nq, nx))
    d /= np.sqrt((d * d).sum(0))
    F = d * rng.uniform(0, 1, (Nq, nx))[None] * c * E[None]
    src, dst = rad_state(E, F), rad_state(E, F)
    oracle_lib.transport_add(src, dst, closure, dx, dt, c, chat, bc=0)
    assert np.abs(dst["Erad"].sum(1) - E.sum(1)).max() < 1e-13 * E.sum(1).max()          # periodic: telescoping sum
    assert np.abs(dst["Frad"].sum(2) - F.sum(2)).max() < 1e-13 * np.abs(F).sum(2).max()
    assert np.abs(dst["Erad"] - E).max() > 1e-3                                            # (it did something)
    # a uniform state has no transport, with either boundary
    Eu, Fu = np.repeat(E[:, :1], nx, axis=1), np.repeat(F[:, :, :1], nx, axis=2)
    for bc in (0, 1):
        s, t = rad_state(Eu, Fu), rad_state(Eu, Fu)
        oracle_lib.transport_add(s, t, closure, dx, dt, c, chat, bc=bc)
        assert np.array_equal(t["Erad"], Eu) and np.array_equal(t["Frad"], Fu)
    # zero-gradient ends: the domain total changes by the difference of the two end fluxes f(u_0), f(u_{nx-1})
    s, t = rad_state(E, F), rad_state(E, F)
    oracle_lib.transport_add(s, t, closure, dx, dt, c, chat, bc=1)
    assert np.allclose(t["Erad"].sum(1) - E.sum(1), -(dt / dx) * (chat / c) * (F[0][:, -1] - F[0][:, 0]), rtol=1e-10, atol=1e-15)


def _whole_state(Nq, nx, rho, mom, Egas, E, F, ks=None):
    return {"rho": np.full(nx, rho), "mom": np.ascontiguousarray(np.repeat(np.asarray(mom, float).reshape(3, 1), nx, 1)),
            "Egas": np.full(nx, Egas), "Erad": np.ascontiguousarray(np.repeat(np.asarray(E, float).reshape(Nq, 1), nx, 1)),
            "Frad": np.ascontiguousarray(np.repeat(np.asarray(F, float).reshape(3, Nq, 1), nx, 2)),
            "kappa_scale": None if ks is None else np.full(nx, ks)}


def test_imex_stage_equations_with_the_brute_force_residual(oracle_lib):
    """Uniform medium (T(U) = 0): Eq. 35 is U^(n+1/2) = U^n + dt S(U^(n+1/2)) and Eq. 36 becomes
    U^(n+1) = U^n + (dt/2) S(U^(n+1/2)) + (dt/2) S(U^(n+1)) = (U^n + U^(n+1/2))/2 + (dt/2) S(U^(n+1)).
    Check both with the residuals of Eq. 37-40 typed from the paper in 30-digit arithmetic."""
    Nq, edges, alpha, kap = 2, [0.2, 2.0, 9.0], [0.0, -1.0], [30.0, 500.0]
    a_rad, c, chat, dt, rho, T0 = 1e-3, 1e3, 1e3, 4e-5, 0.6, 2.1      # c chi dt ~ 0.7 and 12: not yet at equilibrium
    mom0 = rho * 8e-3 * c * np.array([0.6, 0.0, 0.8])
    Egas0 = 1.5 * rho * T0 + 0.5 * (mom0 ** 2).sum() / rho
    E0 = np.array([2e-4, 9e-3])
    F0 = np.array([[0.1, 0.2], [0.0, 0.1], [-0.2, 0.05]]) * c * E0[None, :]
    m = oracle_lib.OracleModel(np.array(edges), np.array(kap), np.array(alpha), a_rad=a_rad)
    st = _whole_state(Nq, 3, rho, mom0, Egas0, E0, F0)
    half = copy(st)
    oracle_lib.source_update(m, half, dt, c, chat)                       # stage 1 by itself
    oracle_lib.imex_step_1d(m, st, 1.0, dt, c, chat, bc=0)
    M = mp.mpf

    def resid(U0, U1, dth):
        p = dict(Nq=Nq, c=M(c), chat=M(chat), dt=M(dth), rho=M(rho), Cv=M(1.5) * M(rho), a_rad=M(a_rad), h=M(1), kB=M(1),
                 edges=[M(e) for e in edges], alpha=[M(a) for a in alpha], chi_lo=[M(rho) * M(k) for k in kap],
                 E0=[M(U0["Erad"][g, 0]) for g in range(Nq)], F0=[[M(U0["Frad"][i, g, 0]) for i in range(3)] for g in range(Nq)],
                 Egas0=M(U0["Egas"][0]), mom0=[M(U0["mom"][i, 0]) for i in range(3)])
        x = [M(U1["Egas"][0])] + [M(U1["mom"][i, 0]) for i in range(3)] + [M(U1["Erad"][g, 0]) for g in range(Nq)]
        for g in range(Nq):
            x += [M(U1["Frad"][i, g, 0]) for i in range(3)]
        return [float(r) for r in _brute_force_residual(p, x)]

    Etot = Egas0 + E0.sum()
    scale = np.array([Etot] + [np.linalg.norm(mom0)] * 3 + [Etot] * Nq + [c * Etot] * (3 * Nq))
    un = _whole_state(Nq, 3, rho, mom0, Egas0, E0, F0)
    assert np.max(np.abs(resid(un, half, dt)) / scale) < 1e-12                        # Eq. 35
    mid = {k: (None if v is None else (0.5 * (un[k] + half[k]) if k in ("mom", "Egas", "Erad", "Frad") else v)) for k, v in un.items()}
    assert np.max(np.abs(resid(mid, st, dt / 2)) / scale) < 1e-12                     # Eq. 36
    # without transport the two stages collapse to backward Euler: V = (U^n + V)/2 + (dt/2) S(V) <=> V = U^n + dt S(V)
    for k in ("mom", "Egas", "Erad", "Frad"):
        assert np.max(np.abs(st[k] - half[k])) <= 1e-12 * np.max(np.abs(half[k]))
    assert abs(st["Erad"][1, 0] - E0[1]) > 0.1 * E0[1]                               # (the step moved the state)
    assert np.max(np.abs(resid(un, st, dt / 2)) / scale) > 1e-6                      # (and the residual can tell)


def test_imex_step_is_the_literal_eq36(oracle_lib):
    """Non-uniform state: the implementation's shortcut U** = (U^n + U^(n+1/2))/2 + (dt/2) T(U^(n+1/2)) against
    Eq. 36 composed literally from T(U^n), T(U^(n+1/2)) and dt S(U^(n+1/2)) = U^(n+1/2) - U*."""
    from paper_2407_18304_b200 import workloads as W
    from parity_util import oracle_model

    wl = W.workload(2, ncells=48)
    st0 = W.to_numpy(wl.make_state())
    m = oracle_model(oracle_lib, wl)
    dx, dt, bc = 1.0, 0.3 / wl.c, 0
    got = copy(st0)
    oracle_lib.imex_step_1d(m, got, dx, dt, wl.c, wl.c_hat, bc)
    ustar = copy(st0)
    oracle_lib.transport_add(st0, ustar, wl.closure, dx, dt, wl.c, wl.c_hat, bc)       # U* = U^n + dt T(U^n)
    half = copy(ustar)
    oracle_lib.source_update(m, half, dt, wl.c, wl.c_hat)                               # U^(n+1/2)
    lit = copy(st0)
    oracle_lib.transport_add(st0, lit, wl.closure, dx, 0.5 * dt, wl.c, wl.c_hat, bc)    # + dt T(U^n)/2
    oracle_lib.transport_add(half, lit, wl.closure, dx, 0.5 * dt, wl.c, wl.c_hat, bc)   # + dt T(U^(n+1/2))/2
    for k in ("mom", "Egas", "Erad", "Frad"):
        lit[k] = lit[k] + 0.5 * (half[k] - ustar[k])                                    # + dt S(U^(n+1/2))/2
    oracle_lib.source_update(m, lit, 0.5 * dt, wl.c, wl.c_hat)                          # U^(n+1)
    Etot = st0["Egas"] + st0["Erad"].sum(0)
    assert np.max(np.abs(got["Erad"] - lit["Erad"]) / Etot) < 1e-12
    assert np.max(np.abs(got["Egas"] - lit["Egas"]) / Etot) < 1e-12
    assert np.max(np.abs(got["Frad"] - lit["Frad"]) / (wl.c * Etot)) < 1e-12
    assert np.max(np.abs(got["mom"] - lit["mom"])) < 1e-12 * np.abs(st0["mom"]).max()
    assert np.abs(got["Erad"] - st0["Erad"]).max() > 1e-6 * st0["Erad"].max()


@pytest.mark.parametrize("Nq", [8, 16])
def test_doppler_setup_relaxes_to_the_moving_equilibrium(oracle_lib, Nq):
    """Section 4.2.1's medium (a_R = k_B = h = c = 1, rho = 1, C_V = 3/2, v = 0.001, chi_0 = 1e5, no radiation at
    t = 0, 64 periodic cells, groups over [1e-3, 1e2], radiation CFL 8) stepped with Eq. 35-36 to t = 1000 WITHOUT
    hydrodynamics.  Its steady state follows from G^0_g = 0, G^i_g = 0 (Eq. 21-22, Eq. 26) and the two conservation
    laws: E_g = B_g + v.F_g/c^2, sum_g F_g = (4/3) a_R T^4 v, so
        (3/2) T + v^2/2 + a_R T^4 (1 + (4/3) v^2) = 3/2 + v_0^2/2,   v (1 + (4/3) a_R T^4) = v_0.
    (The paper's printed 0.7680327097575 includes its hydrodynamic update and is not reproducible without it; the
    exact comoving value of Eq. 56 is 0.768032502191.)"""
    mp.mp.dps = 30
    v0 = mp.mpf("0.001")
    sol = mp.findroot(lambda T, v: [mp.mpf(1.5) * T + v * v / 2 + T ** 4 * (1 + mp.mpf(4) / 3 * v * v) - (mp.mpf(1.5) + v0 * v0 / 2),
                                    v * (1 + mp.mpf(4) / 3 * T ** 4) - v0], (mp.mpf("0.768"), v0))
    nx = 64
    edges = np.logspace(-3, 2, Nq + 1)
    m = oracle_lib.OracleModel(edges, np.full(Nq, 1e5), np.zeros(Nq), a_rad=1.0, newton_tol=1e-11)
    st = _whole_state(Nq, nx, 1.0, [1e-3, 0, 0], 1.5 + 0.5e-6, np.zeros(Nq), np.zeros((3, Nq)))
    dt = 8.0 * 1.0 / 1.0
    for _ in range(125):
        oracle_lib.imex_step_1d(m, st, 1.0, dt, 1.0, 1.0, bc=0)
    T = (st["Egas"] - 0.5 * (st["mom"] ** 2).sum(0) / st["rho"]) / 1.5
    assert np.ptp(T) == 0.0                                                   # stays uniform
    assert abs(T[0] - float(sol[0])) < 5e-11
    assert abs(st["mom"][0, 0] - float(sol[1])) < 5e-10            # (the groups start at x = 1.3e-3: Xi there is 3e-10)
    assert abs(T[0] - 0.768032502191) < 2e-8 and abs(T[0] - 0.768032502191) > 1e-9     # Eq. 56 up to O(v^2/c^2)
