"""Pins for the round-2 extensions of the oracle -- CPU only.

  S_g        the optional source term of Eq. 41 / 50 / the commit
  kind 1     opacities kappa_g (T/T_ref)^p evaluated at the trial temperature
  kind 2     edge opacities tabulated in T, alpha_g from Eq. 20, Eq. 62-63
  free slope Appendix A

Expected values: closed forms, the printed 3063.96 of Eq. 63, invariants, special cases that reduce to
the pinned round-1 path, and the 30-digit brute-force solve of the full implicit system typed from the
paper (tests/test_oracle_update.py) -- never the oracle's own algebra or the CUDA path.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

from paper_2407_18304_b200 import workloads as W

from parity_util import conservation_residual, oracle_model
from test_oracle_update import _brute_force_residual, mp_dY, one_cell_state

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _copy(st):
    return {k: (None if v is None else v.copy()) for k, v in st.items()}


def _brute(oracle_lib, m, st, p, Nq, scale, rtol=1e-11, atol=1e-13):
    x0 = [mp.mpf(st["Egas"][0])] + [mp.mpf(st["mom"][i, 0]) for i in range(3)] + [mp.mpf(st["Erad"][g, 0]) for g in range(Nq)]
    for g in range(Nq):
        x0 += [mp.mpf(st["Frad"][i, g, 0]) for i in range(3)]
    sol = mp.findroot(lambda *x: _brute_force_residual(p, list(x)), x0, tol=1e-40, maxsteps=40)
    sol = [sol[i] for i in range(len(x0))]
    assert max(abs(r) for r in _brute_force_residual(p, sol)) < mp.mpf(10) ** -22
    for gv, rv, sc in zip(x0, sol, scale):
        assert abs(float(gv) - float(rv)) <= rtol * abs(float(rv)) + atol * sc, (float(gv), float(rv))


def _case(seed=0):
    Nq, edges, alpha, kap = 3, [0.05, 0.6, 3.0, 20.0], [-2.0, 1.0, -3.5], [4.0, 0.3, 2.0]
    a_rad, c, chat, dt, rho, T0, beta = 1e-3, 1e3, 2e2, 2e-3, 1.7, 1.3, 3e-3
    rng = np.random.default_rng(seed)
    vdir = rng.normal(size=3)
    vdir /= np.linalg.norm(vdir)
    mom0 = rho * beta * c * vdir
    Egas0 = 1.5 * rho * T0 + 0.5 * (mom0 ** 2).sum() / rho
    E0 = np.array([float(a_rad * (0.8 * T0) ** 4 * mp_dY(edges[g] / (0.8 * T0), edges[g + 1] / (0.8 * T0))) for g in range(Nq)])
    F0 = np.array([0.4 * c * E0[g] * (lambda d: d / np.linalg.norm(d))(rng.normal(size=3)) for g in range(Nq)])
    M = mp.mpf
    p = dict(Nq=Nq, c=M(c), chat=M(chat), dt=M(dt), rho=M(rho), Cv=M(1.5) * M(rho), a_rad=M(a_rad), h=M(1), kB=M(1),
             edges=[M(e) for e in edges], alpha=[M(a) for a in alpha], chi_lo=[M(rho) * M(k) for k in kap],
             E0=[M(e) for e in E0], F0=[[M(f) for f in F0[g]] for g in range(Nq)], Egas0=M(Egas0), mom0=[M(t) for t in mom0])
    scale = [Egas0 + E0.sum()] + [np.linalg.norm(mom0)] * 3 + [Egas0 + E0.sum()] * Nq + [c * (Egas0 + E0.sum())] * (3 * Nq)
    return dict(Nq=Nq, edges=np.array(edges), alpha=np.array(alpha), kap=np.array(kap), a_rad=a_rad, c=c, chat=chat, dt=dt,
                rho=rho, mom0=mom0, Egas0=Egas0, E0=E0, F0=F0, p=p, scale=scale)


# ---------------------------------------------------------------------------
# S_g
# ---------------------------------------------------------------------------
def test_source_term_matches_brute_force(oracle_lib):
    k = _case()
    S = np.array([0.3, 1.5, 0.05]) * k["E0"]
    m = oracle_lib.OracleModel(k["edges"], k["kap"], k["alpha"], a_rad=k["a_rad"])
    st = one_cell_state(k["Nq"], k["rho"], k["mom0"], k["Egas0"], k["E0"], k["F0"].T.copy())
    st["Srad"] = S.reshape(-1, 1).copy()
    stats = oracle_lib.source_update(m, st, k["dt"], k["c"], k["chat"])
    assert stats["n_outer_unconverged"] == 0 and stats["n_newton_unconverged"] == 0
    p = dict(k["p"], S=[mp.mpf(s) for s in S])
    _brute(oracle_lib, m, st, p, k["Nq"], k["scale"])
    # the source really enters: without it the answer differs
    st2 = one_cell_state(k["Nq"], k["rho"], k["mom0"], k["Egas0"], k["E0"], k["F0"].T.copy())
    oracle_lib.source_update(m, st2, k["dt"], k["c"], k["chat"])
    assert np.abs(st2["Erad"] - st["Erad"]).max() > 0.01 * st["Erad"].max()


@pytest.mark.parametrize("idx,n", [(2, 200), (3, 150), (4, 120)])
def test_source_term_conservation_and_special_cases(oracle_lib, idx, n):
    """E_gas + (c/c_hat) sum (E_g - S_g) and the momentum are conserved to round-off for ANY Newton tolerance
    (the commit adds R_g + S_g to E_g and takes (c/c_hat) sum R_g from the gas); S = 0 is
    bit-identical to no source; and (E^t, S) gives the same answer as (E^t + S, 0) up to rounding order
    (Eq. 41, 50 and the commit contain E_g^t and S_g only through their sum)."""
    wl = W.workload(idx, ncells=n)
    st0 = W.to_numpy(wl.make_state())
    rng = np.random.default_rng(idx)
    S = st0["Erad"] * rng.uniform(0.0, 2.0, st0["Erad"].shape)
    for tol in (1e-13, 1e-3):
        m = oracle_model(oracle_lib, wl, newton_tol=tol)
        a = _copy(st0)
        a["Srad"] = S.copy()
        oracle_lib.source_update(m, a, wl.dt, wl.c, wl.c_hat)
        dE = (a["Egas"] + (wl.c / wl.c_hat) * (a["Erad"] - S).sum(0)) - (st0["Egas"] + (wl.c / wl.c_hat) * st0["Erad"].sum(0))
        scale = np.abs(st0["Egas"]) + (wl.c / wl.c_hat) * (np.abs(st0["Erad"]) + S).sum(0)
        assert np.max(np.abs(dE) / scale) <= 1e-13
        _, rP = conservation_residual(st0, a, wl.c, wl.c_hat)
        assert rP <= 1e-13
    m = oracle_model(oracle_lib, wl)
    z, none = _copy(st0), _copy(st0)
    z["Srad"] = np.zeros_like(S)
    oracle_lib.source_update(m, z, wl.dt, wl.c, wl.c_hat)
    oracle_lib.source_update(m, none, wl.dt, wl.c, wl.c_hat)
    for key in ("mom", "Egas", "Erad", "Frad"):
        assert np.array_equal(z[key], none[key]), key
    a, b = _copy(st0), _copy(st0)
    a["Srad"] = S.copy()
    b["Erad"] = st0["Erad"] + S
    oracle_lib.source_update(m, a, wl.dt, wl.c, wl.c_hat)
    oracle_lib.source_update(m, b, wl.dt, wl.c, wl.c_hat)
    Etot = st0["Egas"] + (st0["Erad"] + S).sum(0)
    assert np.max(np.abs(a["Erad"] - b["Erad"]) / Etot) < 1e-13
    assert np.max(np.abs(a["Egas"] - b["Egas"]) / Etot) < 1e-13


def test_source_term_static_relaxation_quartic(oracle_lib):
    """dt -> infinity, static gas, groups covering [0, inf): the cell relaxes to a_R T^4 + C_v T =
    E_gas^t + sum (E_g^t + S_g) with E_g = B_g(T) (north_star's quartic pin, now with sources)."""
    wl = W.workload(1, ncells=50)
    st0 = W.to_numpy(wl.make_state())
    S = 0.5 * st0["Erad"][::-1].copy()
    st = _copy(st0)
    st["Srad"] = S
    oracle_lib.source_update(oracle_model(oracle_lib, wl), st, 1e13, wl.c, wl.c_hat)   # 1/(c chi dt) ~ 1e-13
    Cv = 1.5 * st0["rho"]
    T = st["Egas"] / Cv
    total = st0["Egas"] + st0["Erad"].sum(0) + S.sum(0)
    assert np.max(np.abs(wl.a_rad * T ** 4 + Cv * T - total) / total) < 1e-12
    for g in range(wl.Nq):
        x = wl.edges / T[0]
        ref = wl.a_rad * T[0] ** 4 * float(mp_dY(x[g], x[g + 1] if np.isfinite(x[g + 1]) else mp.inf))
        assert abs(st["Erad"][g, 0] - ref) < 1e-9 * total[0]


# ---------------------------------------------------------------------------
# opacity kind 1: kappa_g (T/T_ref)^p at the trial temperature
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("pT", [1.5, -3.5])
def test_temperature_powerlaw_opacity_matches_brute_force(oracle_lib, pT):
    k = _case(1)
    m = oracle_lib.OracleModel(k["edges"], k["kap"], k["alpha"], a_rad=k["a_rad"], opacity_kind=1, T_ref=0.9, p_T=pT)
    st = one_cell_state(k["Nq"], k["rho"], k["mom0"], k["Egas0"], k["E0"], k["F0"].T.copy())
    stats = oracle_lib.source_update(m, st, k["dt"], k["c"], k["chat"])
    assert stats["n_outer_unconverged"] == 0 and stats["n_newton_unconverged"] == 0
    p = dict(k["p"], pT=mp.mpf(pT), Tref=mp.mpf("0.9"))
    _brute(oracle_lib, m, st, p, k["Nq"], k["scale"])
    st2 = one_cell_state(k["Nq"], k["rho"], k["mom0"], k["Egas0"], k["E0"], k["F0"].T.copy())
    oracle_lib.source_update(oracle_lib.OracleModel(k["edges"], k["kap"], k["alpha"], a_rad=k["a_rad"]), st2, k["dt"], k["c"], k["chat"])
    assert np.abs(st2["Erad"] - st["Erad"]).max() > 1e-3 * st["Erad"].max()


def test_temperature_powerlaw_p0_is_the_table(oracle_lib):
    wl = W.workload(4, ncells=80)
    st0 = W.to_numpy(wl.make_state())
    a, b = _copy(st0), _copy(st0)
    oracle_lib.source_update(oracle_model(oracle_lib, wl), a, wl.dt, wl.c, wl.c_hat)
    oracle_lib.source_update(oracle_model(oracle_lib, wl, opacity_kind=1, T_ref=3.0, p_T=0.0), b, wl.dt, wl.c, wl.c_hat)
    for key in ("mom", "Egas", "Erad", "Frad"):
        assert np.array_equal(a[key], b[key]), key


def test_marshak_c_opacity_scalar_balance_by_bisection(oracle_lib):
    """chi_g' = chi_g (T/T_0)^{3/2} with PC groups, static gas: the converged state satisfies
    E_g = (E_g^t + tau_g(T) B_g(T))/(1 + tau_g(T)), tau_g = c_hat dt chi_g(T), and T solves the scalar energy
    balance C_v T + sum_g E_g(T) = E_gas^t + sum_g E_g^t, found here by bisection in 30-digit arithmetic."""
    mp.mp.dps = 30
    edges = np.array([0.0, 0.7, 2.5, 9.0, np.inf])
    kap = np.array([1.0, 0.5, 0.25, 0.01])
    a_rad, c, rho, Tg, dt, T0 = 1.0, 1.0, 1.3, 1.6, 0.8, 0.5
    E0 = np.array([0.05, 0.2, 0.1, 0.01])
    m = oracle_lib.OracleModel(edges, kap, np.zeros(4), a_rad=a_rad, opacity_kind=1, T_ref=T0, p_T=1.5)
    st = one_cell_state(4, rho, [0, 0, 0], 1.5 * rho * Tg, E0, np.zeros((3, 4)))
    s = oracle_lib.source_update(m, st, dt, c, c)
    assert s["n_newton_unconverged"] == 0
    Cv, total = mp.mpf(1.5) * mp.mpf(rho), mp.mpf(1.5 * rho * Tg) + sum(mp.mpf(e) for e in E0)

    def Eg(T):
        out = []
        for g in range(4):
            tau = mp.mpf(c) * mp.mpf(dt) * mp.mpf(rho) * mp.mpf(kap[g]) * (T / mp.mpf(T0)) ** mp.mpf(1.5)
            hi = mp.inf if not np.isfinite(edges[g + 1]) else mp.mpf(edges[g + 1]) / T
            Bt = mp.mpf(a_rad) * T ** 4 * mp_dY(mp.mpf(edges[g]) / T, hi if hi != mp.inf else mp.mpf(edges[g]) / T + 400)
            out.append((mp.mpf(E0[g]) + tau * Bt) / (1 + tau))
        return out

    lo, hi = mp.mpf("0.1"), mp.mpf(3)
    for _ in range(90):
        mid = (lo + hi) / 2
        lo, hi = (mid, hi) if Cv * mid + sum(Eg(mid)) < total else (lo, mid)
    Tb = (lo + hi) / 2
    assert abs(st["Egas"][0] / float(Cv) - float(Tb)) < 1e-12 * float(Tb)
    for g, ref in enumerate(Eg(Tb)):
        assert abs(st["Erad"][g, 0] - float(ref)) < 1e-11 * float(total)
    assert abs(float(Tb) - Tg) > 0.01


# ---------------------------------------------------------------------------
# opacity kind 2: edge values tabulated in T, alpha from Eq. 20
# ---------------------------------------------------------------------------
def test_edge_table_of_a_power_law_equals_the_power_law_models(oracle_lib):
    """kappa(nu, T) = K (T/T_ref)^p nu^s tabulated at the edges: ln kappa is linear in ln T (the interpolation is
    exact) and Eq. 20 returns alpha = s, so the update equals opacity kind 1 with kappa_lo = K nu_lo^s."""
    wl = W.workload(3, ncells=60)          # nu^-3 opacity, c_hat = 0.1 c
    st0 = W.to_numpy(wl.make_state())
    Tref, pT, NT = 1.7, -0.5, 9
    lnT = np.linspace(math.log(0.05), math.log(50.0), NT)
    lnk = -3.0 * np.log(wl.edges)[:, None] + pT * (lnT[None, :] - math.log(Tref))
    a, b = _copy(st0), _copy(st0)
    oracle_lib.source_update(oracle_model(oracle_lib, wl, opacity_kind=1, T_ref=Tref, p_T=pT), a, wl.dt, wl.c, wl.c_hat)
    oracle_lib.source_update(oracle_model(oracle_lib, wl, opacity_kind=2, lnk_edge=lnk, lnT0=lnT[0], dlnT=lnT[1] - lnT[0]),
                             b, wl.dt, wl.c, wl.c_hat)
    Etot = st0["Egas"] + st0["Erad"].sum(0)
    assert np.max(np.abs(a["Erad"] - b["Erad"]) / Etot) < 1e-12
    assert np.max(np.abs(a["Egas"] - b["Egas"]) / Etot) < 1e-12
    assert np.max(np.abs(a["Frad"] - b["Frad"]) / (wl.c * Etot)) < 1e-12


def _eq62_table(edges_hz, Tgrid):
    """ln chi_0/rho of Eq. 62 at the group edges and table temperatures, CGS, rho = 1."""
    kB, h = 1.380649e-16, 6.62607015e-27
    x = h * edges_hz[:, None] / (kB * Tgrid[None, :])
    return np.log(180.0) - 0.5 * np.log(Tgrid[None, :] / 1e7) - 3.0 * np.log(edges_hz[:, None] / 1e18) + np.log(-np.expm1(-x))


def eq63_setup(Nq):
    """One cell at T = 1e7 K without radiation, CGS units, Eq. 62 tabulated at Nq+1 log-spaced edges
    (x from 1e-6 to 45; T = 1e7 K is a table node).  Returns (model kwargs, state, dt, c, normalisation)."""
    kB, h, aR, c = 1.380649e-16, 6.62607015e-27, 7.565733e-15, 2.99792458e10
    T, rho, mu = 1e7, 1.0, 3.9e-24
    x_edges = np.logspace(-6, math.log10(45.0), Nq + 1)
    edges = x_edges * kB * T / h
    Tgrid = 1e7 * np.exp(np.linspace(-1.0, 1.0, 5))            # node 2 is exactly 1e7 K
    kw = dict(edges=edges, kappa_lo=np.ones(Nq), alpha=np.zeros(Nq), a_rad=aR, k_B=kB, h_planck=h, mean_mass=mu,
              gamma=5.0 / 3.0, opacity_kind=2, lnk_edge=_eq62_table(edges, Tgrid), lnT0=math.log(Tgrid[0]), dlnT=0.5)
    st = one_cell_state(Nq, rho, [0, 0, 0], 1.5 * rho * kB * T / mu, np.zeros(Nq), np.zeros((3, Nq)))
    dt = 1e-32
    return kw, st, dt, c, c * dt * aR * T ** 4


def test_eq63_planck_mean_through_source_update(oracle_lib):
    """for chi_0 of Eq. 62 the Planck mean is 3063.96 (T/1e7 K)^-3.5 cm^-1.  One optically
    thin update (c_hat dt chi << 1) of a cell with no radiation at T = 1e7 K: the emitted energy is
    sum_g E_g = c_hat dt a_R T^4 sum_g chi_B,g [Y(x_g+) - Y(x_g-)], so sum_g E_g / (c_hat dt a_R T^4) is the PPL
    estimate of the Planck mean (alpha from Eq. 20, fixed-slope means of Eq. 30).  It converges at second order
    in the group width, and its Richardson extrapolation from 64, 128 and 256 groups reproduces the printed
    value -- through source_update itself, in CGS (non-unit mgrhd_units)."""
    chiP_ref = float(open(os.path.join(GOLD, "eq63_mean_opacities.txt")).read().split()[0])
    est = {}
    for Nq in (64, 128, 256):
        kw, st, dt, c, norm = eq63_setup(Nq)
        s = oracle_lib.source_update(oracle_lib.OracleModel(**kw), st, dt, c, c)
        assert s["n_newton_unconverged"] == 0
        est[Nq] = st["Erad"].sum() / norm
    e = {k: v / chiP_ref - 1.0 for k, v in est.items()}
    assert 0.02 < e[64] < 0.05                                          # a finite-Nq estimate, not a restatement
    assert 3.8 < e[64] / e[128] < 4.3 and 3.8 < e[128] / e[256] < 4.3    # second order
    rich = (4.0 * est[256] - est[128]) / 3.0
    assert abs(rich / chiP_ref - 1.0) < 3e-5                            # 3063.96 is printed to 6 digits; x < 1e-6 is missing


def test_edge_table_interpolation_in_temperature(oracle_lib):
    """Between table nodes ln kappa is interpolated linearly in ln T and held at the end values outside the
    table (reading S19): one optically thin update at T* gives R_g = c_hat dt chi_B,g B_g with
    chi(T*) from the interpolation typed out here."""
    Nq, edges = 2, np.array([0.5, 2.0, 8.0])
    lnT = np.array([math.log(0.5), math.log(2.0)])
    lnk = np.array([[0.0, 1.0], [-1.0, 2.5], [0.5, 0.7]])
    for Tstar, w in ((1.0, 0.5), (0.2, 0.0), (5.0, 1.0)):
        m = oracle_lib.OracleModel(edges, np.ones(2), np.zeros(2), a_rad=1.0, opacity_kind=2, lnk_edge=lnk,
                                   lnT0=lnT[0], dlnT=lnT[1] - lnT[0])
        rho, dt, c = 2.0, 1e-14, 1.0
        st = one_cell_state(Nq, rho, [0, 0, 0], 1.5 * rho * Tstar, np.zeros(2), np.zeros((3, 2)))
        oracle_lib.source_update(m, st, dt, c, c)
        k = np.exp((1 - w) * lnk[:, 0] + w * lnk[:, 1])
        for g in range(2):
            al = math.log(k[g + 1] / k[g]) / math.log(edges[g + 1] / edges[g])                   # Eq. 20
            chiB = rho * (k[g + 1] - k[g]) / (al * math.log(edges[g + 1] / edges[g]))            # Eq. 30, alpha_Q = -1
            ref = c * dt * chiB * Tstar ** 4 * float(mp_dY(edges[g] / Tstar, edges[g + 1] / Tstar))
            assert abs(st["Erad"][g, 0] - ref) < 1e-12 * ref


# ---------------------------------------------------------------------------
# free-slope spectrum (Appendix A)
# ---------------------------------------------------------------------------
def test_free_slopes_closed_forms(oracle_lib):
    edges = np.logspace(-1, 1, 8)                                   # constant ratio r
    r = edges[1] / edges[0]
    for a in (-2.5, -1.0, 0.0, 1.7):
        # Q_nu = nu^a integrated exactly over each group: every interior slope is a (Eq. A1 with Qbar_g ~ nu_g-^a)
        Q = edges[:-1] ** (a + 1) * (math.log(r) if a == -1.0 else (r ** (a + 1) - 1) / (a + 1))
        al = oracle_lib.free_slopes(edges, Q)
        assert al[0] == -1.0 and al[-1] == -1.0                     # edge groups (Eq. A2)
        assert np.allclose(al[1:-1], a, rtol=0, atol=1e-13)
    # minmod: a local maximum gives 0; the smaller of two same-sign slopes wins
    Q = np.array([1.0, 2.0, 8.0, 2.0, 1.0, 0.5, 0.4]) * (edges[1:] - edges[:-1])
    al = oracle_lib.free_slopes(edges, Q)
    ln = math.log(r)
    assert al[2] == 0.0                                             # s = +ln4/ln r, -ln4/ln r
    assert abs(al[1] - math.log(2.0) / ln) < 1e-13                  # min(ln2, ln4)/ln r
    assert abs(al[4] - (-math.log(2.0) / ln)) < 1e-13               # both -ln2/ln r
    assert abs(al[5] - math.log(0.8) / ln) < 1e-13                  # min(|ln .5|, |ln .8|) keeps the sign
    # a zero or negative neighbour has no logarithm: fixed-slope value (reading S21)
    Q[3] = 0.0
    al = oracle_lib.free_slopes(edges, Q)
    assert al[2] == al[3] == al[4] == -1.0 and al[1] != -1.0
    # fewer than three groups: every group is an edge group
    assert list(oracle_lib.free_slopes(edges[:3], Q[:2])) == [-1.0, -1.0]


def test_free_slope_is_irrelevant_for_piecewise_constant_opacity(oracle_lib):
    """alpha_Q matters only when alpha_chi != 0: with PC opacities the free-slope update is
    bit-identical to the fixed-slope one."""
    wl = W.workload(4, ncells=60)
    wl.alpha = np.zeros_like(wl.alpha)
    st0 = W.to_numpy(wl.make_state())
    a, b = _copy(st0), _copy(st0)
    oracle_lib.source_update(oracle_model(oracle_lib, wl), a, wl.dt, wl.c, wl.c_hat)
    oracle_lib.source_update(oracle_model(oracle_lib, wl, spectrum=1), b, wl.dt, wl.c, wl.c_hat)
    for key in ("mom", "Egas", "Erad", "Frad"):
        assert np.array_equal(a[key], b[key]), key


def test_free_slope_update_matches_brute_force(oracle_lib):
    """Five groups so that three are interior; the root of Eq. 37-40 with alpha_B, alpha_E from Eq. A1-A2 at the
    NEW state (30-digit Newton on the full 24-unknown system) is what the oracle's iteration converges to."""
    Nq = 5
    edges = np.array([0.1, 0.4, 1.2, 3.5, 9.0, 25.0])
    alpha = np.array([-1.5, -2.5, 0.8, -3.0, -2.0])
    kap = np.array([3.0, 1.0, 0.2, 0.6, 0.05])
    a_rad, c, chat, dt, rho, T0, beta = 1e-3, 1e3, 5e2, 3e-3, 1.2, 1.1, 2e-3
    rng = np.random.default_rng(3)
    vdir = rng.normal(size=3)
    vdir /= np.linalg.norm(vdir)
    mom0 = rho * beta * c * vdir
    Egas0 = 1.5 * rho * T0 + 0.5 * (mom0 ** 2).sum() / rho
    E0 = np.array([float(a_rad * (1.4 * T0) ** 4 * mp_dY(edges[g] / (1.4 * T0), edges[g + 1] / (1.4 * T0))) for g in range(Nq)])
    E0 *= np.array([1.0, 0.6, 1.5, 0.8, 2.0])
    F0 = np.array([0.3 * c * E0[g] * (lambda d: d / np.linalg.norm(d))(rng.normal(size=3)) for g in range(Nq)])
    m = oracle_lib.OracleModel(edges, kap, alpha, a_rad=a_rad, spectrum=1)
    st = one_cell_state(Nq, rho, mom0, Egas0, E0, F0.T.copy())
    stats = oracle_lib.source_update(m, st, dt, c, chat)
    assert stats["n_outer_unconverged"] == 0 and stats["n_newton_unconverged"] == 0
    M = mp.mpf
    p = dict(Nq=Nq, c=M(c), chat=M(chat), dt=M(dt), rho=M(rho), Cv=M(1.5) * M(rho), a_rad=M(a_rad), h=M(1), kB=M(1),
             edges=[M(float(e)) for e in edges], alpha=[M(float(a)) for a in alpha], chi_lo=[M(rho) * M(float(k)) for k in kap],
             E0=[M(e) for e in E0], F0=[[M(f) for f in F0[g]] for g in range(Nq)], Egas0=M(Egas0),
             mom0=[M(t) for t in mom0], free=True)
    Etot = Egas0 + E0.sum()
    scale = [Etot] + [np.linalg.norm(mom0)] * 3 + [Etot] * Nq + [c * Etot] * (3 * Nq)
    _brute(oracle_lib, m, st, p, Nq, scale, rtol=1e-10, atol=1e-12)
    # the free slopes are really different from -1 here, and the answer differs from the fixed-slope one
    fixed = one_cell_state(Nq, rho, mom0, Egas0, E0, F0.T.copy())
    oracle_lib.source_update(oracle_lib.OracleModel(edges, kap, alpha, a_rad=a_rad), fixed, dt, c, chat)
    assert np.abs(fixed["Erad"] - st["Erad"]).max() > 1e-4 * st["Erad"].max()
    sl = oracle_lib.free_slopes(edges, st["Erad"][:, 0])
    assert np.abs(sl[1:-1] + 1.0).max() > 0.1


def test_free_slope_conserves_energy_and_momentum(oracle_lib):
    wl = W.workload(4, ncells=150)
    st0 = W.to_numpy(wl.make_state())
    st = _copy(st0)
    s = oracle_lib.source_update(oracle_model(oracle_lib, wl, spectrum=1, newton_tol=1e-6), st, wl.dt, wl.c, wl.c_hat)
    rE, rP = conservation_residual(st0, st, wl.c, wl.c_hat)
    assert rE <= 1e-13 and rP <= 1e-13
    assert s["n_newton_unconverged"] == 0


# ---------------------------------------------------------------------------
# outer_mode 1 ("variant L"): Eq. 51-52 solved implicitly in the velocity -- same root, converges at large radiation inertia
# ---------------------------------------------------------------------------
def test_variant_L_converges_to_the_brute_force_root_where_the_lagged_iteration_diverges(oracle_lib):
    """A radiation-dominated cell in literal units (a_R = c = 1): q = (4/3) sum E_g/(rho c c_hat) ~ 50, far outside
    the premise q << 1 of the lagged-velocity outer loop, which does not converge here.  The implicit-in-v
    outer stage reaches the root of the full system (30-digit solve, same residual function as every other case)."""
    Nq, edges, alpha, kap = 3, [0.05, 0.6, 3.0, 20.0], [-2.0, 1.0, -3.5], [4.0, 0.3, 2.0]
    a_rad, c, chat, dt, rho, T0 = 1.0, 1.0, 1.0, 0.7, 0.05, 1.3
    mom0 = rho * np.array([0.02, -0.01, 0.03])
    Egas0 = 1.5 * rho * T0 + 0.5 * (mom0 ** 2).sum() / rho
    E0 = np.array([float(a_rad * (1.1 * T0) ** 4 * mp_dY(edges[g] / (1.1 * T0), edges[g + 1] / (1.1 * T0))) for g in range(Nq)])
    F0 = np.array([[0.2, -0.1, 0.05], [0.1, 0.3, -0.2], [-0.05, 0.02, 0.1]]) * c * E0[:, None]
    q = 4.0 / 3.0 * E0.sum() / (rho * c * chat)
    assert q > 30
    lag = one_cell_state(Nq, rho, mom0, Egas0, E0, F0.T.copy())
    s0 = oracle_lib.source_update(oracle_lib.OracleModel(np.array(edges), np.array(kap), np.array(alpha), a_rad=a_rad), lag, dt, c, chat)
    assert s0["n_outer_unconverged"] + s0["n_T_nonpositive_steps"] + s0["n_newton_unconverged"] > 0 or not np.isfinite(lag["Erad"]).all()
    m = oracle_lib.OracleModel(np.array(edges), np.array(kap), np.array(alpha), a_rad=a_rad, outer_mode=1)
    st = one_cell_state(Nq, rho, mom0, Egas0, E0, F0.T.copy())
    s1 = oracle_lib.source_update(m, st, dt, c, chat)
    assert s1["n_outer_unconverged"] == 0 and s1["n_newton_unconverged"] == 0 and s1["n_T_nonpositive_steps"] == 0
    assert 2 <= s1["outer_trips_total"] <= 25
    M = mp.mpf
    p = dict(Nq=Nq, c=M(c), chat=M(chat), dt=M(dt), rho=M(rho), Cv=M(1.5) * M(rho), a_rad=M(a_rad), h=M(1), kB=M(1),
             edges=[M(e) for e in edges], alpha=[M(a) for a in alpha], chi_lo=[M(rho) * M(k) for k in kap],
             E0=[M(e) for e in E0], F0=[[M(f) for f in F0[g]] for g in range(Nq)], Egas0=M(Egas0), mom0=[M(t) for t in mom0])
    Etot = Egas0 + E0.sum()
    scale = [Etot] + [np.linalg.norm(mom0) + np.abs(F0).sum() / (c * chat)] * 3 + [Etot] * Nq + [c * Etot] * (3 * Nq)
    _brute(oracle_lib, m, st, p, Nq, scale, rtol=1e-10, atol=1e-12)
    assert abs(st["Egas"][0] - Egas0) > 1e-3 * Egas0


@pytest.mark.parametrize("idx,n", [(2, 150), (4, 100)])
def test_variant_L_equals_the_lagged_iteration_at_small_radiation_inertia(oracle_lib, idx, n):
    """Both outer stages converge to the same state (the root of Eq. 37-40); on the BASELINE workloads (q <= 3e-3) they
    agree to the parity tolerance, and the implicit one needs no more trips."""
    wl = W.workload(idx, ncells=n)
    st0 = W.to_numpy(wl.make_state())
    a, b = _copy(st0), _copy(st0)
    sa = oracle_lib.source_update(oracle_model(oracle_lib, wl), a, wl.dt, wl.c, wl.c_hat)
    sb = oracle_lib.source_update(oracle_model(oracle_lib, wl, outer_mode=1), b, wl.dt, wl.c, wl.c_hat)
    Etot = st0["Egas"] + st0["Erad"].sum(0)
    assert np.max(np.abs(a["Erad"] - b["Erad"]) / Etot) < 1e-12
    assert np.max(np.abs(a["Egas"] - b["Egas"]) / Etot) < 1e-12
    assert np.max(np.abs(a["Frad"] - b["Frad"]) / (1e-10 * np.abs(a["Frad"]) + 1e-12 * wl.c * Etot)) < 1.0
    assert np.max(np.abs(a["mom"] - b["mom"]) / np.abs(a["mom"]).max()) < 1e-10
    assert sb["outer_trips_total"] <= sa["outer_trips_total"] and sb["n_outer_unconverged"] == 0


def test_variant_L_on_literal_units_conserves_and_converges(oracle_lib):
    """SURVEY 8(d) "variant L": config 2 with the literal units a_R = c = 1 (q up to several hundred): every cell converges
    in a handful of trips and energy and momentum are conserved to round-off; the lagged iteration fails on most cells."""
    wl = W.workload(2, ncells=300)
    wl.a_rad, wl.c, wl.c_hat, wl.dt = 1.0, 1.0, 1.0, 1.0
    st0 = W.to_numpy(wl.make_state())
    st = _copy(st0)
    s = oracle_lib.source_update(oracle_model(oracle_lib, wl, outer_mode=1), st, wl.dt, wl.c, wl.c_hat)
    assert s["n_outer_unconverged"] == 0 and s["n_newton_unconverged"] == 0 and s["n_T_nonpositive_steps"] == 0
    assert max(i for i, cnt in enumerate(s["outer_hist"]) if cnt) <= 20
    rE, rP = conservation_residual(st0, st, wl.c, wl.c_hat)
    assert rE <= 1e-13 and rP <= 1e-13
    lag = _copy(st0)
    s0 = oracle_lib.source_update(oracle_model(oracle_lib, wl), lag, wl.dt, wl.c, wl.c_hat)
    assert s0["n_outer_unconverged"] + s0["n_T_nonpositive_steps"] > 50
