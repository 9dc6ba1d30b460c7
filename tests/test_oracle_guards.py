"""Pins for the guard branches of the oracle (readings S8, S9) -- CPU only.

S8(i)  the Wien-limit fallback chi_F = chi_{g-} is continuous with Eq. 27 across its 1e-280 threshold:
       Eq. 27 evaluated in 60-digit arithmetic on both sides of the threshold differs from chi_{g-} by the
       O(1/x) the Wien expansion of Eq. 27 predicts.
S8(ii) a cell in which 1 + c_hat chi_F dt <= 0 fires: the update equals the 30-digit brute-force solve of
       Eq. 37-40 with chi_F := chi_E in exactly those groups.
S9     the T <= 0 guard at the start of a later outer trip: the cell keeps the previous trip's result, which
       is the exact one-trip update (conservation to round-off, counters).
"""
import math

import mpmath as mp
import numpy as np

from guard_cases import s8ii_case, s9_case
from parity_util import conservation_residual, oracle_model
from test_oracle_update import _brute_force_residual, one_cell_state


def _mp_group(xlo, xhi, dps=60):
    """(dY, Xi_lo, Xi_hi) of a Wien-tail group from the defining series, in `dps`-digit arithmetic."""
    with mp.workdps(dps):
        C = 15 / mp.pi ** 4
        Z = lambda x: C * mp.nsum(lambda n: mp.exp(-n * x) * (x ** 3 / n + 3 * x ** 2 / n ** 2 + 6 * x / n ** 3 + 6 / n ** 4),  # noqa: E731
                                  [1, mp.inf])
        Xi = lambda x: C * x ** 4 / mp.expm1(x)  # noqa: E731
        xlo, xhi = mp.mpf(xlo), mp.mpf(xhi)
        return Z(xlo) - Z(xhi), Xi(xlo), Xi(xhi)


def test_s8i_wien_fallback_is_continuous_with_eq27(oracle_lib):
    r, alpha, chi_lo = 1.3, -1.7, 2.5
    lnr = math.log(r)
    chi_hi = chi_lo * r ** alpha
    chiB = chiE = oracle_lib.chi_mean(chi_lo, lnr, alpha, -1.0)
    # walk up the Wien tail until the oracle's guard fires (a_R T^4 = 1, so the threshold is den < 1e-280)
    last_ok = first_guard = None
    for x in np.arange(600.0, 700.0, 0.25):
        Bt = oracle_lib.planck_dY(x, r * x)
        Xl, Xh = oracle_lib.planck_Xi(x), oracle_lib.planck_Xi(r * x)
        val, guard = oracle_lib.chi_flux(chiB, chiE, alpha, chi_lo, Bt, Xh - Xl, chi_hi * Xh - chi_lo * Xl, 1.0)
        if guard:
            first_guard = (x, val)
            break
        last_ok = (x, val, Bt, Xl, Xh)
    assert last_ok is not None and first_guard is not None and first_guard[1] == chi_lo
    # Wien expansion of Eq. 27: chi_F = chi_- [1 + ((chiB/chi_-)(4 + alpha) - 4)/x + O(1/x^2)]
    slope = (chiB / chi_lo) * (4 + alpha) - 4
    for x in (last_ok[0], first_guard[0]):
        dY, Xl, Xh = _mp_group(x, r * x)
        with mp.workdps(60):
            num = (mp.mpf(chiB) + mp.mpf(chiE) / 3) * dY + (mp.mpf(alpha) * chiE * dY - (chi_hi * Xh - chi_lo * Xl)) / 3
            den = mp.mpf(4) / 3 * dY - (Xh - Xl) / 3
            exact = num / den                                    # Eq. 27, no guard
            assert abs(exact / chi_lo - 1 - slope / x) < 30 / x ** 2
            # the value the oracle returns on either side of the threshold is within that O(1/x) of Eq. 27
            ret = last_ok[1] if x == last_ok[0] else first_guard[1]
            assert abs(ret - exact) <= (abs(slope) / x + 30 / x ** 2) * chi_lo
    # just below the threshold the double-precision Eq. 27 still agrees with the 60-digit value
    dY, Xl, Xh = _mp_group(last_ok[0], r * last_ok[0])
    with mp.workdps(60):
        exact = ((mp.mpf(chiB) + mp.mpf(chiE) / 3) * dY + (mp.mpf(alpha) * chiE * dY - (chi_hi * Xh - chi_lo * Xl)) / 3) \
            / (mp.mpf(4) / 3 * dY - (Xh - Xl) / 3)
    assert abs(last_ok[1] - float(exact)) < 1e-11 * chi_lo


def test_s8ii_fallback_matches_brute_force_with_chiF_replaced(oracle_lib):
    """Two groups; the first (r = 10, alpha = 2, Rayleigh-Jeans range) has chi_F < 0 with c_hat chi_F dt < -1."""
    Nq, edges, alpha, kap = 2, [1e-2, 1e-1, 1.0], [2.0, 0.0], [1.0, 1.0]
    a_rad, c, chat, dt, rho, T0, ks = 1e-3, 1e3, 1e3, 1.0, 1.3, 1.1, 50.0
    mom0 = rho * np.array([1.0, -2.0, 0.5])
    Egas0 = 1.5 * rho * T0 + 0.5 * (mom0 ** 2).sum() / rho
    E0 = np.array([1e-7, 1e-4])
    F0 = np.array([[30.0, -10.0, 5.0], [-20.0, 40.0, 10.0]]) * E0[:, None]
    m = oracle_lib.OracleModel(np.array(edges), np.array(kap), np.array(alpha), a_rad=a_rad)
    st = one_cell_state(Nq, rho, mom0, Egas0, E0, F0.T.copy(), kscale=ks)
    stats = oracle_lib.source_update(m, st, dt, c, chat)
    assert stats["n_denominator_nonpositive"] == 1
    assert stats["n_outer_unconverged"] == 0 and stats["n_newton_unconverged"] == 0
    M = mp.mpf
    p = dict(Nq=Nq, c=M(c), chat=M(chat), dt=M(dt), rho=M(rho), Cv=M(1.5) * M(rho), a_rad=M(a_rad), h=M(1), kB=M(1),
             edges=[M(e) for e in edges], alpha=[M(a) for a in alpha], chi_lo=[M(rho) * M(ks) * M(k) for k in kap],
             E0=[M(e) for e in E0], F0=[[M(f) for f in F0[g]] for g in range(Nq)], Egas0=M(Egas0),
             mom0=[M(t) for t in mom0], chiF_is_chiE=(0,))
    x0 = [M(st["Egas"][0])] + [M(st["mom"][i, 0]) for i in range(3)] + [M(st["Erad"][g, 0]) for g in range(Nq)]
    for g in range(Nq):
        x0 += [M(st["Frad"][i, g, 0]) for i in range(3)]
    sol = mp.findroot(lambda *x: _brute_force_residual(p, list(x)), x0, tol=1e-40, maxsteps=30)
    sol = [sol[i] for i in range(len(x0))]
    assert max(abs(r) for r in _brute_force_residual(p, sol)) < mp.mpf(10) ** -22
    Etot = Egas0 + E0.sum()
    scale = [Etot] + [np.linalg.norm(mom0)] * 3 + [Etot] * Nq + [c * Etot] * (3 * Nq)
    for gv, rv, sc in zip(x0, sol, scale):
        assert abs(float(gv) - float(rv)) <= 1e-11 * abs(float(rv)) + 1e-13 * sc
    assert abs(st["Egas"][0] - Egas0) > 1e-9 * Egas0


def test_s8ii_many_cells_counters_and_conservation(oracle_lib):
    gc = s8ii_case()
    st0 = {k: v.copy() for k, v in gc.state.items()}
    st = {k: v.copy() for k, v in gc.state.items()}
    s = oracle_lib.source_update(oracle_model(oracle_lib, gc), st, gc.dt, gc.c, gc.c_hat)
    assert s["n_denominator_nonpositive"] == 2 * gc.ncells       # the two rising-opacity groups of every cell
    assert s["n_newton_unconverged"] == s["n_outer_unconverged"] == s["n_T_nonpositive_steps"] == 0
    rE, rP = conservation_residual(st0, st, gc.c, gc.c_hat)
    assert rE <= 1e-13 and rP <= 1e-13


def test_s9_invalid_state_after_first_trip_keeps_that_trip(oracle_lib):
    """T <= 0 at the start of outer trip k+1 (kinetic energy of the updated momentum exceeds the gas energy):
    the iteration stops there and the cell holds the result of trip k -- still an exact (conservative) update."""
    gc = s9_case()
    st0 = {k: v.copy() for k, v in gc.state.items()}
    st = {k: v.copy() for k, v in gc.state.items()}
    s = oracle_lib.source_update(oracle_model(oracle_lib, gc), st, gc.dt, gc.c, gc.c_hat)
    assert s["n_T_nonpositive_steps"] == gc.ncells and s["n_outer_unconverged"] == 0
    assert s["outer_trips_total"] >= gc.ncells and s["outer_hist"][0] == 0
    rE, rP = conservation_residual(st0, st, gc.c, gc.c_hat)
    assert rE <= 1e-13 and rP <= 1e-13
    assert np.isfinite(st["Erad"]).all() and np.isfinite(st["Frad"]).all() and np.isfinite(st["mom"]).all()
    # the stored state is indeed one with more kinetic than total gas energy (that is why the iteration stopped)
    ekin = (st["mom"] ** 2).sum(0) / (2 * st["rho"])
    assert (ekin >= st["Egas"]).mean() > 0.5
    # cells that stopped after ONE trip equal a run limited to one outer trip
    one = {k: v.copy() for k, v in gc.state.items()}
    oracle_lib.source_update(oracle_model(oracle_lib, gc, outer_maxit=1), one, gc.dt, gc.c, gc.c_hat)
    same = np.all(one["Erad"] == st["Erad"], axis=0)
    assert same.sum() >= s["outer_hist"][1]
