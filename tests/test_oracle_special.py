"""Pins for the oracle's L1/L2 pieces (Eq. 11, 23, 27, 30, 63) -- CPU only.

Every expected value here comes from the mathematics (adaptive quadrature of the defining
integrals in 30-digit arithmetic, closed forms) or from a number the paper prints; none
comes from the oracle itself or from the CUDA path.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

mp.mp.dps = 30
C15 = 15 / mp.pi ** 4
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def planck_integrand(t):
    return t ** 3 / mp.expm1(t)


def _tail_points(x):
    """Break points for quadrature of the decaying integrand from x upward (scale length ~1)."""
    x = mp.mpf(x)
    return [x + d for d in (0, 1, 2, 4, 8, 16, 32, 64, 150)]


def _scaled_quad(xlo, pts):
    """int t^3/(e^t-1) dt over pts, computed as e^-xlo * int t^3 e^(xlo-t)/(1-e^-t) dt so that mp.quad's
    absolute stopping rule sees an O(1) integrand even deep in the Wien tail."""
    g = lambda t: t ** 3 * mp.exp(xlo - t) / (-mp.expm1(-t))  # noqa: E731
    return mp.exp(-xlo) * mp.quad(g, pts)


def Y_quad(xlo, xhi):
    """(15/pi^4) int_xlo^xhi t^3/(e^t-1) dt by adaptive quadrature (beyond xlo+150 the integrand is < e^-100 relative)."""
    xlo, xhi = mp.mpf(xlo), mp.mpf(xhi)
    pts = [p for p in _tail_points(xlo) if p < xhi] + [min(xhi, xlo + 150)]
    if xlo < 1 < xhi:
        pts = sorted(set(pts + [mp.mpf(1)]))
    return C15 * _scaled_quad(xlo, pts)


def Z_quad(x):
    return C15 * _scaled_quad(mp.mpf(x), _tail_points(x))


XS = [1e-4, 3e-3, 0.05, 0.3, 0.999, 1.0, 1.001, 1.7, 2.5, 5.0, 12.0, 40.0, 120.0, 400.0, 700.0]


@pytest.mark.parametrize("x", XS)
def test_Y_and_Z_match_quadrature(oracle_lib, x):
    # PAPER.md:177 Eq. 11 with Q = B: group integral of the Planck function, here from 0 (Y) and to inf (Z)
    Yq = Y_quad(0, x)
    Zq = Z_quad(x)
    assert abs(oracle_lib.planck_Y(x) - Yq) <= 1e-15 * Yq
    assert abs(oracle_lib.planck_Z(x) - Zq) <= 1e-15 * Zq
    assert abs(Yq + Zq - 1) < mp.mpf(10) ** -24   # the quadrature itself is consistent


def test_branches_agree_at_the_branch_point(oracle_lib):
    # Y from the Maclaurin series just below x=1 and 1-Z from the exponential series just above
    lo, hi = np.nextafter(1.0, 0.0), 1.0
    assert abs(oracle_lib.planck_Y(lo) - oracle_lib.planck_Y(hi)) < 1e-15
    assert abs(oracle_lib.planck_Y(lo) + oracle_lib.planck_Z(lo) - 1.0) < 3e-16
    assert abs(oracle_lib.planck_Y(hi) + oracle_lib.planck_Z(hi) - 1.0) < 3e-16


GROUPS = [(1e-4, 3e-4), (1e-2, 1.0), (0.5, 0.9), (0.9, 1.1), (1.0, 100.0), (3.0, 4.6), (30.0, 46.0),
          (200.0, 266.0), (500.0, 690.0), (650.0, 700.0), (0.0, 0.01), (0.0, 5.0), (2.0, math.inf),
          (150.0, math.inf), (0.0, math.inf)]


@pytest.mark.parametrize("xlo,xhi", GROUPS)
def test_group_integral_matches_quadrature(oracle_lib, xlo, xhi):
    # relative 1e-13 (north_star), including tail-to-tail groups where Y+ - Y- would cancel
    ref = Y_quad(xlo, xhi if math.isfinite(xhi) else max(xlo, 1.0) + 400)
    got = oracle_lib.planck_dY(xlo, xhi)
    assert abs(got - ref) <= 1e-13 * ref


def test_group_integrals_sum_to_one_with_end_groups(oracle_lib):
    # sum_g B_g = a_R T^4 c/4pi when the groups cover [0, inf)
    for T in (0.3, 1.0, 7.0):
        edges = np.array([0.0, 1e-2, 0.3, 1.0, 4.0, 30.0, 1e2, np.inf]) / T
        s = sum(oracle_lib.planck_dY(edges[g], edges[g + 1]) for g in range(len(edges) - 1))
        assert abs(s - 1.0) < 4e-16


@pytest.mark.parametrize("x", XS + [0.0, math.inf])
def test_Xi_closed_form(oracle_lib, x):
    # (4 pi / c) nu B_nu = a_R T^4 (15/pi^4) x^4/(e^x-1); zero at nu = 0 and nu = inf
    if x == 0.0 or math.isinf(x):
        assert oracle_lib.planck_Xi(x) == 0.0
        return
    ref = C15 * mp.mpf(x) ** 4 / mp.expm1(mp.mpf(x))
    assert abs(oracle_lib.planck_Xi(x) - ref) <= 4e-16 * ref


def test_temperature_derivative_identity(oracle_lib):
    # d/dT [a T^4 dY(nu-/T, nu+/T)] = (4 Bt - Db)/T, checked against a high-order finite difference
    # of the quadrature (not of the oracle).  Used by the Jacobian entry of Eq. 46.
    for (nlo, nhi, T) in [(0.01, 0.3, 1.0), (1.0, 3.0, 0.7), (8.0, 30.0, 1.3), (0.5, 60.0, 2.0)]:
        B = lambda t: mp.mpf(t) ** 4 * Y_quad(nlo / mp.mpf(t), nhi / mp.mpf(t))  # noqa: E731
        dBdT_fd = mp.diff(B, T)
        Bt = T ** 4 * oracle_lib.planck_dY(nlo / T, nhi / T)
        Db = T ** 4 * (oracle_lib.planck_Xi(nhi / T) - oracle_lib.planck_Xi(nlo / T))
        assert abs((4 * Bt - Db) / T - dBdT_fd) <= 1e-12 * abs(dBdT_fd)


# ---------------------------------------------------------------------------
# Eq. 30 / Eq. 23 / Eq. 27
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("r,a_chi,a_Q", [(3.16, -2.0, -1.0), (1.54, 1.7, -1.0), (10.0, -3.0, 2.0),
                                         (2.0, -1.0, 0.0), (1.33, 2.0, -3.5), (5.0, 0.5, -1.5), (2.0, 1.0, -1.0)])
def test_eq30_matches_quadrature_of_eq23(oracle_lib, r, a_chi, a_Q):
    # Eq. 23 with chi = chi_lo (nu/nu-)^a_chi (Eq. 19) and Q = (nu/nu-)^a_Q (Eq. 28)
    chi_lo, nlo = 2.5, 0.7
    nhi = nlo * r
    num = mp.quad(lambda nu: chi_lo * (nu / nlo) ** a_chi * (nu / nlo) ** a_Q, [nlo, nhi])
    den = mp.quad(lambda nu: (nu / nlo) ** a_Q, [nlo, nhi])
    got = oracle_lib.chi_mean(chi_lo, math.log(r), a_chi, a_Q)
    assert abs(got - num / den) <= 1e-14 * abs(num / den)


def test_eq30_special_cases(oracle_lib):
    # alpha_chi = 0 reduces to the PC value whatever alpha_Q is
    for aQ in (-3.0, -1.0, 0.0, 2.2):
        assert oracle_lib.chi_mean(1.7, math.log(2.4), 0.0, aQ) == 1.7
    # fixed slope alpha_Q = -1: chi_lo (r^a - 1)/(a ln r)
    r, a = 1.54, -3.3
    assert abs(oracle_lib.chi_mean(1.0, math.log(r), a, -1.0) - (r ** a - 1) / (a * math.log(r))) < 1e-15


def test_eq27_reduces_to_chi_for_piecewise_constant(oracle_lib):
    # chi_F,diff = chi_0,g when chi_B = chi_E = chi_0,g (alpha = 0, D = chi Db)
    rng = np.random.default_rng(5)
    for _ in range(20):
        chi, Bt, Db = rng.uniform(0.1, 10), rng.uniform(0.1, 2), rng.uniform(-1, 1)
        got, guard = oracle_lib.chi_flux(chi, chi, 0.0, chi, Bt, Db, chi * Db, 1.0)
        assert guard == 0 and abs(got - chi) < 1e-14 * chi


def test_eq27_general_value(oracle_lib):
    # Eq. 27 typed out once, independent numbers
    chiB, chiE, al, Bt, Db, D = 2.0, 3.0, -1.5, 0.7, 0.2, 0.9
    ref = ((chiB + chiE / 3) * Bt + (al * chiE * Bt - D) / 3) / (4 * Bt / 3 - Db / 3)
    got, guard = oracle_lib.chi_flux(chiB, chiE, al, 1.0, Bt, Db, D, 1.0)
    assert guard == 0 and abs(got - ref) < 1e-15
    # underflowed group (S8 i): falls back to the lower-edge opacity
    got, guard = oracle_lib.chi_flux(chiB, chiE, al, 1.25, 0.0, 0.0, 0.0, 1.0)
    assert guard == 1 and got == 1.25


def test_eq63_printed_planck_and_rosseland_means(oracle_lib):
    """for chi_0 of Eq. 62 the Planck and Rosseland means are
    (3063.96, 101.248)(T/1e7 K)^-3.5 cm^-1.  Rebuild both from the oracle's group quantities with
    many PPL groups (alpha from the edge values, Eq. 20; alpha_Q = -1) -- this pins planck_dY, planck_Xi,
    chi_mean and the dB/dT identity against numbers the paper prints."""
    chiP_ref, chiR_ref = map(float, open(os.path.join(GOLD, "eq63_mean_opacities.txt")).read().split())
    kB, h, T = 1.380649e-16, 6.62607015e-27, 1e7
    chi0 = lambda x: 180.0 * (x * kB * T / h / 1e18) ** -3 * (-math.expm1(-x))  # noqa: E731  Eq. 62 at T = 1e7 K
    xe = np.logspace(-8, math.log10(80.0), 24001)   # integrand of the Planck mean is flat as x -> 0: start low
    num = den = rn = rd = 0.0
    for g in range(len(xe) - 1):
        lnr = math.log(xe[g + 1] / xe[g])
        al = math.log(chi0(xe[g + 1]) / chi0(xe[g])) / lnr                      # Eq. 20
        chiB = oracle_lib.chi_mean(chi0(xe[g]), lnr, al, -1.0)                   # Eq. 30
        dY = oracle_lib.planck_dY(xe[g], xe[g + 1])
        num += chiB * dY
        den += dY
        dBdT = 4 * dY - (oracle_lib.planck_Xi(xe[g + 1]) - oracle_lib.planck_Xi(xe[g]))
        rn += dBdT
        rd += dBdT / chi0(math.sqrt(xe[g] * xe[g + 1]))
    assert abs(num / den - chiP_ref) < 0.006      # printed to 6 significant digits
    assert abs(rn / rd - chiR_ref) < 0.0006


# ---------------------------------------------------------------------------
# closure and linear algebra
# ---------------------------------------------------------------------------
def test_closure_limits(oracle_lib):
    v = np.array([0.3, -0.2, 0.5])
    # isotropic limit f -> 0: P = E/3 I ; free-streaming f = 1: P = E n n   (Levermore 1984)
    out = oracle_lib.vP(0, 2.0, np.array([0.0, 0.0, 0.0]), v, 1.0)
    assert np.allclose(out, 2.0 / 3 * v, rtol=1e-15)
    out = oracle_lib.vP(0, 2.0, np.array([1e-9, 0.0, 0.0]), v, 1.0)
    assert np.allclose(out, 2.0 / 3 * v, rtol=1e-12)
    n = np.array([2.0, -1.0, 2.0]) / 3.0
    out = oracle_lib.vP(0, 2.0, 2.0 * n, v, 1.0)
    assert np.allclose(out, 2.0 * n * (n @ v), rtol=1e-14)
    # trace of P is E for any f: sum_i P^{ii} = E  -> check with the three unit velocities
    F = np.array([0.3, 0.4, -0.2])
    tr = sum(oracle_lib.vP(0, 1.3, F, e, 1.0)[i] for i, e in enumerate(np.eye(3)))
    assert abs(tr - 1.3) < 1e-15
    # Eddington switch
    assert np.allclose(oracle_lib.vP(1, 1.3, F, v, 1.0), 1.3 / 3 * v, rtol=1e-15)


def test_arrowhead_elimination_matches_dense_lu(oracle_lib):
    # the O(Nq) Gauss-Jordan elimination of the arrowhead Jacobian (Eq. 48)
    rng = np.random.default_rng(11)
    for Nq in (1, 2, 3, 5, 8):
        J0g = np.full(Nq, rng.uniform(1, 10))
        Jg0 = rng.uniform(-2, 2, Nq)
        Jgg = -1.0 - 1.0 / rng.uniform(1e-3, 1e3, Nq)
        rhs = rng.normal(size=Nq + 1)
        A = np.zeros((Nq + 1, Nq + 1))
        A[0, 0] = 1.0
        A[0, 1:] = J0g
        A[1:, 0] = Jg0
        A[np.arange(1, Nq + 1), np.arange(1, Nq + 1)] = Jgg
        x_lu = oracle_lib.lu_solve(A, rhs)
        x_ah = oracle_lib.arrowhead_solve(1.0, J0g, Jg0, Jgg, rhs)
        assert np.allclose(A @ x_lu, rhs, rtol=0, atol=1e-12 * np.abs(rhs).max())
        assert np.allclose(x_ah, x_lu, rtol=1e-12, atol=1e-14)


def test_lu_solve_against_numpy(oracle_lib):
    rng = np.random.default_rng(3)
    for n in (1, 2, 7, 33):
        A = rng.normal(size=(n, n))
        b = rng.normal(size=n)
        assert np.allclose(oracle_lib.lu_solve(A, b), np.linalg.solve(A, b), rtol=1e-10, atol=1e-12)
