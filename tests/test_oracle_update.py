"""Pins for the oracle's whole update (Eq. 37-52) -- CPU only.

Expected values come from numbers the paper prints (tests/golden), closed forms, invariants,
bisection of a scalar equation built from 30-digit quadrature, and a brute-force 30-digit
Newton solve of the full (4+4Nq) system typed from Eq. 21-22 and 37-40 -- never from the
oracle's own algebra or from the CUDA path.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

from paper_2407_18304_b200 import workloads as W

mp.mp.dps = 30
GOLD = os.path.join(os.path.dirname(__file__), "golden")
C15 = 15 / mp.pi ** 4


def mp_dY(xlo, xhi):
    """(15/pi^4) int t^3/(e^t-1), scaled so mp.quad's absolute stopping rule works in the tail."""
    xlo, xhi = mp.mpf(xlo), mp.mpf(xhi)
    top = min(xhi, xlo + 150)
    pts = [xlo + d for d in (0, 1, 2, 4, 8, 16, 32, 64) if xlo + d < top] + [top]
    if xlo < 1 < top:
        pts = sorted(set(pts + [mp.mpf(1)]))
    g = lambda t: t ** 3 * mp.exp(xlo - t) / (-mp.expm1(-t))  # noqa: E731
    return C15 * mp.exp(-xlo) * mp.quad(g, pts)


def mp_Xi(x):
    x = mp.mpf(x)
    if x == 0 or x == mp.inf:
        return mp.mpf(0)
    return C15 * x ** 4 / mp.expm1(x)


def one_cell_state(Nq, rho, mom, Egas, E, F, kscale=None):
    st = {
        "rho": np.array([rho], dtype=np.float64),
        "mom": np.array(mom, dtype=np.float64).reshape(3, 1).copy(),
        "Egas": np.array([Egas], dtype=np.float64),
        "Erad": np.array(E, dtype=np.float64).reshape(Nq, 1).copy(),
        "Frad": np.array(F, dtype=np.float64).reshape(3, Nq, 1).copy(),
        "kappa_scale": None if kscale is None else np.array([kscale], dtype=np.float64),
    }
    return st


def model_of(oracle, wl, **kw):
    args = dict(a_rad=wl.a_rad, k_B=wl.k_B, h_planck=wl.h_planck, mean_mass=wl.mean_mass, gamma=wl.gamma,
                closure=wl.closure, newton_tol=wl.newton_tol, newton_maxit=wl.newton_maxit,
                outer_maxit=wl.outer_maxit, outer_tol=wl.outer_tol, outer_stop=wl.outer_stop,
                outer_rel_tol=wl.outer_rel_tol)
    args.update(kw)
    return oracle.OracleModel(wl.edges, wl.kappa_lo, wl.alpha, **args)


# ---------------------------------------------------------------------------
# printed equilibrium temperature, Eq. 56
# ---------------------------------------------------------------------------
def test_eq56_printed_equilibrium_temperature(oracle_lib):
    """a_R = k_B = h = c = 1, rho = 1, C_V = 3/2, T_gas,0 = 1, E_rad = 0.  One source
    update with dt -> inf relaxes to the root of a_R T^4 + C_V rho T = C_V rho T_gas,0, printed as
    T = 0.768032502191; then E_g is the group-integrated Planck function at that T (north_star)."""
    T_print = float(open(os.path.join(GOLD, "eq56_equilibrium_T.txt")).read())
    edges = np.array([0.0, 1e-2, 1.0, 1e2, np.inf])
    m = oracle_lib.OracleModel(edges, np.full(4, 1e5), np.zeros(4))       # chi_0 = 1e5 as in PAPER.md:552
    st = one_cell_state(4, 1.0, [0, 0, 0], 1.5, [0, 0, 0, 0], np.zeros((3, 4)))
    stats = oracle_lib.source_update(m, st, 1e9, 1.0, 1.0)
    assert stats["n_newton_unconverged"] == 0
    T = st["Egas"][0] / 1.5
    assert abs(T - T_print) < 5e-13                                        # all 12 printed digits
    assert abs(T ** 4 + 1.5 * T - 1.5) < 2e-13                              # Newton tolerance of Eq. 49
    # groups: compare at the 30-digit root of the same quartic (which must itself reproduce the printed digits);
    # a relative error dT/T in T shows up as ~x_lo dT/T in a Wien-tail group, hence the (1 + x_lo) factor
    T_root = mp.findroot(lambda t: t ** 4 + mp.mpf(3) / 2 * t - mp.mpf(3) / 2, mp.mpf(T_print))
    assert abs(T_root - T_print) < 5e-13
    for g in range(4):
        ref = T_root ** 4 * mp_dY(edges[g] / T_root, edges[g + 1] / T_root)
        assert abs(st["Erad"][g, 0] - ref) <= 3e-13 * (1 + edges[g] / T_print) * ref
    assert abs(st["Erad"].sum() - T ** 4) < 2e-13


def test_static_relaxation_quartic_config1(oracle_lib):
    """Config 1 at dt -> inf, v = 0: every cell relaxes to a_R T^4 + C_v T = E_gas + sum E_g (energy
    balance with E_g = B_g(T)) -- checked against numpy's polynomial roots."""
    wl = W.workload(1, 257)
    st = W.to_numpy(wl.make_state())
    E0 = st["Egas"] + st["Erad"].sum(0)
    rho = st["rho"].copy()
    oracle_lib.source_update(model_of(oracle_lib, wl), st, 1e12, wl.c, wl.c_hat)
    T = st["Egas"] / (1.5 * rho)
    for i in range(0, 257, 16):
        roots = np.roots([wl.a_rad, 0, 0, 1.5 * rho[i], -E0[i]])
        Tq = [r.real for r in roots if abs(r.imag) < 1e-12 and r.real > 0][0]
        assert abs(T[i] - Tq) < 1e-12 * Tq
    assert (np.abs(st["Erad"].sum(0) - wl.a_rad * T ** 4) / E0).max() < 3e-13   # Eq. 49 tolerance, relative to E_tot
    for g in range(4):                                                     # E_g = group-integrated Planck function
        ref = float(T[0] ** 4 * mp_dY(wl.edges[g] / T[0], wl.edges[g + 1] / T[0]))
        assert abs(st["Erad"][g, 0] - ref) < 1e-12 * ref + 1e-16


# ---------------------------------------------------------------------------
# conservation
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("idx,n", [(1, 512), (2, 512), (3, 256), (4, 128), (5, 64)])
@pytest.mark.parametrize("tol", [1e-13, 1e-3])
def test_energy_and_momentum_conserved_to_roundoff(oracle_lib, idx, n, tol):
    """Total energy E_gas + (c/chat) sum E_g and momentum rho v + sum F_g/(c chat) are conserved to
    round-off *regardless of how well Newton converged* -- run with eps = 1e-3 too."""
    wl = W.workload(idx, n)
    st = W.to_numpy(wl.make_state())
    s0 = {k: (None if v is None else v.copy()) for k, v in st.items()}
    stats = oracle_lib.source_update(model_of(oracle_lib, wl, newton_tol=tol), st, wl.dt, wl.c, wl.c_hat)
    k = wl.c / wl.c_hat
    Etot = s0["Egas"] + k * s0["Erad"].sum(0)
    dE = (st["Egas"] + k * st["Erad"].sum(0)) - Etot
    assert np.abs(dE / Etot).max() < 1e-13
    q = 1.0 / (wl.c * wl.c_hat)
    scale = np.sqrt((s0["mom"] ** 2).sum(0)) + q * np.sqrt((s0["Frad"] ** 2).sum(0)).sum(0) + 1e-300
    dP = (st["mom"] + q * st["Frad"].sum(1)) - (s0["mom"] + q * s0["Frad"].sum(1))
    assert np.abs(dP / scale).max() < 1e-13
    assert all(np.isfinite(v).all() for v in st.values() if v is not None)
    if tol == 1e-13:
        assert stats["n_newton_unconverged"] == 0 and stats["n_outer_unconverged"] == 0
        assert stats["n_denominator_nonpositive"] == 0 and stats["n_T_nonpositive_steps"] == 0


# ---------------------------------------------------------------------------
# inner solve: scalar monotone energy balance by bisection (PC, v = 0), chat != c
# ---------------------------------------------------------------------------
def test_inner_solve_matches_bisection_of_scalar_balance(oracle_lib):
    """With v = 0 and PC opacities Eq. 38/42 give E_g' (1 + tau_g) = E_g + tau_g Bt_g(T'), tau_g = chat dt chi_g,
    and Eq. 37: C_v T' + (c/chat) sum_g E_g' = E_gas + (c/chat) sum_g E_g.  Solve that scalar monotone equation by
    bisection with Bt_g from 30-digit quadrature and compare with the oracle's Newton/LU result."""
    edges = np.array([0.0, 0.3, 1.5, 4.0, 11.0, np.inf])
    kap = np.array([3.0, 0.02, 40.0, 1.0, 0.3])
    a_rad, c, chat, dt, rho = 0.7, 10.0, 2.5, 0.13, 1.9
    E = np.array([0.2, 0.01, 0.4, 0.3, 1e-3])
    Egas = 1.5 * rho * 0.8
    m = oracle_lib.OracleModel(edges, kap, np.zeros(5), a_rad=a_rad)
    st = one_cell_state(5, rho, [0, 0, 0], Egas, E, np.zeros((3, 5)))
    oracle_lib.source_update(m, st, dt, c, chat)
    tau = [mp.mpf(chat * dt * rho * k) for k in kap]
    Cv = mp.mpf(1.5 * rho)

    def Enew(T):
        return [(mp.mpf(E[g]) + tau[g] * a_rad * T ** 4 * mp_dY(edges[g] / T, edges[g + 1] / T)) / (1 + tau[g])
                for g in range(5)]

    def bal(T):
        return Cv * T + (mp.mpf(c) / chat) * sum(Enew(T)) - (mp.mpf(Egas) + (mp.mpf(c) / chat) * mp.mpf(E.sum()))

    lo, hi = mp.mpf("0.01"), mp.mpf(5)
    assert bal(lo) < 0 < bal(hi)
    for _ in range(70):
        mid = (lo + hi) / 2
        lo, hi = (mid, hi) if bal(mid) < 0 else (lo, mid)
    Tb = (lo + hi) / 2
    assert abs(st["Egas"][0] / float(Cv) - float(Tb)) < 2e-13 * float(Tb)
    for g, ref in enumerate(Enew(Tb)):
        assert abs(st["Erad"][g, 0] - float(ref)) < 1e-12 * float(ref)


# ---------------------------------------------------------------------------
# whole update: brute-force solve of the full implicit system in 30-digit arithmetic
# ---------------------------------------------------------------------------
def _mp_eq30(chilo, lnr, a_chi, a_Q):
    """Eq. 30 (reading S1) typed out: chi_lo [(r^(aQ+1)-1)/(aQ+1)]^-1 [(r^(ax+aQ+1)-1)/(ax+aQ+1)], ln r at exponent 0."""
    br = lambda q: lnr if q == 0 else mp.expm1(q * lnr) / q  # noqa: E731
    return chilo * br(a_chi + a_Q + 1) / br(a_Q + 1)


def _mp_free_slopes(edges, Q):
    """Eq. A1-A2 typed out in mpmath; edge groups -1."""
    Nq = len(Q)
    qb = [Q[g] / (edges[g + 1] - edges[g]) for g in range(Nq)]
    nb = [mp.sqrt(edges[g + 1] * edges[g]) for g in range(Nq)]
    out = [mp.mpf(-1)] * Nq
    for g in range(1, Nq - 1):
        sm = mp.log(qb[g] / qb[g - 1]) / mp.log(nb[g] / nb[g - 1])
        sp = mp.log(qb[g + 1] / qb[g]) / mp.log(nb[g + 1] / nb[g])
        out[g] = mp.mpf(0) if sm * sp <= 0 else (sm if abs(sm) < abs(sp) else sp)
    return out


def _brute_force_residual(p, x):
    """Residuals of Eq. 37-40 with the four-force of Eq. 21-22 at the NEW state, opacity means from Eq. 30
    (alpha_Q = -1), chi_F from Eq. 27, M1 closure group by group.  Typed from the paper, in mpmath."""
    Nq, c, chat, dt, rho = p["Nq"], p["c"], p["chat"], p["dt"], p["rho"]
    Egas = x[0]
    mom = x[1:4]
    E = x[4:4 + Nq]
    F = [x[4 + Nq + 3 * g: 4 + Nq + 3 * g + 3] for g in range(Nq)]
    v = [mi / rho for mi in mom]
    T = (Egas - sum(mi ** 2 for mi in mom) / (2 * rho)) / p["Cv"]
    aT4 = p["a_rad"] * T ** 4
    res = [None] * (4 + 4 * Nq)
    sumG0c = mp.mpf(0)
    sumG = [mp.mpf(0)] * 3
    # options of the round-2 extensions (absent = the round-1 system):
    #   "S": source terms S_g;  "pT","Tref": chi(T) = chi (T/Tref)^pT at the NEW temperature;
    #   "free": alpha_Q of Appendix A recomputed from the NEW B_g and E_g
    S = p.get("S", [mp.mpf(0)] * Nq)
    tscale = (T / p["Tref"]) ** p["pT"] if "pT" in p else mp.mpf(1)
    Bts = [aT4 * mp_dY(p["h"] * p["edges"][g] / (p["kB"] * T), p["h"] * p["edges"][g + 1] / (p["kB"] * T)) for g in range(Nq)]
    aB = aE = [mp.mpf(-1)] * Nq
    if p.get("free"):
        aB, aE = _mp_free_slopes(p["edges"], Bts), _mp_free_slopes(p["edges"], E)
    for g in range(Nq):
        nlo, nhi, al, chilo = p["edges"][g], p["edges"][g + 1], p["alpha"][g], p["chi_lo"][g] * tscale
        lnr = mp.log(nhi / nlo) if al != 0 else mp.mpf(1)
        chihi = chilo * mp.exp(al * lnr) if al != 0 else chilo
        chiB, chiE = (_mp_eq30(chilo, lnr, al, aB[g]), _mp_eq30(chilo, lnr, al, aE[g])) if al != 0 else (chilo, chilo)
        xlo, xhi = p["h"] * nlo / (p["kB"] * T), p["h"] * nhi / (p["kB"] * T)
        Bt = Bts[g]
        Db = aT4 * (mp_Xi(xhi) - mp_Xi(xlo))
        D = aT4 * (chihi * mp_Xi(xhi) - chilo * mp_Xi(xlo))
        chiF = ((chiB + chiE / 3) * Bt + (al * chiE * Bt - D) / 3) / (mp.mpf(4) / 3 * Bt - Db / 3)   # Eq. 27
        if g in p.get("chiF_is_chiE", ()):       # reading S8(ii): groups in which 1 + c_hat chi_F dt <= 0
            assert 1 + chat * chiF * dt <= 0
            chiF = chiE
        Fn = mp.sqrt(sum(f ** 2 for f in F[g]))
        f = Fn / (c * E[g])
        chiEdd = (3 + 4 * f ** 2) / (5 + 2 * mp.sqrt(4 - 3 * f ** 2))                     # Levermore 1984
        n = [fi / Fn for fi in F[g]]
        ndv = sum(n[i] * v[i] for i in range(3))
        vP = [E[g] * ((1 - chiEdd) / 2 * v[i] + (3 * chiEdd - 1) / 2 * n[i] * ndv) for i in range(3)]
        vF = sum(v[i] * F[g][i] for i in range(3))
        # -c G0_g (Eq. 21) and -G^i_g (Eq. 22), in energy-density units (4 pi B_g = c Bt)
        mcG0 = c * chiB * Bt - c * chiE * E[g] + (1 + al) * chiF * vF / c
        mG = [-chiF * F[g][i] / c + v[i] * (chiB * Bt - D / 3) / c + (1 + al) * chiE * vP[i] / c for i in range(3)]
        res[4 + g] = E[g] - p["E0"][g] - (chat / c) * dt * mcG0 - S[g]                    # Eq. 38 (+ S_g, Eq. 41)
        for i in range(3):
            res[4 + Nq + 3 * g + i] = F[g][i] - p["F0"][g][i] - chat * c * dt * mG[i]      # Eq. 40
            sumG[i] += -mG[i]
        sumG0c += -mcG0
    res[0] = Egas - p["Egas0"] - dt * sumG0c                                              # Eq. 37
    for i in range(3):
        res[1 + i] = mom[i] - p["mom0"][i] - dt * sumG[i]                                  # Eq. 39
    return res


@pytest.mark.parametrize("case", [0, 1])
def test_whole_update_matches_brute_force_solve(oracle_lib, case):
    """The iteration converges to the root of the fully implicit per-cell system ("render this
    scheme fully implicit").  Solve that (4+4Nq) system by Newton in 30-digit arithmetic, from the paper's
    equations typed out above, and compare every field."""
    if case == 0:
        Nq, edges, alpha, kap = 3, [0.05, 0.6, 3.0, 20.0], [-2.0, 1.0, -3.5], [4.0, 0.3, 2.0]
        a_rad, c, chat, dt, rho, T0, beta = 1e-3, 1e3, 2e2, 2e-3, 1.7, 1.3, 3e-3
    else:
        Nq, edges, alpha, kap = 2, [0.2, 2.0, 9.0], [0.0, -1.0], [30.0, 500.0]
        a_rad, c, chat, dt, rho, T0, beta = 1e-3, 1e3, 1e3, 1e-2, 0.6, 2.1, 8e-3
    rng = np.random.default_rng(case)
    vdir = rng.normal(size=3)
    vdir /= np.linalg.norm(vdir)
    mom0 = rho * beta * c * vdir
    Egas0 = 1.5 * rho * T0 + 0.5 * (mom0 ** 2).sum() / rho
    E0 = np.array([float(a_rad * (0.8 * T0) ** 4 * mp_dY(edges[g] / (0.8 * T0), edges[g + 1] / (0.8 * T0)))
                   for g in range(Nq)])
    F0 = np.array([0.4 * c * E0[g] * (lambda d: d / np.linalg.norm(d))(rng.normal(size=3)) for g in range(Nq)])
    m = oracle_lib.OracleModel(np.array(edges), np.array(kap), np.array(alpha), a_rad=a_rad)
    st = one_cell_state(Nq, rho, mom0, Egas0, E0, F0.T.copy())
    stats = oracle_lib.source_update(m, st, dt, c, chat)
    assert stats["n_outer_unconverged"] == 0 and stats["n_newton_unconverged"] == 0

    M = mp.mpf
    p = dict(Nq=Nq, c=M(c), chat=M(chat), dt=M(dt), rho=M(rho), Cv=M(1.5) * M(rho), a_rad=M(a_rad), h=M(1), kB=M(1),
             edges=[M(e) for e in edges], alpha=[M(a) for a in alpha], chi_lo=[M(rho) * M(k) for k in kap],
             E0=[M(e) for e in E0], F0=[[M(f) for f in F0[g]] for g in range(Nq)], Egas0=M(Egas0),
             mom0=[M(t) for t in mom0])
    x0 = [M(st["Egas"][0])] + [M(st["mom"][i, 0]) for i in range(3)] + [M(st["Erad"][g, 0]) for g in range(Nq)]
    for g in range(Nq):
        x0 += [M(st["Frad"][i, g, 0]) for i in range(3)]
    # starting from the input state also works but takes longer; the root is what is compared
    sol = mp.findroot(lambda *x: _brute_force_residual(p, list(x)), x0, tol=1e-40, maxsteps=30)
    sol = [sol[i] for i in range(len(x0))]
    res = _brute_force_residual(p, sol)
    assert max(abs(r) for r in res) < mp.mpf(10) ** -22
    Etot = Egas0 + E0.sum()
    got = [float(t) for t in x0]
    ref = [float(t) for t in sol]
    scale = [Etot] + [np.linalg.norm(mom0)] * 3 + [Etot] * Nq + [c * Etot] * (3 * Nq)
    for gv, rv, sc in zip(got, ref, scale):
        assert abs(gv - rv) <= 1e-11 * abs(rv) + 1e-13 * sc
    # and the update really moved the state (the comparison above is not vacuous)
    assert abs(st["Egas"][0] - Egas0) > 1e-6 * Egas0


# ---------------------------------------------------------------------------
# grey limit (Eq. 5-6)
# ---------------------------------------------------------------------------
def _grey_residual(p, x):
    """Eq. 37-40 with the grey four-force of Eq. 5-6 (chi_P = chi_E = chi_F = chi), Eddington closure."""
    c, chat, dt, rho, chi = p["c"], p["chat"], p["dt"], p["rho"], p["chi"]
    Egas, mom, E, F = x[0], x[1:4], x[4], x[5:8]
    v = [mi / rho for mi in mom]
    T = (Egas - sum(mi ** 2 for mi in mom) / (2 * rho)) / p["Cv"]
    B = p["a_rad"] * T ** 4                                     # 4 pi B / c
    vF = sum(v[i] * F[i] for i in range(3))
    mcG0 = c * chi * B - c * chi * E + (2 * chi - chi) * vF / c                          # Eq. 5
    mG = [-chi * F[i] / c + v[i] * chi * B / c + chi * v[i] * E / 3 / c + (chi - chi) * v[i] * E / c
          for i in range(3)]                                                              # Eq. 6, P = E/3 I
    res = [Egas - p["Egas0"] + dt * mcG0, None, None, None, E - p["E0"] - (chat / c) * dt * mcG0]
    for i in range(3):
        res[1 + i] = mom[i] - p["mom0"][i] + dt * mG[i]
        res.append(F[i] - p["F0"][i] - chat * c * dt * mG[i])
    return res


def test_Nq1_reduces_to_grey_mixed_frame_update(oracle_lib):
    """Nq = 1 with edges {0, inf} and PC opacity: Db = D = 0, chi_F = chi, and the update must solve the grey
    system of Eq. 5-6 (north_star: 'the Nq=1 case reducing to the grey mixed-frame update')."""
    a_rad, c, chat, dt, rho, chi_s = 1e-3, 1e3, 5e2, 4e-3, 1.3, 2.0
    mom0 = np.array([3.0, -1.0, 2.0])
    T0 = 1.4
    Egas0 = 1.5 * rho * T0 + 0.5 * (mom0 ** 2).sum() / rho
    E0 = a_rad * 0.9 ** 4
    F0 = np.array([0.1, 0.2, -0.15]) * c * E0
    m = oracle_lib.OracleModel(np.array([0.0, np.inf]), np.array([chi_s]), np.zeros(1), a_rad=a_rad, closure=1)
    st = one_cell_state(1, rho, mom0, Egas0, [E0], F0.reshape(3, 1))
    oracle_lib.source_update(m, st, dt, c, chat)
    M = mp.mpf
    p = dict(c=M(c), chat=M(chat), dt=M(dt), rho=M(rho), chi=M(rho) * M(chi_s), Cv=M(1.5) * M(rho), a_rad=M(a_rad),
             Egas0=M(Egas0), mom0=[M(t) for t in mom0], E0=M(E0), F0=[M(t) for t in F0])
    x0 = [M(st["Egas"][0])] + [M(st["mom"][i, 0]) for i in range(3)] + [M(st["Erad"][0, 0])] + \
         [M(st["Frad"][i, 0, 0]) for i in range(3)]
    sol = mp.findroot(lambda *x: _grey_residual(p, list(x)), x0, tol=1e-40, maxsteps=30)
    scale = [Egas0] + [np.linalg.norm(mom0)] * 3 + [Egas0] + [c * Egas0] * 3
    for i in range(8):
        assert abs(float(x0[i]) - float(sol[i])) <= 1e-11 * abs(float(sol[i])) + 1e-13 * scale[i]
    assert abs(st["Erad"][0, 0] - E0) > 1e-3 * E0


def test_frequency_independent_opacity_multigroup_equals_grey(oracle_lib):
    """with a frequency-independent opacity the multigroup scheme reduces to the grey one.
    With the Eddington closure (linear in E_g) the sums over groups of E_g and F_g, rho v and E_gas of an
    Nq-group run over [0, inf) equal the Nq = 1 run started from the summed state."""
    a_rad, c, chat, dt, rho, kap = 1e-3, 1e3, 1e3, 3e-3, 0.8, 5.0
    edges = np.array([0.0, 0.5, 1.5, 3.0, 6.0, 12.0, np.inf])
    Nq = 6
    rng = np.random.default_rng(7)
    mom0 = rho * 4.0 * np.array([0.6, 0.0, -0.8])
    Egas0 = 1.5 * rho * 1.2 + 0.5 * (mom0 ** 2).sum() / rho
    E0 = np.array([float(a_rad * mp_dY(edges[g], edges[g + 1])) for g in range(Nq)]) * rng.uniform(0.5, 1.5, Nq)
    F0 = rng.uniform(-0.3, 0.3, (3, Nq)) * c * E0
    mg = oracle_lib.OracleModel(edges, np.full(Nq, kap), np.zeros(Nq), a_rad=a_rad, closure=1)
    m1 = oracle_lib.OracleModel(np.array([0.0, np.inf]), np.array([kap]), np.zeros(1), a_rad=a_rad, closure=1)
    sg = one_cell_state(Nq, rho, mom0, Egas0, E0, F0)
    s1 = one_cell_state(1, rho, mom0, Egas0, [E0.sum()], F0.sum(1).reshape(3, 1))
    oracle_lib.source_update(mg, sg, dt, c, chat)
    oracle_lib.source_update(m1, s1, dt, c, chat)
    assert abs(sg["Egas"][0] - s1["Egas"][0]) < 1e-12 * Egas0
    assert abs(sg["Erad"].sum() - s1["Erad"][0, 0]) < 1e-12 * Egas0
    assert np.abs(sg["mom"][:, 0] - s1["mom"][:, 0]).max() < 1e-12 * np.linalg.norm(mom0)
    assert np.abs(sg["Frad"].sum(1)[:, 0] - s1["Frad"][:, 0, 0]).max() < 1e-12 * c * Egas0


# ---------------------------------------------------------------------------
# diffusion limit and moving equilibrium (Eq. 26, Eq. 16)
# ---------------------------------------------------------------------------
@pytest.mark.parametrize("alpha", [0.0, -2.0, 1.0])
def test_diffusion_limit_flux_eq26(oracle_lib, alpha):
    """at high optical depth in a moving medium the group flux tends to
    F_g,diff = v (4/3 Bt_g - Db_g / 3) (Eq. 26, energy-density units) for ANY opacity slope, because chi_F is
    Eq. 27.  One update with dt -> inf, Eddington closure; agreement to O(beta^2)."""
    a_rad, c, rho, T0, beta = 1.0, 1.0, 1.0, 1.0, 1e-3
    edges = np.array([0.5, 1.0, 2.0, 4.0, 8.0])
    Nq = 4
    v = beta * c * np.array([1.0, 0.0, 0.0])
    # heavy gas (mean_mass tiny => huge C_v) so that T and v stay put while radiation relaxes
    m = oracle_lib.OracleModel(edges, np.full(Nq, 1e3), np.full(Nq, alpha), a_rad=a_rad, closure=1, mean_mass=1e-8)
    rho_big = 1e8
    Cv = rho_big * 1.0 / ((5.0 / 3.0 - 1.0) * 1e-8)
    mom0 = rho_big * v
    Egas0 = Cv * T0 + 0.5 * (mom0 ** 2).sum() / rho_big
    E0 = np.array([float(a_rad * T0 ** 4 * mp_dY(edges[g] / T0, edges[g + 1] / T0)) for g in range(Nq)])
    st = one_cell_state(Nq, rho_big, mom0, Egas0, E0, np.zeros((3, Nq)), kscale=1.0 / rho_big)
    oracle_lib.source_update(m, st, 1e6, c, c)
    for g in range(Nq):
        Bt = a_rad * T0 ** 4 * mp_dY(edges[g] / T0, edges[g + 1] / T0)
        Db = a_rad * T0 ** 4 * (mp_Xi(edges[g + 1] / T0) - mp_Xi(edges[g] / T0))
        Fdiff = float(v[0] * (mp.mpf(4) / 3 * Bt - Db / 3))
        assert abs(st["Frad"][0, g, 0] - Fdiff) < 2e-5 * abs(Fdiff)      # 1 + O(beta^2), beta = 1e-3 (and 1/tau)
        assert abs(st["Frad"][1, g, 0]) < 1e-12 * abs(Fdiff)


def test_moving_equilibrium_eq16_is_stationary(oracle_lib):
    """PAPER.md:218-222 Eq. 16: for constant chi the state E = aT^4 (1 + 4/3 beta^2), F = 4/3 v aT^4 makes
    c G0 = G = 0.  Grey (Nq = 1, edges {0, inf}), Eddington closure: one update must leave it unchanged up to the
    O(beta^2) cross terms that Eq. 16 drops (v^j P^ji with P = E/3 I gives F = (1 + 1/3(1+4/3 beta^2)) v aT^4)."""
    a_rad, c, rho, T0, beta = 1e-3, 1e3, 2.0, 1.1, 1e-3
    v = beta * c * np.array([0.0, 0.6, 0.8])
    aT4 = a_rad * T0 ** 4
    E0 = aT4 * (1 + 4.0 / 3.0 * beta ** 2)
    F0 = 4.0 / 3.0 * v * aT4
    mom0 = rho * v
    Egas0 = 1.5 * rho * T0 + 0.5 * (mom0 ** 2).sum() / rho
    m = oracle_lib.OracleModel(np.array([0.0, np.inf]), np.array([50.0]), np.zeros(1), a_rad=a_rad, closure=1)
    st = one_cell_state(1, rho, mom0, Egas0, [E0], F0.reshape(3, 1))
    oracle_lib.source_update(m, st, 10.0, c, c)
    assert abs(st["Erad"][0, 0] - E0) < 10 * beta ** 2 * beta ** 2 * E0 + 1e-12 * E0
    assert np.abs(st["Frad"][:, 0, 0] - F0).max() < 2 * beta ** 2 * np.linalg.norm(F0)
    assert abs(st["Egas"][0] - Egas0) < 1e-6 * beta ** 2 * Egas0 + 1e-13 * Egas0


# ---------------------------------------------------------------------------
# controls
# ---------------------------------------------------------------------------
def test_argument_errors(oracle_lib):
    st = one_cell_state(2, 1.0, [0, 0, 0], 1.5, [0.1, 0.1], np.zeros((3, 2)))
    good = oracle_lib.OracleModel(np.array([0.1, 1.0, 10.0]), np.ones(2), np.zeros(2))
    with pytest.raises(ValueError):
        oracle_lib.source_update(good, st, -1.0, 1.0, 1.0)                    # dt <= 0
    with pytest.raises(ValueError):
        oracle_lib.source_update(good, st, 1.0, 1.0, 2.0)                     # chat > c
    bad = oracle_lib.OracleModel(np.array([0.1, 0.05, 10.0]), np.ones(2), np.zeros(2))
    with pytest.raises(ValueError):
        oracle_lib.source_update(bad, st, 1.0, 1.0, 1.0)                      # non-ascending edges
    bad = oracle_lib.OracleModel(np.array([0.0, 1.0, 10.0]), np.ones(2), np.array([-1.0, 0.0]))
    with pytest.raises(ValueError):
        oracle_lib.source_update(bad, st, 1.0, 1.0, 1.0)                      # slope in a group touching nu = 0


def test_outer_iteration_counts_are_a_handful(oracle_lib):
    # "never require more than a handful of outer iterations"
    for idx, n in ((2, 256), (4, 64)):
        wl = W.workload(idx, n)
        st = W.to_numpy(wl.make_state())
        stats = oracle_lib.source_update(model_of(oracle_lib, wl, outer_stop=0), st, wl.dt, wl.c, wl.c_hat)
        assert stats["n_outer_unconverged"] == 0
        assert np.nonzero(stats["outer_hist"])[0].max() <= 8
