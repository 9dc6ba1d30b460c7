"""GPU parity of the round-2 model options against the oracle: the source term S_g and the temperature
power-law opacities (tuned kernel), the free-slope spectrum fit and the tabulated edge opacities with
alpha from Eq. 20 (general kernel, one warp per cell), at several group counts including ragged ones and
both groups-per-lane instantiations, plus cross-checks between the two kernels.
"""
import math

import numpy as np
import pytest

from paper_2407_18304_b200 import workloads as W

from parity_util import afloor_quasi_newton, assert_parity, conservation_residual, oracle_model
from test_oracle_next import eq63_setup

pytestmark = pytest.mark.gpu

COUNTERS = ("n_newton_unconverged", "n_outer_unconverged", "n_T_nonpositive_steps", "n_denominator_nonpositive",
            "n_chiF_guard")


@pytest.fixture(scope="module")
def gpu():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device is visible")
    from paper_2407_18304_b200 import binding

    binding.load_library()
    return binding


def _copy(st):
    return {k: (None if v is None else v.copy()) for k, v in st.items()}


def run_gpu(gpu, wl, st0, dt, host=False):
    import torch

    ctx = gpu.Context.from_workload(wl)
    if host:
        got = _copy(st0)
        ctx.source_update_host(got, dt, wl.c, wl.c_hat)
    else:
        dev = {k: (None if v is None else torch.from_numpy(v).cuda()) for k, v in st0.items()}
        ctx.source_update(dev, dt, wl.c, wl.c_hat)
        torch.cuda.synchronize()
        got = W.to_numpy(dev)
    stats = ctx.get_stats()
    ctx.free()
    return got, stats


def both(gpu, oracle, wl, st0, dt):
    ref = _copy(st0)
    ostats = oracle.source_update(oracle_model(oracle, wl), ref, dt, wl.c, wl.c_hat)
    got, gstats = run_gpu(gpu, wl, st0, dt)
    return ref, got, gstats, ostats


def check(ref, got, st0, wl, gs, os_, label, counters=True):
    ref = {k: v for k, v in ref.items() if k != "Srad"}
    quasi = getattr(wl, "opacity_kind", 0) != 0 or getattr(wl, "spectrum", 0) != 0
    assert_parity(ref, got, st0, wl.c, wl.c_hat, label=label,
                  afloor=afloor_quasi_newton(wl.newton_tol) if quasi else 1e-14)
    if counters:
        for key in COUNTERS:
            assert gs[key] == os_[key], (label, key, gs[key], os_[key])
        assert abs(gs["newton_evals_total"] - os_["newton_evals_total"]) <= 0.02 * os_["newton_evals_total"]
        assert abs(gs["outer_trips_total"] - os_["outer_trips_total"]) <= 0.02 * os_["outer_trips_total"]


def source_of(st0, seed):
    rng = np.random.default_rng(seed)
    S = st0["Erad"] * rng.uniform(0.0, 2.0, st0["Erad"].shape)
    S[:, ::7] = 0.0
    return np.ascontiguousarray(S)


# ---------------------------------------------------------------------------------------------------
# S_g (tuned kernel)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("index,n", [(1, 1000), (2, 3001), (3, 1203), (4, 1501), (5, 517)])
def test_source_term_parity_and_conservation(gpu, oracle_lib, index, n):
    wl = W.workload(index, ncells=n)
    st0 = W.to_numpy(wl.make_state())
    st0["Srad"] = source_of(st0, index)
    dt = wl.dt_of_call(0)
    ref, got, gs, os_ = both(gpu, oracle_lib, wl, st0, dt)
    base = {k: v for k, v in st0.items() if k != "Srad"}
    scale_state = dict(base, Erad=st0["Erad"] + st0["Srad"])       # tolerances relative to E^t + S
    check(ref, got, scale_state, wl, gs, os_, f"config {index} with S_g")
    # E_gas + (c/c_hat) sum (E_g - S_g) and the momentum are conserved to round-off
    shifted = dict(got, Erad=got["Erad"] - st0["Srad"])
    rE, rP = conservation_residual(scale_state, dict(shifted, Erad=shifted["Erad"] + st0["Srad"]), wl.c, wl.c_hat)
    dE = (got["Egas"] + (wl.c / wl.c_hat) * (got["Erad"] - st0["Srad"]).sum(0)) - (st0["Egas"] + (wl.c / wl.c_hat) * st0["Erad"].sum(0))
    sc = np.abs(st0["Egas"]) + (wl.c / wl.c_hat) * (np.abs(st0["Erad"]) + st0["Srad"]).sum(0)
    assert np.max(np.abs(dE) / sc) <= 1e-13 and rP <= 1e-13
    assert np.array_equal(got["Srad"], st0["Srad"]) and np.array_equal(got["rho"], st0["rho"])
    # the source matters
    plain, _ = run_gpu(gpu, wl, base, dt)
    assert np.abs(plain["Erad"] - got["Erad"]).max() > 1e-3 * np.abs(got["Erad"]).max()


def test_source_term_zero_is_bit_identical_and_host_path(gpu, oracle_lib):
    wl = W.workload(4, ncells=2000 + 5)
    st0 = W.to_numpy(wl.make_state())
    a, _ = run_gpu(gpu, wl, st0, wl.dt)
    z = dict(st0, Srad=np.zeros_like(st0["Erad"]))
    b, _ = run_gpu(gpu, wl, z, wl.dt)
    for key in ("mom", "Egas", "Erad", "Frad"):
        assert np.array_equal(a[key], b[key]), key
    s = dict(st0, Srad=source_of(st0, 9))
    d, _ = run_gpu(gpu, wl, s, wl.dt)
    h, _ = run_gpu(gpu, wl, s, wl.dt, host=True)
    for key in ("mom", "Egas", "Erad", "Frad"):
        assert np.array_equal(d[key], h[key]), key


def test_source_term_invalid_cell_left_untouched(gpu, oracle_lib):
    wl = W.workload(2, ncells=64)
    st0 = W.to_numpy(wl.make_state())
    st0["Srad"] = source_of(st0, 1) + 1e-3
    st0["Egas"][10] = 0.5 * (st0["mom"][:, 10] ** 2).sum() / (2 * st0["rho"][10])
    ref, got, gs, os_ = both(gpu, oracle_lib, wl, st0, wl.dt)
    for key in ("Egas", "Erad", "Frad", "mom"):
        assert np.array_equal(got[key][..., 10], st0[key][..., 10]), key
        assert np.array_equal(ref[key][..., 10], st0[key][..., 10]), key
    assert gs["n_T_nonpositive_steps"] == os_["n_T_nonpositive_steps"] == 1


# ---------------------------------------------------------------------------------------------------
# opacity kind 1: chi ~ (T/T_ref)^p at the trial temperature (tuned kernel)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("index,n,pT", [(4, 1501, 1.5), (3, 1203, -3.5), (2, 3001, 1.5), (5, 517, 1.5), (1, 1000, 1.5)])
def test_temperature_powerlaw_opacity(gpu, oracle_lib, index, n, pT):
    """Marshak (c) of PAPER.md:499 (chi_g (T/T_0)^{3/2}) on the BASELINE workloads' shapes; -3.5 is the
    temperature exponent of the means of Eq. 63."""
    wl = W.workload(index, ncells=n)
    wl.opacity_kind, wl.T_ref, wl.p_T = 1, 1.3, pT
    st0 = W.to_numpy(wl.make_state())
    dt = wl.dt_of_call(0)
    ref, got, gs, os_ = both(gpu, oracle_lib, wl, st0, dt)
    check(ref, got, st0, wl, gs, os_, f"config {index}, chi ~ T^{pT}")
    rE, rP = conservation_residual(st0, got, wl.c, wl.c_hat)
    assert rE <= 1e-13 and rP <= 1e-13
    wl0 = W.workload(index, ncells=n)
    plain, _ = run_gpu(gpu, wl0, st0, dt)
    assert np.abs(plain["Erad"] - got["Erad"]).max() > 1e-3 * np.abs(got["Erad"]).max()


# ---------------------------------------------------------------------------------------------------
# general kernel: free-slope spectrum, tabulated edge opacities
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("index,n", [(2, 1001), (3, 703), (4, 601), (5, 203)])
def test_free_slope_parity(gpu, oracle_lib, index, n):
    wl = W.workload(index, ncells=n)
    wl.spectrum = 1
    st0 = W.to_numpy(wl.make_state())
    if index == 4:
        st0["Erad"][::5, ::3] = 0.0          # zero energies: no logarithm, fixed-slope value (reading S21)
    dt = wl.dt_of_call(0)
    ref, got, gs, os_ = both(gpu, oracle_lib, wl, st0, dt)
    check(ref, got, st0, wl, gs, os_, f"config {index}, free slope")
    rE, rP = conservation_residual(st0, got, wl.c, wl.c_hat)
    assert rE <= 1e-13 and rP <= 1e-13
    fixed, _ = run_gpu(gpu, W.workload(index, ncells=n), st0, dt)
    assert np.abs(fixed["Erad"] - got["Erad"]).max() > 1e-6 * np.abs(got["Erad"]).max()


@pytest.mark.parametrize("Nq", [3, 5, 31, 33, 47, 64])
def test_general_kernel_equals_tuned_kernel_for_piecewise_constant(gpu, oracle_lib, Nq):
    """alpha_chi = 0: the free-slope option changes nothing, so the general kernel (which the
    option selects) must reproduce the tuned kernel and the oracle -- ragged group counts, both groups-per-lane
    instantiations, with a source term."""
    wl = W.workload(4 if Nq <= 32 else 5, ncells=257)
    wl.Nq = Nq
    wl.edges = np.logspace(-3.0, 3.0, Nq + 1)
    wl.kappa_lo = wl.kappa_lo[:Nq].copy()
    wl.alpha = np.zeros(Nq)
    st0 = W.to_numpy(wl.make_state())
    st0["Srad"] = source_of(st0, Nq)
    tuned, _ = run_gpu(gpu, wl, st0, wl.dt)
    wl.spectrum = 1
    ref, got, gs, os_ = both(gpu, oracle_lib, wl, st0, wl.dt)
    scale_state = dict({k: v for k, v in st0.items() if k != "Srad"}, Erad=st0["Erad"] + st0["Srad"])
    check(ref, got, scale_state, wl, gs, os_, f"general kernel, PC, Nq={Nq}")
    assert_parity({k: v for k, v in tuned.items() if k != "Srad"}, got, scale_state, wl.c, wl.c_hat, label="general vs tuned")


@pytest.mark.parametrize("index,n", [(3, 703), (4, 601), (5, 203)])
def test_edge_table_of_a_power_law(gpu, oracle_lib, index, n):
    """kappa = K (T/T_ref)^p nu^s tabulated at the edges: parity with the oracle's table path, and (since ln kappa
    is linear in ln T and Eq. 20 returns alpha = s) agreement with the tuned kernel's opacity kind 1."""
    wl = W.workload(index, ncells=n)
    s_exp = {3: -3.0, 4: -2.0, 5: -1.5}[index]
    Tref, pT, NT = 1.7, -0.5, 9
    lnT = np.linspace(math.log(0.02), math.log(80.0), NT)
    wl.kappa_lo = wl.edges[:-1] ** s_exp
    wl.alpha = np.full(wl.Nq, s_exp)
    st0 = W.to_numpy(wl.make_state())
    wl.opacity_kind, wl.T_ref, wl.p_T = 1, Tref, pT
    tuned, _ = run_gpu(gpu, wl, st0, wl.dt_of_call(0))
    wl.opacity_kind = 2
    wl.lnk_edge = s_exp * np.log(wl.edges)[:, None] + pT * (lnT[None, :] - math.log(Tref))
    wl.lnT0, wl.dlnT = lnT[0], lnT[1] - lnT[0]
    ref, got, gs, os_ = both(gpu, oracle_lib, wl, st0, wl.dt_of_call(0))
    check(ref, got, st0, wl, gs, os_, f"config {index}, edge table")
    assert_parity(tuned, got, st0, wl.c, wl.c_hat, label="edge table vs kind 1", afloor=afloor_quasi_newton(wl.newton_tol))


@pytest.mark.parametrize("Nq", [16, 64])
def test_eq62_table_in_cgs_units(gpu, oracle_lib, Nq):
    """The setup of the Eq. 63 pin (tests/test_oracle_next.py): Eq. 62 tabulated at the edges, CGS units,
    T = 1e7 K, one optically thin update; and a second, optically thick one (dt = 1e-9 s) with radiation
    present and moving gas, where alpha from Eq. 20 differs from group to group."""
    kw, st, dt, c, norm = eq63_setup(Nq)

    class WL:
        pass

    wl = WL()
    for k, v in kw.items():
        setattr(wl, k, v)
    wl.Nq, wl.c, wl.c_hat, wl.closure = Nq, c, c, 0
    wl.newton_tol, wl.newton_maxit, wl.outer_maxit, wl.outer_tol, wl.outer_stop, wl.outer_rel_tol = 1e-13, 50, 50, 1e-13, 1, 1e-12
    n = 130
    rng = np.random.default_rng(5)
    st0 = {k: (None if v is None else np.ascontiguousarray(np.repeat(v, n, axis=-1))) for k, v in st.items()}
    st0["Egas"] *= rng.uniform(0.5, 2.0, n)
    ref, got, gs, os_ = both(gpu, oracle_lib, wl, st0, dt)
    # (E_g ~ 1e-17 E_gas here: compare the emitted energies relatively, group by group)
    big = ref["Erad"] > 1e-6 * ref["Erad"].max()
    assert np.max(np.abs(got["Erad"][big] / ref["Erad"][big] - 1.0)) < 1e-10
    est = got["Erad"][:, 0].sum() / (norm * (st0["Egas"][0] / st["Egas"][0]) ** 4) * (st0["Egas"][0] / st["Egas"][0]) ** 3.5
    assert abs(est / 3063.96 - 1.0) < (0.7 if Nq == 16 else 0.05)
    # optically thick, with radiation and motion
    T = st0["Egas"] / (1.5 * 1.0 * kw["k_B"] / kw["mean_mass"])
    x = kw["h_planck"] * kw["edges"][:, None] / (kw["k_B"] * T[None, :])
    for g in range(Nq):
        st0["Erad"][g] = kw["a_rad"] * (0.9 * T) ** 4 * np.array([oracle_lib.planck_dY(a / 0.9, b / 0.9) for a, b in zip(x[g], x[g + 1])])
    v = rng.normal(size=(3, n)) * 1e6
    st0["mom"] = st0["rho"][None, :] * v
    st0["Egas"] = st0["Egas"] + 0.5 * st0["rho"] * (v * v).sum(0)
    st0["Frad"] = rng.normal(size=(3, Nq, n)) * 0.05 * c * st0["Erad"][None]
    ref, got, gs, os_ = both(gpu, oracle_lib, wl, st0, 1e-9)
    check(ref, got, st0, wl, gs, os_, f"Eq. 62 table, CGS, Nq={Nq}")
    rE, rP = conservation_residual(st0, got, c, c)
    assert rE <= 1e-13 and rP <= 1e-13


# ---------------------------------------------------------------------------------------------------
# outer_mode 1 ("variant L"): implicit-in-v outer stage (general kernel)
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("index,n,literal", [(2, 1001, True), (2, 1001, False), (4, 601, False), (5, 203, False)])
def test_variant_L_parity(gpu, oracle_lib, index, n, literal):
    """Literal units (a_R = c = 1: radiation inertia q up to several hundred, where the lagged-velocity outer loop of
    PAPER.md:453-467 diverges) and the scaled units of the BASELINE workloads, both groups-per-lane instantiations."""
    wl = W.workload(index, ncells=n)
    if literal:
        wl.a_rad, wl.c, wl.c_hat, wl.dt = 1.0, 1.0, 1.0, 1.0
    wl.outer_mode = 1
    st0 = W.to_numpy(wl.make_state())
    dt = wl.dt_of_call(0)
    ref, got, gs, os_ = both(gpu, oracle_lib, wl, st0, dt)
    assert os_["n_outer_unconverged"] == 0 and os_["n_newton_unconverged"] == 0
    check(ref, got, st0, wl, gs, os_, f"variant L, config {index}, literal={literal}")
    rE, rP = conservation_residual(st0, got, wl.c, wl.c_hat)
    assert rE <= 1e-13 and rP <= 1e-13
    if not literal:      # same converged state as the paper's outer stage (tuned kernel)
        wl0 = W.workload(index, ncells=n)
        lag, _ = run_gpu(gpu, wl0, st0, dt)
        assert_parity(lag, got, st0, wl.c, wl.c_hat, label="variant L vs lagged")
