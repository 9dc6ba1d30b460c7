"""GPU parity: mgrhd_source_update (CUDA, through the C ABI) against the CPU oracle, element by
element on the same seeded inputs -- the five BASELINE.json workloads at sizes the oracle
finishes in seconds (several CTAs and a ragged tail), edge cases, and the host-buffer path.
"""
import numpy as np
import pytest

from paper_2407_18304_b200 import workloads as W

from parity_util import assert_parity, conservation_residual, oracle_model

pytestmark = pytest.mark.gpu

# cells: not a multiple of the cells per CTA (96-384) nor of 32, spans many CTAs
SIZES = {1: 4096, 2: 5000 + 37, 3: 3000 + 19, 4: 2000 + 5, 5: 1000 + 3}


@pytest.fixture(scope="module")
def gpu():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device is visible")
    from paper_2407_18304_b200 import binding

    binding.load_library()   # must exist: no fallback
    return binding


def run_both(gpu, oracle, wl, st_host, dt, nstates=1, host_path=False):
    """Returns (ref, got, gpu_stats, oracle_stats) after one update of copies of st_host."""
    import torch

    ref = {k: (None if v is None else v.copy()) for k, v in st_host.items()}
    ostats = oracle.source_update(oracle_model(oracle, wl), ref, dt, wl.c, wl.c_hat)
    ctx = gpu.Context.from_workload(wl)
    if host_path:
        got = {k: (None if v is None else v.copy()) for k, v in st_host.items()}
        ctx.source_update_host(got, dt, wl.c, wl.c_hat)
    else:
        dev = {k: (None if v is None else torch.from_numpy(v).cuda()) for k, v in st_host.items()}
        ctx.source_update(dev, dt, wl.c, wl.c_hat)
        torch.cuda.synchronize()
        got = W.to_numpy(dev)
    gstats = ctx.get_stats()
    ctx.free()
    return ref, got, gstats, ostats


@pytest.mark.parametrize("index", [1, 2, 3, 4, 5])
def test_workload_parity(gpu, oracle_lib, index):
    wl = W.workload(index, ncells=SIZES[index])
    st0 = W.to_numpy(wl.make_state())
    dt = wl.dt_of_call(0)
    ref, got, gs, os_ = run_both(gpu, oracle_lib, wl, st0, dt)
    assert_parity(ref, got, st0, wl.c, wl.c_hat, label=wl.name)
    rE, rP = conservation_residual(st0, got, wl.c, wl.c_hat)
    assert rE <= 1e-13 and rP <= 1e-13, (rE, rP)
    assert gs["n_cells"] == wl.ncells
    for key in ("n_newton_unconverged", "n_outer_unconverged", "n_T_nonpositive_steps",
                "n_denominator_nonpositive", "n_chiF_guard"):
        assert gs[key] == os_[key], (key, gs[key], os_[key])
    # iteration counts may differ by rounding in a few cells, never systematically
    assert abs(gs["newton_evals_total"] - os_["newton_evals_total"]) <= 0.02 * os_["newton_evals_total"]
    assert abs(gs["outer_trips_total"] - os_["outer_trips_total"]) <= 0.02 * os_["outer_trips_total"]


@pytest.mark.parametrize("form", [0, 1])
def test_planck_edge_functions_vs_oracle(gpu, oracle_lib, form):
    """The kernel's edge functions (form 0: per-interval polynomial rows; form 1: three branches) against the oracle's
    long-double series, over every row and branch, both sides of every switch point (each row boundary of form 0),
    the Wien tail down to underflow, and the 0 / inf edges."""
    import torch

    switch = 1.0 if form == 0 else 1.25
    bounds = [0.5 * 2.0 ** b * (1 + m / 8) for b in range(7) for m in range(8)] + [64.0, 1.25, 5.5, 8.0]
    xs = np.concatenate([np.logspace(-6, np.log10(744.0), 6000), [0.0, 700.0, 745.0, 760.0, np.inf],
                         bounds, [np.nextafter(v, 0) for v in bounds], [np.nextafter(v, np.inf) for v in bounds]])
    yz, xi, is_y = (t.cpu().numpy() for t in gpu.planck_edge_functions(torch.from_numpy(xs).cuda(), form))
    for x, a, b, k in zip(xs, yz, xi, is_y):
        ref = oracle_lib.planck_Y(x) if k else oracle_lib.planck_Z(x)
        rxi = oracle_lib.planck_Xi(x)
        assert abs(a - ref) <= 4e-15 * abs(ref) + 1e-290, (x, a, ref, k)
        assert abs(b - rxi) <= 4e-15 * abs(rxi) + 1e-290, (x, b, rxi)
        assert k == (1 if x < switch else 0)


def test_successive_calls_config5(gpu, oracle_lib):
    """Config 5 is 100 successive updates with dt varied per call; check the first few."""
    import torch

    wl = W.workload(5, ncells=517)
    st0 = W.to_numpy(wl.make_state())
    ref = {k: (None if v is None else v.copy()) for k, v in st0.items()}
    dev = {k: (None if v is None else torch.from_numpy(v).cuda()) for k, v in st0.items()}
    ctx = gpu.Context.from_workload(wl)
    m = oracle_model(oracle_lib, wl)
    for call in range(4):
        dt = wl.dt_of_call(call)
        before = W.to_numpy(dev)
        oracle_lib.source_update(m, ref, dt, wl.c, wl.c_hat)
        ctx.source_update(dev, dt, wl.c, wl.c_hat)
        torch.cuda.synchronize()
        got = W.to_numpy(dev)
        assert_parity(ref, got, before, wl.c, wl.c_hat, label=f"config5 call {call}")
        rE, rP = conservation_residual(before, got, wl.c, wl.c_hat)
        assert rE <= 1e-13 and rP <= 1e-13, (call, rE, rP)
        # keep the two trajectories from drifting apart through the tolerance: restart the oracle from the GPU state
        ref = {k: (None if v is None else v.copy()) for k, v in got.items()}
    ctx.free()


def test_host_buffer_path(gpu, oracle_lib):
    """mgrhd_source_update_host (slab pipeline) gives the same answer as the device path's oracle."""
    wl = W.workload(2, ncells=3 * 1024 + 77)
    st0 = W.to_numpy(wl.make_state())
    ref, got, gs, _ = run_both(gpu, oracle_lib, wl, st0, wl.dt, host_path=True)
    assert_parity(ref, got, st0, wl.c, wl.c_hat, label="host path")
    assert np.array_equal(got["rho"], st0["rho"])
    assert gs["n_cells"] == wl.ncells


@pytest.mark.parametrize("n", [0, 1, 31, 129])
def test_tiny_and_empty(gpu, oracle_lib, n):
    wl = W.workload(2, ncells=max(n, 1))
    st0 = W.to_numpy(wl.make_state())
    if n == 0:
        st0 = {k: (None if v is None else np.ascontiguousarray(v[..., :0])) for k, v in st0.items()}
        import torch

        dev = {k: (None if v is None else torch.from_numpy(v).cuda()) for k, v in st0.items()}
        ctx = gpu.Context.from_workload(wl)
        ctx.source_update(dev, wl.dt, wl.c, wl.c_hat)      # no-op, must not fail
        assert ctx.get_stats()["n_cells"] == 0
        ctx.free()
        return
    ref, got, _, _ = run_both(gpu, oracle_lib, wl, st0, wl.dt)
    assert_parity(ref, got, st0, wl.c, wl.c_hat, label=f"n={n}")


def test_degenerate_cells(gpu, oracle_lib):
    """Exact zeros in E_g and F_g, zero velocity, Eddington closure, Nq=1 grey, Nq=64 max, c_hat<c."""
    # (a) zeros: config 4 with some groups' energies/fluxes zeroed and some cells at rest
    wl = W.workload(4, ncells=300)
    st0 = W.to_numpy(wl.make_state())
    st0["Erad"][::3, ::2] = 0.0
    st0["Frad"][:, ::3, ::2] = 0.0
    st0["Frad"][:, :, 5::7] = 0.0
    v2 = (st0["mom"][:, 1::5] ** 2).sum(0) / (2 * st0["rho"][1::5])
    st0["Egas"][1::5] -= v2
    st0["mom"][:, 1::5] = 0.0
    ref, got, _, _ = run_both(gpu, oracle_lib, wl, st0, wl.dt)
    assert_parity(ref, got, st0, wl.c, wl.c_hat, label="zeros")
    # (b) Eddington closure
    wl.closure = 1
    st0 = W.to_numpy(wl.make_state())
    ref, got, _, _ = run_both(gpu, oracle_lib, wl, st0, wl.dt)
    assert_parity(ref, got, st0, wl.c, wl.c_hat, label="eddington")
    # (c) grey: Nq = 1, edges {0, inf}, PC (scaled units of configs 2-5, so the lagged-velocity loop contracts)
    wl1 = W.workload(2, ncells=200)
    wl1.edges = np.array([0.0, np.inf]); wl1.kappa_lo = np.array([2.5]); wl1.alpha = np.zeros(1); wl1.Nq = 1
    st0 = W.to_numpy(wl1.make_state())
    ref, got, _, _ = run_both(gpu, oracle_lib, wl1, st0, wl1.dt)
    assert_parity(ref, got, st0, wl1.c, wl1.c_hat, label="grey")
    # (d) reduced speed of light with the maximum group count
    wl5 = W.workload(5, ncells=130)
    wl5.c_hat = 0.05 * wl5.c
    st0 = W.to_numpy(wl5.make_state())
    ref, got, _, _ = run_both(gpu, oracle_lib, wl5, st0, wl5.dt)
    assert_parity(ref, got, st0, wl5.c, wl5.c_hat, label="Nq=64, c_hat=0.05c")



@pytest.mark.parametrize("Nq,lo_exp", [(2, -2.0), (3, -2.0), (5, -3.0), (7, 0.5), (13, -3.0), (27, -3.0),
                                        (31, 0.5), (33, -3.0), (47, -4.0), (63, -4.0), (50, 0.5)])
def test_ragged_group_counts(gpu, oracle_lib, Nq, lo_exp):
    """Group counts that are not a multiple of the lanes per cell (ragged last step of loop A and of
    the flux loops, every kernel instantiation), and group structures whose LOWEST edge is not in the
    Rayleigh-Jeans range (lo_exp = 0.5: x_0 = 3.2/T, the called edge-function path of the prologue)."""
    wl = W.workload(4 if Nq <= 32 else 5, ncells=257)
    wl.Nq = Nq
    wl.edges = np.logspace(lo_exp, lo_exp + 4.0 + (2.0 if Nq > 8 else 0.0), Nq + 1)
    wl.kappa_lo = wl.kappa_lo[:Nq].copy()
    # wide groups (few of them) with rising opacity can make Eq. 27 negative (S8): keep alpha <= 0 there
    wl.alpha = wl.alpha[:Nq].copy() if Nq >= 16 else np.minimum(wl.alpha[:Nq], 0.0)
    st0 = W.to_numpy(wl.make_state())
    ref, got, gs, os_ = run_both(gpu, oracle_lib, wl, st0, wl.dt)
    assert_parity(ref, got, st0, wl.c, wl.c_hat, label=f"Nq={Nq}, lowest edge 1e{lo_exp}")
    rE, rP = conservation_residual(st0, got, wl.c, wl.c_hat)
    assert rE <= 1e-13 and rP <= 1e-13, (rE, rP)
    for key in ("n_newton_unconverged", "n_outer_unconverged", "n_denominator_nonpositive", "n_chiF_guard"):
        assert gs[key] == os_[key], (key, gs[key], os_[key])



@pytest.mark.parametrize("index", [2, 3, 4, 5])
def test_bit_reproducible_and_independent_of_scheduling(gpu, index):
    """A cell's result depends on that cell alone: the same state updated twice, as a whole or as its
    first third only (other chunks, other neighbours in the warp, other lane assignments in the flux
    pass), and through the host-buffer path (slabs), gives the same bits."""
    import torch

    wl = W.workload(index, ncells=3001)
    st0 = W.to_numpy(wl.make_state())
    dt = wl.dt_of_call(0)

    def run(state, host=False):
        ctx = gpu.Context.from_workload(wl)
        if host:
            out = {k: (None if v is None else v.copy()) for k, v in state.items()}
            ctx.source_update_host(out, dt, wl.c, wl.c_hat)
        else:
            dev = {k: (None if v is None else torch.from_numpy(v.copy()).cuda()) for k, v in state.items()}
            ctx.source_update(dev, dt, wl.c, wl.c_hat)
            torch.cuda.synchronize()
            out = W.to_numpy(dev)
        ctx.free()
        return out

    a, b, h = run(st0), run(st0), run(st0, host=True)
    m = 1000
    part = {k: (None if v is None else np.ascontiguousarray(v[..., :m])) for k, v in st0.items()}
    c = run(part)
    for key in ("mom", "Egas", "Erad", "Frad"):
        assert np.array_equal(a[key], b[key]), key
        assert np.array_equal(a[key], h[key]), key
        assert np.array_equal(a[key][..., :m], c[key]), key


def test_invalid_state_left_untouched(gpu, oracle_lib):
    """A cell whose kinetic energy exceeds its total gas energy (T <= 0) is counted and left as is."""
    wl = W.workload(2, ncells=64)
    st0 = W.to_numpy(wl.make_state())
    st0["Egas"][10] = 0.5 * (st0["mom"][:, 10] ** 2).sum() / (2 * st0["rho"][10])
    ref, got, gs, os_ = run_both(gpu, oracle_lib, wl, st0, wl.dt)
    for key in ("Egas", "Erad", "Frad", "mom"):
        assert np.array_equal(got[key][..., 10], st0[key][..., 10])
        assert np.array_equal(ref[key][..., 10], st0[key][..., 10])
    assert gs["n_T_nonpositive_steps"] == os_["n_T_nonpositive_steps"] == 1
    assert_parity(ref, got, st0, wl.c, wl.c_hat, label="invalid cell")


def test_argument_errors(gpu):
    import torch

    wl = W.workload(2, ncells=32)
    dev = wl.make_state(device="cuda")
    ctx = gpu.Context.from_workload(wl)
    for bad in (dict(dt=0.0), dict(dt=-1.0), dict(c_hat=2 * wl.c), dict(c_hat=0.0), dict(c=0.0)):
        kw = dict(dt=wl.dt, c=wl.c, c_hat=wl.c_hat)
        kw.update(bad)
        with pytest.raises(gpu.MgrhdError, match="MGRHD_ERR_RANGE"):
            ctx.source_update(dev, kw["dt"], kw["c"], kw["c_hat"])
    torch.cuda.synchronize()
    ctx.free()
