"""GPU parity of the 1-D explicit transport (Eq. 34) and of the two-stage IMEX step (Eq. 35-36) against the
oracle, through the C ABI: random rows at sizes that span several tiles with a ragged tail (and rows shorter
than a tile), both closures, both boundary conditions, reduced speed of light; the IMEX step on the shapes of
the BASELINE workloads read as 1-D rows; and section 4.2.1's moving medium stepped to its steady state."""
import numpy as np
import pytest

from paper_2407_18304_b200 import workloads as W

from parity_util import assert_parity, conservation_residual, oracle_model

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def gpu():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device is visible")
    from paper_2407_18304_b200 import binding

    binding.load_library()
    return binding


def to_dev(st):
    import torch

    return {k: (None if v is None else torch.from_numpy(np.ascontiguousarray(v)).cuda()) for k, v in st.items()}


def copy(st):
    return {k: (None if v is None else v.copy()) for k, v in st.items()}


@pytest.mark.parametrize("nx", [1, 2, 3, 4, 6, 254, 255, 508, 510, 1000 + 13, 2 * 508 + 2, 5 * 254 + 1])   # odd: one cell per thread; even: two (16-byte accesses)
@pytest.mark.parametrize("closure,bc,chat_frac", [(0, 0, 1.0), (0, 1, 0.2), (1, 0, 0.5)])
def test_transport_add_parity(gpu, oracle_lib, nx, closure, bc, chat_frac):
    import torch

    wl = W.workload(2, ncells=nx)
    wl.closure = closure
    wl.c_hat = chat_frac * wl.c
    st0 = W.to_numpy(wl.make_state())
    st0["Erad"][:, ::5] *= 3.0                       # rough profile
    st0["Frad"][:, :, 1::7] = 0.0                    # F = 0 cells (isotropic branch)
    if nx > 4:
        st0["Erad"][1, 3] = 0.0                      # E = 0
    dx, wdt = 0.7, 0.4 * 0.7 / wl.c_hat
    ref = copy(st0)
    oracle_lib.transport_add(st0, ref, closure, dx, wdt, wl.c, wl.c_hat, bc)
    ctx = gpu.Context.from_workload(wl)
    src, dst = to_dev(st0), to_dev(st0)
    ctx.transport_add(src, dst, dx, wdt, wl.c, wl.c_hat, bc)
    torch.cuda.synchronize()
    got = W.to_numpy(dst)
    ctx.free()
    scaleE = np.abs(st0["Erad"]).max(axis=1, keepdims=True)
    assert np.max(np.abs(got["Erad"] - ref["Erad"]) / scaleE) < 1e-14
    assert np.max(np.abs(got["Frad"] - ref["Frad"]) / (wl.c * scaleE[None])) < 1e-14
    for key in ("mom", "Egas", "rho"):
        assert np.array_equal(got[key], st0[key])     # gas fields: no transport term
    if nx > 3:
        assert np.abs(got["Erad"] - st0["Erad"]).max() > 0


@pytest.mark.parametrize("index,nx,bc", [(2, 3001, 0), (2, 3000, 1), (3, 1203, 1), (4, 1501, 0), (4, 1500, 0), (5, 517, 0)])
def test_imex_step_parity(gpu, oracle_lib, index, nx, bc):
    import torch

    wl = W.workload(index, ncells=nx)
    st0 = W.to_numpy(wl.make_state())
    dx = 1.0
    dt = 0.5 * dx / wl.c_hat                         # radiation CFL 0.5
    ref = copy(st0)
    os_ = oracle_lib.imex_step_1d(oracle_model(oracle_lib, wl), ref, dx, dt, wl.c, wl.c_hat, bc)
    ctx = gpu.Context.from_workload(wl)
    U, Wk = to_dev(st0), to_dev(st0)
    Wk["Erad"].fill_(float("nan"))                   # scratch content must not matter
    ctx.imex_step_1d(U, Wk, dx, dt, wl.c, wl.c_hat, bc)
    torch.cuda.synchronize()
    got = W.to_numpy(U)
    gs = ctx.get_stats()
    ctx.free()
    assert os_["n_outer_unconverged"] == 0 and os_["n_newton_unconverged"] == 0
    assert_parity(ref, got, st0, wl.c, wl.c_hat, label=f"IMEX step, config {index}")
    assert gs["n_cells"] == 2 * nx                   # two source updates
    assert abs(gs["newton_evals_total"] - os_["newton_evals_total"]) <= 0.02 * os_["newton_evals_total"]
    if bc == 0:                                      # periodic: the domain totals are conserved
        E0 = (st0["Egas"] + (wl.c / wl.c_hat) * st0["Erad"].sum(0)).sum()
        E1 = (got["Egas"] + (wl.c / wl.c_hat) * got["Erad"].sum(0)).sum()
        assert abs(E1 - E0) < 1e-12 * abs(E0)
    assert np.abs(got["Erad"] - st0["Erad"]).max() > 1e-6 * st0["Erad"].max()


def test_doppler_medium_steady_state_on_gpu(gpu, oracle_lib):
    """Section 4.2.1's setup (no hydro): 125 IMEX steps at radiation CFL 8; T against the closed form of
    tests/test_oracle_transport.py (0.768032517352...) and against the oracle run."""
    import torch

    Nq, nx = 16, 64
    edges = np.logspace(-3, 2, Nq + 1)

    class WL:
        pass

    wl = WL()
    wl.edges, wl.kappa_lo, wl.alpha, wl.Nq = edges, np.full(Nq, 1e5), np.zeros(Nq), Nq
    wl.a_rad = wl.k_B = wl.h_planck = wl.mean_mass = 1.0
    wl.gamma, wl.closure, wl.newton_tol, wl.newton_maxit, wl.outer_maxit = 5.0 / 3.0, 0, 1e-11, 50, 50
    wl.outer_tol, wl.outer_stop, wl.outer_rel_tol, wl.c, wl.c_hat = 1e-13, 1, 1e-12, 1.0, 1.0
    st0 = {"rho": np.ones(nx), "mom": np.zeros((3, nx)), "Egas": np.full(nx, 1.5 + 0.5e-6), "Erad": np.zeros((Nq, nx)),
           "Frad": np.zeros((3, Nq, nx)), "kappa_scale": None}
    st0["mom"][0] = 1e-3
    ref = copy(st0)
    m = oracle_model(oracle_lib, wl)
    ctx = gpu.Context.from_workload(wl)
    U, Wk = to_dev(st0), to_dev(st0)
    for _ in range(125):
        oracle_lib.imex_step_1d(m, ref, 1.0, 8.0, 1.0, 1.0, 0)
        ctx.imex_step_1d(U, Wk, 1.0, 8.0, 1.0, 1.0, 0)
    torch.cuda.synchronize()
    got = W.to_numpy(U)
    ctx.free()
    T = (got["Egas"] - 0.5 * (got["mom"] ** 2).sum(0)) / 1.5
    Tref = (ref["Egas"] - 0.5 * (ref["mom"] ** 2).sum(0)) / 1.5
    assert np.ptp(T) == 0.0
    assert abs(T[0] - 0.768032517352241857) < 5e-11
    assert abs(T[0] - Tref[0]) < 1e-13
    assert np.max(np.abs(got["Erad"] - ref["Erad"])) < 1e-12 * ref["Erad"].max()
    assert np.max(np.abs(got["Frad"][0] - ref["Frad"][0])) < 1e-10 * np.abs(ref["Frad"][0]).max()


def test_imex_step_with_the_general_kernel_models(gpu, oracle_lib):
    """The IMEX step dispatches its two source updates like mgrhd_source_update: free-slope spectrum (general kernel)."""
    import torch

    from parity_util import afloor_quasi_newton

    wl = W.workload(2, ncells=700)
    wl.spectrum = 1
    st0 = W.to_numpy(wl.make_state())
    dx, dt = 1.0, 0.5 / wl.c_hat
    ref = copy(st0)
    oracle_lib.imex_step_1d(oracle_model(oracle_lib, wl), ref, dx, dt, wl.c, wl.c_hat, 0)
    ctx = gpu.Context.from_workload(wl)
    U, Wk = to_dev(st0), to_dev(st0)
    ctx.imex_step_1d(U, Wk, dx, dt, wl.c, wl.c_hat, 0)
    torch.cuda.synchronize()
    got = W.to_numpy(U)
    ctx.free()
    assert_parity(ref, got, st0, wl.c, wl.c_hat, label="IMEX step, free slope", afloor=afloor_quasi_newton(wl.newton_tol))


def test_transport_argument_errors(gpu):
    import torch

    wl = W.workload(2, ncells=64)
    a, b = wl.make_state(device="cuda"), wl.make_state(device="cuda")
    ctx = gpu.Context.from_workload(wl)
    with pytest.raises(gpu.MgrhdError, match="MGRHD_ERR_ARG"):
        ctx.transport_add(a, a, 1.0, 1e-3, wl.c, wl.c_hat, 0)          # src and dst alias
    with pytest.raises(gpu.MgrhdError, match="MGRHD_ERR_ARG"):
        ctx.transport_add(a, b, 1.0, 1e-3, wl.c, wl.c_hat, 2)          # unknown boundary condition
    with pytest.raises(gpu.MgrhdError, match="MGRHD_ERR_RANGE"):
        ctx.transport_add(a, b, 0.0, 1e-3, wl.c, wl.c_hat, 0)          # dx <= 0
    with pytest.raises(gpu.MgrhdError, match="MGRHD_ERR_RANGE"):
        ctx.imex_step_1d(a, b, 1.0, 0.0, wl.c, wl.c_hat, 0)            # dt <= 0
    with pytest.raises(gpu.MgrhdError, match="MGRHD_ERR_RANGE"):
        ctx.imex_step_1d(a, b, 1.0, 1e-3, wl.c, 2 * wl.c, 0)           # c_hat > c
    src = dict(a, Srad=torch.zeros_like(a["Erad"]))
    with pytest.raises(gpu.MgrhdError, match="MGRHD_ERR_ARG"):
        ctx.imex_step_1d(src, b, 1.0, 1e-3, wl.c, wl.c_hat, 0)         # a per-update source has no place in the two stages
    torch.cuda.synchronize()
    before = {k: v.clone() for k, v in a.items() if v is not None}
    ctx.imex_step_1d(a, b, 1.0, 1e-3, wl.c, wl.c_hat, 0)               # and a valid call still works
    torch.cuda.synchronize()
    assert not torch.equal(before["Erad"], a["Erad"])
    ctx.free()
