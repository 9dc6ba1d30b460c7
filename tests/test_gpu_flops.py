"""The algorithmic flop counters behind `roofline.achieved`: the instrumented instantiation of
each kernel must (a) leave the results bit-identical to the plain one, and (b) return a count that lies between the
two closed forms obtained from the iteration counters with the cheapest and the dearest branch of the edge functions
(the per-piece constants are retyped here from DESIGN.md section 8, not read from the library).
"""
import numpy as np
import pytest

from paper_2407_18304_b200 import workloads as W

pytestmark = pytest.mark.gpu

# DESIGN.md section 8, retyped
EDGE_MIN, EDGE_MAX = 32, 96
GROUP, CELL_EVAL, STEP_CELL, STEP_GROUP = 39, 27, 10, 4
OUTER_CELL, OUTER_GROUP, CELL, CELL_GROUP, POW_T = 50, 102, 16, 7, 64
TAB_CELL, TAB_EDGE, TAB_ALPHA, MEANS_VAR, EQ30_FIXED, EQ30_FREE, SLOPE_FIT = 33, 35, 32, 6, 34, 66, 36
OUTER_GROUP_L, OUTER_CELL_L = 126, 107


@pytest.fixture(scope="module")
def gpu():
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device is visible")
    from paper_2407_18304_b200 import binding

    binding.load_library()
    return binding


def run(gpu, wl, st0, dt, count):
    import torch

    ctx = gpu.Context.from_workload(wl)
    dev = {k: (None if v is None else torch.from_numpy(v).cuda()) for k, v in st0.items()}
    ctx.set_flop_counting(count)
    ctx.reset_stats()
    ctx.source_update(dev, dt, wl.c, wl.c_hat)
    torch.cuda.synchronize()
    stats = ctx.get_stats()
    ctx.free()
    return W.to_numpy(dev), stats


def bounds(wl, n, stats, kind=0, spectrum=0, outer_mode=0):
    Nq = wl.Nq
    ev, tr = stats["newton_evals_total"], stats["outer_trips_total"]
    group = GROUP + (TAB_EDGE + TAB_ALPHA if kind == 2 else 0) + (MEANS_VAR if (kind == 2 or spectrum == 1) else 0) \
        + (2 * SLOPE_FIT if spectrum == 1 else 0)
    eq30 = 2 * EQ30_FREE if spectrum == 1 else (EQ30_FIXED if kind == 2 else 0)
    cell_eval = CELL_EVAL + (POW_T if kind == 1 else 0) + (TAB_CELL + TAB_EDGE if kind == 2 else 0)
    oc, og = (OUTER_CELL_L, OUTER_GROUP_L) if outer_mode == 1 else (OUTER_CELL, OUTER_GROUP)
    fixed = n * (CELL + CELL_GROUP * Nq) + tr * (oc + og * Nq)
    # every evaluation but the last of each Newton iteration is followed by a step: between ev - tr and ev steps
    lo = fixed + ev * (cell_eval + Nq * group + (Nq + 1) * EDGE_MIN) + max(ev - tr - n, 0) * (STEP_CELL + STEP_GROUP * Nq)
    hi = fixed + ev * (cell_eval + Nq * (group + eq30) + (Nq + 1) * EDGE_MAX) + ev * (STEP_CELL + STEP_GROUP * Nq)
    return lo, hi


@pytest.mark.parametrize("index,n", [(2, 2000), (4, 1500), (5, 300)])
def test_tuned_kernel_flop_counter(gpu, index, n):
    wl = W.workload(index, ncells=n)
    st0 = W.to_numpy(wl.make_state())
    dt = wl.dt_of_call(0)
    plain, s0 = run(gpu, wl, st0, dt, False)
    counted, s1 = run(gpu, wl, st0, dt, True)
    for k in ("mom", "Egas", "Erad", "Frad"):
        assert np.array_equal(plain[k], counted[k]), k
    assert s0["flops"] == 0
    assert s0["newton_evals_total"] == s1["newton_evals_total"] and s0["outer_trips_total"] == s1["outer_trips_total"]
    lo, hi = bounds(wl, n, s1)
    assert lo <= s1["flops"] <= hi, (lo, s1["flops"], hi)


@pytest.mark.parametrize("option", ["free_slope", "edge_table", "variant_L", "ktemp_L"])
def test_general_kernel_flop_counter(gpu, option):
    n = 400
    wl = W.workload(4, ncells=n)
    kind = spectrum = outer_mode = 0
    if option == "free_slope":
        wl.spectrum = spectrum = 1
    elif option == "edge_table":
        # kappa = K (T/T_ref)^-0.5 nu^-1.5 at the edges, NT points in ln T
        NT = 9
        lnT = np.linspace(np.log(0.05), np.log(20.0), NT)
        wl.opacity_kind = kind = 2
        wl.lnT0, wl.dlnT = float(lnT[0]), float(lnT[1] - lnT[0])
        wl.lnk_edge = np.ascontiguousarray(np.log(3.0) - 1.5 * np.log(wl.edges)[:, None] - 0.5 * lnT[None, :])
    elif option == "variant_L":
        wl.outer_mode = outer_mode = 1
    else:
        wl.outer_mode = outer_mode = 1
        wl.opacity_kind, wl.T_ref, wl.p_T = 1, 1.0, 1.5
        kind = 1
    st0 = W.to_numpy(wl.make_state())
    dt = wl.dt_of_call(0)
    plain, s0 = run(gpu, wl, st0, dt, False)
    counted, s1 = run(gpu, wl, st0, dt, True)
    for k in ("mom", "Egas", "Erad", "Frad"):
        assert np.array_equal(plain[k], counted[k]), k
    assert s0["flops"] == 0 and s1["flops"] > 0
    assert s0["newton_evals_total"] == s1["newton_evals_total"]
    lo, hi = bounds(wl, n, s1, kind=kind, spectrum=spectrum, outer_mode=outer_mode)
    assert lo <= s1["flops"] <= hi, (option, lo, s1["flops"], hi)
