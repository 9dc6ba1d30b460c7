"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (whole
workload in HBM, one mgrhd_source_update call): the oracle cannot run 16.7 M cells, so it is run on
sampled cells (spread over the whole index range, including the first and last cell) and compared
element by element; properties that hold at any size (conservation to round-off, finiteness, every
cell processed, nothing unconverged) are checked on the whole grid."""
import numpy as np
import pytest

from paper_2407_18304_b200 import workloads as W

from parity_util import afloor_quasi_newton, assert_parity, oracle_model

pytestmark = pytest.mark.gpu

SAMPLES = {2: 4096, 3: 2048, 4: 1536, 5: 512}


def _sample_indices(n: int, k: int):
    idx = np.unique(np.concatenate([np.linspace(0, n - 1, k - 64).astype(np.int64),
                                    np.arange(32), np.arange(n - 32, n)]))
    return idx


@pytest.mark.parametrize("index,variant", [(2, "default"), (3, "default"), (4, "default"), (5, "default"),
                                           (4, "ktemp"), (4, "source"), (3, "free_slope"), (3, "edge_table")])
def test_full_size_sampled_parity(oracle_lib, index, variant):
    """`variant`: the model options of SURVEY 8(f) as bench.py --variant builds them, at the full size of the workload."""
    import torch

    import bench

    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device is visible")
    from paper_2407_18304_b200 import binding

    wl = bench.apply_variant(W.workload(index), variant)
    n = wl.ncells
    quasi = variant in ("ktemp", "free_slope", "edge_table")
    free, _ = torch.cuda.mem_get_info()
    if free < 1.3 * wl.state_bytes() + (2 << 30):
        pytest.skip("not enough free device memory for the full-size state")
    dev = wl.make_state(device="cuda")
    if variant == "source":
        g = torch.Generator(device="cuda").manual_seed(99)
        dev["Srad"] = dev["Erad"] * (2.0 * torch.rand(dev["Erad"].shape, generator=g, device="cuda", dtype=torch.float64))
    idx = _sample_indices(n, SAMPLES[index] if variant == "default" else SAMPLES[index] // 2)
    tidx = torch.from_numpy(idx).cuda()
    take = lambda st: {k: (None if v is None else np.ascontiguousarray(v.index_select(v.dim() - 1, tidx).cpu().numpy()))
                       for k, v in st.items()}                                                  # noqa: E731
    st0 = take(dev)
    ctx = binding.Context.from_workload(wl)
    E0 = torch.empty(n, dtype=torch.float64, device="cuda")
    P0 = torch.empty(3, n, dtype=torch.float64, device="cuda")
    E1, P1 = torch.empty_like(E0), torch.empty_like(P0)
    dt = wl.dt_of_call(0)
    ctx.conserved_totals(dev, wl.c, wl.c_hat, E0, P0)
    if variant == "source":                        # conserved: E_gas + (c/c_hat) sum (E_g - S_g)
        E0 += (wl.c / wl.c_hat) * dev["Srad"].sum(0)
    Es = dev["Egas"].abs() + (wl.c / wl.c_hat) * dev["Erad"].abs().sum(0)
    Ps = dev["mom"].pow(2).sum(0).sqrt() + dev["Frad"].pow(2).sum(0).sqrt().sum(0) / (wl.c * wl.c_hat)
    ctx.source_update(dev, dt, wl.c, wl.c_hat)
    ctx.conserved_totals(dev, wl.c, wl.c_hat, E1, P1)
    torch.cuda.synchronize()
    stats = ctx.get_stats()
    # whole grid: conservation to round-off, everything finite, every cell done, nothing unconverged
    assert float(((E1 - E0).abs() / Es).max()) <= 1e-13
    dP = (P1 - P0).pow(2).sum(0).sqrt()
    assert float(torch.where(Ps > 0, dP / Ps, dP).max()) <= 1e-13
    for k in ("mom", "Egas", "Erad", "Frad"):
        assert bool(torch.isfinite(dev[k]).all()), k
    assert stats["n_cells"] == n
    assert stats["n_newton_unconverged"] == 0 and stats["n_outer_unconverged"] == 0
    assert stats["n_T_nonpositive_steps"] == 0 and stats["n_denominator_nonpositive"] == 0
    # sampled cells: element by element against the oracle
    got = take(dev)
    ref = {k: (None if v is None else v.copy()) for k, v in st0.items()}
    oracle_lib.source_update(oracle_model(oracle_lib, wl), ref, dt, wl.c, wl.c_hat)
    scale = dict(st0)
    if variant == "source":
        scale["Erad"] = st0["Erad"] + st0["Srad"]
    assert_parity({k: v for k, v in ref.items() if k != "Srad"}, got, scale, wl.c, wl.c_hat,
                  label=f"{wl.name} full size, {len(idx)} sampled cells",
                  afloor=afloor_quasi_newton(wl.newton_tol) if quasi else 1e-14)
    ctx.free()
    del dev, E0, P0, E1, P1, Es, Ps
    torch.cuda.empty_cache()


@pytest.mark.parametrize("index,ncells", [(3, 1 << 21), (4, 1 << 21), (5, 1 << 21)])
def test_chunked_distribution_is_bit_reproducible(index, ncells):
    """Sizes at which the warps take chunks from the global counter (who computes which cell then
    depends on timing): two runs give the same bits, and the first cells the same bits as a small
    run of those cells alone (one contiguous share per warp, other neighbours, other lane assignments)."""
    import torch

    if not torch.cuda.is_available():
        pytest.fail("GPU test selected but no CUDA device is visible")
    from paper_2407_18304_b200 import binding

    wl = W.workload(index, ncells=ncells)
    dt = wl.dt_of_call(0)
    pristine = wl.make_state(device="cuda")

    def run(state):
        st = {k: (None if v is None else v.clone()) for k, v in state.items()}
        ctx = binding.Context.from_workload(wl)
        ctx.source_update(st, dt, wl.c, wl.c_hat)
        torch.cuda.synchronize()
        ctx.free()
        return st

    a, b = run(pristine), run(pristine)
    m = 3001
    part = {k: (None if v is None else v[..., :m].contiguous()) for k, v in pristine.items()}
    c = run(part)
    for key in ("mom", "Egas", "Erad", "Frad"):
        assert torch.equal(a[key], b[key]), key
        assert torch.equal(a[key][..., :m], c[key]), key
