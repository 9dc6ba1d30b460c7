"""mgrhd_source_update_static (include/mgrhd.h): the source update with its scratch and counters in static device
arrays of the library, for callers that cannot allocate device memory.  Checked against the existing path
(mgrhd_init + mgrhd_source_update) on the same inputs, two calls in a row on the same buffers, then a call with a
different group structure (so the scratch holds another layout's leftovers), the size limit, and that the device's
free memory does not move across a call.  Collected last on purpose (the suite runs with `pytest -x`).
"""
import numpy as np
import pytest

from paper_2407_18304_b200 import workloads as W

from parity_util import assert_parity

pytestmark = pytest.mark.gpu

FIELDS = ("mom", "Egas", "Erad", "Frad")
COUNTERS = ("n_cells", "n_newton_unconverged", "n_outer_unconverged", "n_T_nonpositive_steps", "n_chiF_guard",
            "n_denominator_nonpositive", "newton_evals_total", "outer_trips_total")


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

    return {k: (None if v is None else torch.from_numpy(v.copy()).cuda()) for k, v in st.items()}


def existing_path(gpu, wl, st0, dts):
    """The reference for this test: mgrhd_init + mgrhd_source_update, one call per dt on the same buffers."""
    import torch

    ctx = gpu.Context.from_workload(wl)
    dev = to_dev(st0)
    outs, stats = [], []
    for dt in dts:
        ctx.reset_stats()
        ctx.source_update(dev, dt, wl.c, wl.c_hat)
        torch.cuda.synchronize()
        outs.append(W.to_numpy(dev))
        stats.append(ctx.get_stats())
    ctx.free()
    return outs, stats


def same(gpu, wl, before, ref, got, rstats, gstats, label):
    assert_parity(ref, got, before, wl.c, wl.c_hat, label=label)        # the tolerance of the parity tests
    for k in FIELDS:                                                      # same kernel, same parameters: same bits
        assert np.array_equal(ref[k], got[k]), (label, k)
    for k in COUNTERS:
        assert rstats[k] == gstats[k], (label, k, rstats[k], gstats[k])


@pytest.mark.parametrize("index,n", [(4, 3001), (2, 5000)])
def test_static_entry_point_matches_the_existing_path_twice_in_a_row(gpu, index, n):
    import torch

    wl = W.workload(index, ncells=n)
    st0 = W.to_numpy(wl.make_state())
    dts = [wl.dt_of_call(0), 0.37 * wl.dt_of_call(0)]
    refs, rstats = existing_path(gpu, wl, st0, dts)
    dev = to_dev(st0)
    before = st0
    for call, dt in enumerate(dts):
        gstats = gpu.source_update_static(wl, dev, dt, wl.c, wl.c_hat, want_stats=True)
        got = W.to_numpy(dev)
        same(gpu, wl, before, refs[call], got, rstats[call], gstats, f"config {index}, call {call}")
        before = refs[call]
    # a third call without counters on a side stream, after the scratch has held another group structure's data
    other = W.workload(3, ncells=1500)
    gpu.source_update_static(other, to_dev(W.to_numpy(other.make_state())), other.dt, other.c, other.c_hat)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    dev = to_dev(st0)
    torch.cuda.synchronize()
    assert gpu.source_update_static(wl, dev, dts[0], wl.c, wl.c_hat, stream=side.cuda_stream) is None
    side.synchronize()
    got = W.to_numpy(dev)
    for k in FIELDS:
        assert np.array_equal(refs[0][k], got[k]), k


def test_static_entry_point_allocates_nothing_and_states_its_limit(gpu):
    import torch

    wl = W.workload(4, ncells=20000)
    dev = to_dev(W.to_numpy(wl.make_state()))
    gpu.source_update_static(wl, dev, wl.dt, wl.c, wl.c_hat)              # first call: set-up, lazy module loading
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        gpu.source_update_static(wl, dev, wl.dt, wl.c, wl.c_hat, want_stats=True)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    # Nq = 64: 256 + 24 * 16 * 256 bytes of scratch per CTA, one CTA per 64 cells up to one per SM
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    per_cta = 24 * 16 * 256
    big = W.workload(5, ncells=72 * 400)
    bdev = to_dev(W.to_numpy(big.make_state()))
    keep = W.to_numpy(bdev)
    if 256 + per_cta * min(sms, 400) > gpu.STATIC_SCRATCH_BYTES:
        with pytest.raises(gpu.MgrhdError, match="MGRHD_ERR_SIZE.*static array holds"):
            gpu.source_update_static(big, bdev, big.dt, big.c, big.c_hat)
        torch.cuda.synchronize()
        now = W.to_numpy(bdev)
        for k in FIELDS:
            assert np.array_equal(keep[k], now[k]), k                     # rejected: nothing was touched
    small = W.workload(5, ncells=72 * 100 + 5)                            # 113 CTAs: 11.1 MB, fits
    st0 = W.to_numpy(small.make_state())
    refs, rstats = existing_path(gpu, small, st0, [small.dt])
    sdev = to_dev(st0)
    gstats = gpu.source_update_static(small, sdev, small.dt, small.c, small.c_hat, want_stats=True)
    same(gpu, small, st0, refs[0], W.to_numpy(sdev), rstats[0], gstats, "config 5, 7205 cells")
    # models the tuned kernel does not run are refused, n = 0 is a no-op
    wl.spectrum = 1
    with pytest.raises(gpu.MgrhdError, match="MGRHD_ERR_ARG"):
        gpu.source_update_static(wl, dev, wl.dt, wl.c, wl.c_hat)
    wl.spectrum = 0
    one = W.workload(4, ncells=1)
    empty = {k: (None if v is None else np.ascontiguousarray(v[..., :0])) for k, v in W.to_numpy(one.make_state()).items()}
    stats = gpu.source_update_static(one, to_dev(empty), one.dt, one.c, one.c_hat, want_stats=True)
    assert stats["n_cells"] == 0
