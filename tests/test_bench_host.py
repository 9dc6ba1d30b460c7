"""Host-side logic of bench.py that needs no GPU: model variants, the traffic table keyed by the kernel sources'
hash, the CPU-sample plan, and the --gpus / WORLD_SIZE consistency check."""
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402
from paper_2407_18304_b200 import workloads as W  # noqa: E402


def test_variants_set_the_model_fields():
    wl = bench.apply_variant(W.workload(4, ncells=10), "ktemp")
    assert (wl.opacity_kind, wl.p_T) == (1, 1.5) and wl.name.endswith("+ktemp")
    wl = bench.apply_variant(W.workload(4, ncells=10), "free_slope")
    assert wl.spectrum == 1
    wl = bench.apply_variant(W.workload(4, ncells=10), "edge_table")
    assert wl.opacity_kind == 2 and wl.lnk_edge.shape == (33, 33) and wl.dlnT > 0
    # the table is the continuous opacity nu^-1.5 T^-0.5 at the edges
    assert np.allclose(wl.lnk_edge[:, 0], -1.5 * np.log(wl.edges) - 0.5 * wl.lnT0)
    wl = bench.apply_variant(W.workload(4, ncells=10), "default")
    assert not hasattr(wl, "spectrum") and wl.name == W.workload(4).name


def test_traffic_is_tied_to_the_kernel_sources(tmp_path, monkeypatch):
    sha = bench.kernel_source_sha()
    assert len(sha) == 16 and sha == bench.kernel_source_sha()
    prof = tmp_path / "profiles"
    prof.mkdir()
    (prof / "traffic.csv").write_text(f"wlA, 1000, 2.0e9, 3.0e9, {sha}, cap.md\nwlA, 1000, 9e9, 9e9, deadbeefdeadbeef, old.md\n"
                                      f"wlB, 10, 1, 1, deadbeefdeadbeef, old.md\n")
    monkeypatch.setattr(bench, "ROOT", str(tmp_path))
    monkeypatch.setattr(bench, "kernel_source_sha", lambda: sha)
    t, src = bench.ncu_traffic("wlA", 4000)
    assert t == 4 * 5.0e9 and src == "cap.md"            # scaled linearly in cells, the matching capture only
    assert bench.ncu_traffic("wlB", 10) == (None, None)  # a capture of other sources is not reported
    assert bench.ncu_traffic("wlC", 10) == (None, None)


def test_cpu_sample_plan_is_bounded():
    class A:
        cpu_sample_cells = None

    for idx in (1, 2, 3, 4, 5):
        wl = W.workload(idx)
        M, slabs, cores = bench.cpu_sample_plan(A, wl)
        assert 256 <= M <= wl.ncells and 1 <= slabs <= cores and M * slabs <= wl.ncells


def test_gpus_flag_must_match_world_size():
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--cells", "64"], env=env,
                       capture_output=True, text=True, timeout=300)
    assert r.returncode != 0 and "WORLD_SIZE" in (r.stderr + r.stdout)


def test_stopping_decisions_are_told_apart_from_arithmetic_differences():
    """parity_util.unexplained_cells (used by bench.py's parity sample): a result that is the oracle's own with the
    stopping thresholds moved is 'a stopping test on the other side of its threshold'; a perturbed result is not."""
    import copy

    import oracle
    from parity_util import bad_cells, oracle_model, unexplained_cells

    oracle.build()
    wl = W.workload(2, ncells=400)
    st0 = W.to_numpy(wl.make_state())
    ref = {k: (None if v is None else v.copy()) for k, v in st0.items()}
    oracle.source_update(oracle_model(oracle, wl), ref, wl.dt, wl.c, wl.c_hat)
    loose = copy.copy(wl)
    loose.newton_tol, loose.outer_tol, loose.outer_rel_tol = 2 * wl.newton_tol, 2 * wl.outer_tol, 2 * wl.outer_rel_tol
    got = {k: (None if v is None else v.copy()) for k, v in st0.items()}
    oracle.source_update(oracle_model(oracle, loose), got, wl.dt, wl.c, wl.c_hat)    # stops earlier in some cells
    assert bad_cells(ref, ref, st0, wl.c, wl.c_hat).size == 0
    early = bad_cells(ref, got, st0, wl.c, wl.c_hat, afloor=1e-17)                     # (tight floor: make some cells differ)
    assert early.size > 0
    assert unexplained_cells(oracle, wl, st0, got, wl.dt, early, afloor=1e-17).size == 0
    got["Erad"][3, 7] *= 1.0 + 1e-8                                                   # an arithmetic error
    got["mom"][1, 11] += 1e-7 * abs(got["mom"][1, 11]) + 1e-12
    cells = bad_cells(ref, got, st0, wl.c, wl.c_hat)
    assert set(cells) >= {7, 11}
    assert set(unexplained_cells(oracle, wl, st0, got, wl.dt, cells)) == {7, 11}
