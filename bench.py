"""bench.py -- throughput of mgrhd_source_update on the BASELINE.json workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 1..5] [--impl ours|reference]

One "step" = one mgrhd_source_update over the whole workload (all SURVEY section 8(a) rows:
load, Newton/outer iterations, store), starting from the same pristine state every step (the
restore is a device-to-device copy outside the timed events; it also evicts L2).  Default
workload: config 4 (256^3 cells, Nq=32, "rapidly variable opacity"), the one north_star's
target is quoted on.  Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "source-update cell-groups/sec (FP64)"
UNIT = "cell-groups/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", type=int, default=4, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--cells", type=int, default=None, help="override the workload's cell count (debugging)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--cpu-sample-cells", type=int, default=None)
    ap.add_argument("--sustained", type=int, default=0, metavar="CALLS",
                    help="BASELINE.json config 5 as stated: CALLS successive updates of the same buffers, dt varied "
                         "per call, device-timed per call, conservation residuals checked after every call")
    ap.add_argument("--variant", default="default", choices=["default", "source", "ktemp", "free_slope", "edge_table", "literal_units"],
                    help="model option on top of the workload (SURVEY 8(f) rows): S_g present; kappa (T/T_ref)^1.5; "
                         "free-slope spectrum fit; edge opacities tabulated in T with alpha from Eq. 20; the survey's "
                         "variant L: literal units a_R = c = 1 (radiation inertia q >> 1) with the implicit-in-v outer stage")
    ap.add_argument("--imex", action="store_true",
                    help="SURVEY 8(f) NEXT-3: time the explicit 1-D transport kernel (HBM roofline) and whole two-stage "
                         "IMEX steps (Eq. 35-36) on the workload read as one periodic row of cells")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def workload_label(wl) -> str:
    return f"config{wl.index}:{wl.name}"


# --------------------------------------------------------------------------------------
# clocks: sampled through NVML while the timed region runs
# --------------------------------------------------------------------------------------
class ClockSampler:
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown",
               0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting"}

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml

            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
            self._h = pynvml.nvmlDeviceGetHandleByIndex(phys)
            self._nv = pynvml
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self._h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self._nv = None

    def _run(self):
        nv = self._nv
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self._h, nv.NVML_CLOCK_SM))
                mask = nv.nvmlDeviceGetCurrentClocksEventReasons(self._h)
                for bit, name in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.02)

    def start(self):
        if self._nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

    def stop(self) -> dict:
        self._stop.set()
        if self._thread is not None:
            self._thread.join()
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# --------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py touches oracle/)
# --------------------------------------------------------------------------------------
def oracle_model(oracle, wl):
    extra = {k: getattr(wl, k) for k in ("spectrum", "opacity_kind", "T_ref", "p_T", "lnT0", "dlnT", "lnk_edge", "outer_mode") if hasattr(wl, k)}
    return oracle.OracleModel(wl.edges, wl.kappa_lo, wl.alpha, a_rad=wl.a_rad, k_B=wl.k_B, h_planck=wl.h_planck,
                              mean_mass=wl.mean_mass, gamma=wl.gamma, closure=wl.closure, newton_tol=wl.newton_tol,
                              newton_maxit=wl.newton_maxit, outer_maxit=wl.outer_maxit, outer_tol=wl.outer_tol,
                              outer_stop=wl.outer_stop, outer_rel_tol=wl.outer_rel_tol, **extra)


def default_cpu_sample(wl) -> int:
    """Cells the single-threaded oracle (dense LU, O(Nq^3) per Newton step) finishes in roughly 10-20 s."""
    return {1: 65536, 2: 65536, 3: 32768, 4: 16384, 5: 4096}[wl.index]


def time_oracle(wl, host_state: dict, dt: float) -> tuple[float, dict]:
    """Seconds for one oracle update of host_state (in place) on one host core, and its stats."""
    import oracle

    oracle.build()
    m = oracle_model(oracle, wl)
    t0 = time.perf_counter()
    st = oracle.source_update(m, host_state, dt, wl.c, wl.c_hat)
    return time.perf_counter() - t0, st


def run_reference(args) -> None:
    """--impl reference: the oracle as it stands, on the host, on a bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2407_18304_b200 import workloads as W

    wl = apply_variant(W.workload(args.workload, ncells=args.cells), args.variant)
    sample = min(wl.ncells, args.cpu_sample_cells or max(1024, default_cpu_sample(wl) // 4))
    st0 = W.to_numpy(wl.make_state(ncells=sample))
    if args.variant == "source":
        import numpy as np

        st0["Srad"] = st0["Erad"] * np.random.default_rng(1234).uniform(0.0, 2.0, st0["Erad"].shape)
    times = []
    for step in range(args.warmup + args.steps):
        st = {k: (None if v is None else v.copy()) for k, v in st0.items()}
        dt, _ = time_oracle(wl, st, wl.dt_of_call(0))
        if step >= args.warmup:
            times.append(dt)
    total = sum(times)
    value = sample * wl.Nq * args.steps / total
    desc = f"first {sample} cells of {workload_label(wl)} per step, single thread, dense LU"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_label(wl), "cells": sample, "Nq": wl.Nq},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def apply_variant(wl, variant: str):
    """Model options of SURVEY 8(f) on the shapes of the BASELINE workloads (same state recipe)."""
    import math

    import numpy as np

    if variant == "ktemp":                     # PAPER.md:499, Marshak (c): chi_g (T/T_0)^{3/2}
        wl.opacity_kind, wl.T_ref, wl.p_T = 1, 1.0, 1.5
    elif variant == "free_slope":              # Appendix A
        wl.spectrum = 1
    elif variant == "edge_table":              # Eq. 20 on a continuous opacity kappa ~ nu^-1.5 T^-0.5 (free-free-like, cf. Eq. 62)
        lnT = np.linspace(math.log(1e-2), math.log(1e2), 33)
        k_edge = wl.edges ** -1.5
        wl.opacity_kind = 2
        wl.lnk_edge = np.log(k_edge)[:, None] - 0.5 * lnT[None, :]
        wl.lnT0, wl.dlnT = float(lnT[0]), float(lnT[1] - lnT[0])
    elif variant == "literal_units":           # SURVEY 8(d) "variant L": q = (4/3) sum E_g/(rho c c_hat) up to several hundred
        wl.a_rad, wl.c, wl.dt = 1.0, 1.0, 1.0
        wl.c_hat = wl.c_hat / 1e3 if wl.c_hat < 1e3 else 1.0
        wl.outer_mode = 1
    if variant != "default":
        wl.name = f"{wl.name}+{variant}"
    return wl


def kernel_source_sha() -> str:
    """sha256 over the CUDA sources: ties an ncu traffic figure under profiles/ to the kernel it was taken from."""
    import hashlib

    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2407_18304_b200", "csrc")
    for name in sorted(os.listdir(d)):
        h.update(open(os.path.join(d, name), "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(workload_name: str, cells: int):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the update kernel from the `ncu --set full`
    capture recorded in profiles/traffic.csv (workload, cells, read bytes, write bytes, kernel source sha, file),
    scaled linearly to `cells` (persistent grid-stride kernel).  None when there is no capture of this
    workload taken from the kernel sources as they are now."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return None, None
    sha = kernel_source_sha()
    for line in open(path):
        f = [t.strip() for t in line.split(",")]
        if len(f) >= 6 and f[0] == workload_name and f[4] == sha:
            return (float(f[2]) + float(f[3])) * cells / float(f[1]), f[5]
    return None, None


# --------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------
def alloc_like(state: dict, pin: bool = False) -> dict:
    import torch

    out = {}
    for k, v in state.items():
        if v is None:
            out[k] = None
        elif pin:
            out[k] = torch.empty(v.shape, dtype=v.dtype, pin_memory=True)
        else:
            out[k] = torch.empty_like(v)
    return out


def copy_state(dst: dict, src: dict, non_blocking: bool = False) -> None:
    for k, v in src.items():
        if v is not None:
            dst[k].copy_(v, non_blocking=non_blocking)


def state_nbytes(state: dict, keys=None) -> int:
    return sum(v.numel() * 8 for k, v in state.items() if v is not None and (keys is None or k in keys))


def run_ours(args) -> None:
    import torch
    import torch.distributed as dist

    from paper_2407_18304_b200 import binding, build, workloads as W

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}: launch with torch.distributed.run "
                         f"--nproc-per-node {args.gpus} (a plain `python bench.py --gpus N` spawns it itself)")
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    binding.load_library()

    wl = apply_variant(W.workload(args.workload, ncells=args.cells), args.variant)
    n, Nq = wl.ncells, wl.Nq
    dt = wl.dt_of_call(0)
    # weak scaling: every rank updates its own n cells (disjoint seeded cell ranges); no collective on the data path
    pristine = wl.make_state(device="cuda", cell_start=rank * n, ncells=n)
    if args.variant == "source":               # S_g = E_g^(t) x U[0, 2) (seeded)
        g = torch.Generator(device="cuda").manual_seed(1234 + rank)
        pristine["Srad"] = pristine["Erad"] * (2.0 * torch.rand(pristine["Erad"].shape, generator=g, device="cuda", dtype=torch.float64))
    work = alloc_like(pristine)
    # L2: a state well above the 126 MB L2 evicts itself (and is restored from the pristine copy before every
    # step, another full sweep); smaller states get an explicit flush -- a 512 MB write -- before every timed step
    flush = None
    if state_nbytes(pristine) < (512 << 20):
        flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    ctx = binding.Context.from_workload(wl)
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- conservation + iteration statistics + algorithmic flops: one untimed instrumented pass -------
    E0 = torch.empty(n, dtype=torch.float64, device="cuda")
    P0 = torch.empty(3, n, dtype=torch.float64, device="cuda")
    E1, P1 = torch.empty_like(E0), torch.empty_like(P0)
    copy_state(work, pristine)
    ctx.conserved_totals(work, wl.c, wl.c_hat, E0, P0)
    ctx.set_flop_counting(True)
    ctx.reset_stats()
    ctx.source_update(work, dt, wl.c, wl.c_hat)
    stats = ctx.get_stats()
    ctx.set_flop_counting(False)
    ctx.conserved_totals(work, wl.c, wl.c_hat, E1, P1)
    if pristine.get("Srad") is not None:       # E_gas + (c/c_hat) sum (E_g - S_g) is what is conserved
        E0 += (wl.c / wl.c_hat) * pristine["Srad"].sum(0)
    Es = pristine["Egas"].abs() + (wl.c / wl.c_hat) * pristine["Erad"].abs().sum(0)
    resE = float(((E1 - E0).abs() / Es).max())
    Ps = pristine["mom"].pow(2).sum(0).sqrt() + pristine["Frad"].pow(2).sum(0).sqrt().sum(0) / (wl.c * wl.c_hat)
    dP = (P1 - P0).pow(2).sum(0).sqrt()
    resP = float(torch.where(Ps > 0, dP / Ps, dP).max())
    finite = all(bool(torch.isfinite(work[k]).all()) for k in ("mom", "Egas", "Erad", "Frad"))
    del E0, P0, E1, P1, Es, Ps, dP
    flops_per_launch = float(stats["flops"])

    # ---- timed region: W warm-up + K timed steps, CUDA events on the launch stream ---------------------
    launches0 = ctx.launch_count()
    for _ in range(args.warmup):
        copy_state(work, pristine)
        ctx.source_update(work, dt, wl.c, wl.c_hat)
    barrier()
    launches0 = ctx.launch_count()
    sampler = ClockSampler(local)
    sampler.start()
    evs = []
    for _ in range(args.steps):
        copy_state(work, pristine)           # untimed restore (also evicts the previous step from L2)
        if flush is not None:
            flush.fill_(1)                   # L2 flush for states that would otherwise stay resident
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        ctx.source_update(work, dt, wl.c, wl.c_hat)
        e1.record(stream)
        evs.append((e0, e1))
    barrier()
    clocks = sampler.stop()
    gpu_launches = ctx.launch_count() - launches0
    step_ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = torch.tensor([sum(step_ms)], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(total_ms, op=dist.ReduceOp.MAX)
    total_s = float(total_ms.item()) * 1e-3
    value = world * n * Nq * args.steps / total_s
    ms_per_step = 1e3 * total_s / args.steps

    # ---- roofline (rank 0's kernel): ALU-bound; HBM figures alongside ----------------------------------
    dfma = binding.measure_dfma_peak(1 << 22)              # FMA/s, measured now on this device
    peak_tflops = 2.0 * dfma / 1e12
    avg_launch_s = (sum(step_ms) / len(step_ms)) * 1e-3
    achieved_tflops = flops_per_launch / avg_launch_s / 1e12
    alg_bytes = 8.0 * n * ((5 + 4 * Nq) + (4 + 4 * Nq) + (0 if pristine["kappa_scale"] is None else 1)
                           + (Nq if pristine.get("Srad") is not None else 0))
    traffic, traffic_src = ncu_traffic(workload_label(wl), n)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    counted = flops_per_launch > 0
    roofline = {
        "bound": "alu", "achieved": achieved_tflops if counted else None, "peak": peak_tflops, "unit": "TFLOP/s",
        "frac": achieved_tflops / peak_tflops if counted else None,
        "note": None if counted else "no flop count returned by the instrumented pass",
        "traffic": traffic,
        "traffic_source": traffic_src and f"profiles/{traffic_src} (ncu --set full, scaled linearly in cells; kernel sources sha {kernel_source_sha()})",
        "peak_source": "FP64 FMA rate measured in this run by mgrhd_measure_dfma_peak (x2 flop/FMA)",
        "algorithmic_flops_per_launch": flops_per_launch,
        "algorithmic_flops_per_cell_group": flops_per_launch / (n * Nq),
        "hbm": {"achieved_gbs": alg_bytes / avg_launch_s / 1e9, "peak_gbs": hbm_peak,
                "frac": alg_bytes / avg_launch_s / 1e9 / hbm_peak, "algorithmic_bytes_per_launch": alg_bytes,
                "peak_source": "MEASURED_PEAKS.json hbm_gbs" if peaks else "fallback 6650 GB/s"},
    }

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_label(wl), "cells_per_gpu": n, "Nq": Nq, "dt": dt, "c": wl.c,
                   "c_hat": wl.c_hat, "newton_tol": wl.newton_tol, "outer_stop": wl.outer_stop,
                   "variant": args.variant,
                   "l2": ("state (%.3f GB) larger than L2; restored from a pristine copy before every step"
                          if flush is None else
                          "state (%.3f GB) fits in or near L2: flushed by a 512 MB write before every timed step")
                         % (state_nbytes(pristine) / 1e9)},
        "clocks": clocks, "gpu_launches": gpu_launches, "roofline": roofline,
        "step_ms": step_ms,
        "iterations": {"newton_evals_per_cell": stats["newton_evals_total"] / n,
                       "outer_trips_per_cell": stats["outer_trips_total"] / n,
                       "newton_evals_max": int(max(i for i, c in enumerate(stats["newton_hist"]) if c)),
                       "outer_trips_max": int(max(i for i, c in enumerate(stats["outer_hist"]) if c)),
                       "n_newton_unconverged": stats["n_newton_unconverged"],
                       "n_outer_unconverged": stats["n_outer_unconverged"],
                       "n_T_nonpositive_steps": stats["n_T_nonpositive_steps"],
                       "n_chiF_guard": stats["n_chiF_guard"],
                       "n_denominator_nonpositive": stats["n_denominator_nonpositive"]},
        "conservation": {"energy_residual_max": resE, "momentum_residual_max": resP, "all_finite": finite},
    }

    # ---- end to end through the C ABI with HOST buffers (copies inside the timed region) ---------------
    if not args.no_e2e:
        line["e2e"] = run_e2e(args, wl, ctx, pristine, dt, world, dist if world > 1 else None)

    # ---- CPU oracle beside it (rank 0, N = 1 only), with a parity check on the same cells --------------
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"], line["parity_sample"] = run_cpu_baseline(args, wl, pristine, work, dt)

    ctx.free()
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def run_e2e(args, wl, ctx, pristine, dt, world, dist):
    """The same metric through mgrhd_source_update_host: pinned HOST buffers in, HOST buffers out,
    every host<->device copy inside the timed region.  Falls back to fewer cells if the host cannot
    pin the whole state."""
    import torch

    n, Nq = wl.ncells, wl.Nq
    cells = n
    host = None
    while host is None:
        try:
            sub = {k: (None if v is None else v[..., :cells]) for k, v in pristine.items()}
            host = alloc_like(sub, pin=True)
        except RuntimeError:
            host = None
            cells //= 4
            if cells < 1024:
                return {"value": None, "unit": UNIT, "error": "could not allocate pinned host buffers"}
    sub = {k: (None if v is None else v[..., :cells]) for k, v in pristine.items()}
    times = []
    for step in range(1 + args.e2e_steps):
        copy_state(host, sub)                       # untimed: put U^(t) into the host buffers
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        t0 = time.perf_counter()
        ctx.source_update_host(host, dt, wl.c, wl.c_hat)   # synchronous: returns with U^(t+1) on the host
        t1 = time.perf_counter()
        if step >= 1:
            times.append(t1 - t0)
    t = torch.tensor([sum(times)], dtype=torch.float64, device="cuda")
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total = float(t.item())
    h2d = state_nbytes(host)
    d2h = state_nbytes(host, keys=("mom", "Egas", "Erad", "Frad"))
    return {"value": world * cells * Nq * len(times) / total, "unit": UNIT, "h2d_bytes_per_step": h2d,
            "d2h_bytes_per_step": d2h, "cells_per_gpu": cells, "steps": len(times),
            "ms_per_step": 1e3 * total / len(times), "timer": "host wall clock around the synchronous C-ABI call",
            "host_memory": "pinned"}


def cpu_sample_plan(args, wl):
    """(cells per slab, slabs): one slab per host core, each about half the single-core sample."""
    cores = max(1, len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1))
    M = min(wl.ncells, max(256, (args.cpu_sample_cells or default_cpu_sample(wl)) // 2))
    return M, max(1, min(cores, wl.ncells // M)), cores


def run_cpu_baseline(args, wl, pristine, work, dt):
    """The oracle as it stands on a bounded sample of the same state: first on ONE host core (M cells), then on
    ALL host cores (one thread per core, each its own slab of M cells, no shared state), and parity of the GPU
    result on every cell the oracle computed."""
    from concurrent.futures import ThreadPoolExecutor

    import numpy as np

    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from parity_util import afloor_quasi_newton, bad_cells, compare, unexplained_cells

    from paper_2407_18304_b200 import workloads as W

    M, slabs, cores = cpu_sample_plan(args, wl)
    # pristine / work: device or host state dicts whose first M*slabs cells are U^(t) and the GPU's U^(t+1)
    host = W.to_numpy({k: (None if v is None else v[..., :M * slabs]) for k, v in pristine.items()})
    got = W.to_numpy({k: (None if v is None else v[..., :M * slabs]) for k, v in work.items()})   # last timed step's result

    def slab(j):
        return {k: (None if v is None else v[..., j * M:(j + 1) * M].copy()) for k, v in host.items()}   # (a copy: the oracle updates in place)

    first = slab(0)
    secs1, ost = time_oracle(wl, first, dt)                      # one core
    refs = [slab(j) for j in range(slabs)]
    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=slabs) as ex:            # ctypes releases the GIL: real threads
        list(ex.map(lambda r: time_oracle(wl, r, dt), refs))
    secs_all = time.perf_counter() - t0
    ref = {k: (None if host[k] is None else np.concatenate([r[k] for r in refs], axis=-1)) for k in host}
    scale = dict(host)
    if host.get("Srad") is not None:
        scale["Erad"] = host["Erad"] + host["Srad"]
    quasi = getattr(wl, "opacity_kind", 0) != 0 or getattr(wl, "spectrum", 0) != 0
    afloor = afloor_quasi_newton(wl.newton_tol) if quasi else 1e-14      # tests/parity_util.py: why
    res = compare(ref, got, scale, wl.c, wl.c_hat, afloor=afloor)
    # cells outside the tolerance: a stopping test that fell on the other side of its threshold (the GPU's result is
    # then the oracle's with the thresholds moved by a factor <= 4), or an arithmetic difference (a failure)
    import oracle as _oracle
    out = bad_cells(ref, got, scale, wl.c, wl.c_hat, afloor=afloor)
    unexplained = unexplained_cells(_oracle, wl, host, got, dt, out, afloor=afloor) if 0 < out.size <= 64 else out
    cpu = {"value": slabs * M * wl.Nq / secs_all, "unit": UNIT, "cores": slabs, "kind": "oracle",
           "sample": f"first {slabs} x {M} cells of {workload_label(wl)}, one update each, one thread per core, dense LU",
           "seconds": secs_all, "value_1core": M * wl.Nq / secs1, "seconds_1core": secs1, "host_cores_available": cores}
    parity = {"cells": slabs * M, "tolerance": f"|d| <= 1e-10|ref| + {afloor:g} S_cell", "ok": unexplained.size == 0,
              "cells_outside_tolerance": int(out.size),
              "of_which_a_stopping_test_on_the_other_side_of_its_threshold": int(out.size - unexplained.size),
              "worst_excess_ratio": {k: v[1] for k, v in res.items()},
              "worst_relative_error_reported": {k: v[2] for k, v in res.items()},   # |d|/|ref| over |ref| > 1e-290, not gated
              "oracle_newton_evals_per_cell": ost["newton_evals_total"] / M}
    return cpu, parity


def run_sustained(args) -> None:
    """Config 5 as BASELINE.json states it: successive updates on the same buffers (no restore), dt_i = dt0 *
    10^U[-.5,.5], one CUDA-event pair per call, conservation residuals reduced on the device after every call."""
    import torch

    from paper_2407_18304_b200 import binding, build, workloads as W

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    build.build()
    wl = W.workload(5, ncells=args.cells)
    n, Nq, calls = wl.ncells, wl.Nq, args.sustained
    st = wl.make_state(device="cuda")
    ctx = binding.Context.from_workload(wl)
    stream = torch.cuda.current_stream()
    E0 = torch.empty(n, dtype=torch.float64, device="cuda")
    P0 = torch.empty(3, n, dtype=torch.float64, device="cuda")
    E1, P1 = torch.empty_like(E0), torch.empty_like(P0)
    resE = torch.zeros(calls, dtype=torch.float64, device="cuda")
    resP = torch.zeros(calls, dtype=torch.float64, device="cuda")
    M, slabs, _ = cpu_sample_plan(args, wl)
    keep0 = {k: (None if v is None else v[..., :M * slabs].clone()) for k, v in st.items()}     # U^(t) of call 0
    keep1 = None

    def counted_flops(dt_i):
        """Algorithmic flops of the update this state is about to get: instrumented pass on a clone, untimed."""
        clone = W.clone_state(st)
        ctx.set_flop_counting(True)
        ctx.reset_stats()
        ctx.source_update(clone, dt_i, wl.c, wl.c_hat)
        f = float(ctx.get_stats()["flops"])
        ctx.set_flop_counting(False)
        ctx.reset_stats()
        del clone
        return f

    flops_first = counted_flops(wl.dt_of_call(0))
    flops_last = 0.0
    sampler = ClockSampler(0)
    sampler.start()
    evs, launches0 = [], ctx.launch_count()
    for i in range(calls):
        dt = wl.dt_of_call(i)
        if i == calls - 1 and calls > 1:
            torch.cuda.synchronize()
            st_stats = ctx.get_stats()
            flops_last = counted_flops(dt)
            launches0 += 1
        ctx.conserved_totals(st, wl.c, wl.c_hat, E0, P0)
        Es = st["Egas"].abs() + (wl.c / wl.c_hat) * st["Erad"].abs().sum(0)
        Ps = st["mom"].pow(2).sum(0).sqrt() + st["Frad"].pow(2).sum(0).sqrt().sum(0) / (wl.c * wl.c_hat)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        ctx.source_update(st, dt, wl.c, wl.c_hat)
        e1.record(stream)
        evs.append((e0, e1))
        if i == 0:
            keep1 = {k: (None if v is None else v[..., :M * slabs].clone()) for k, v in st.items()}
        ctx.conserved_totals(st, wl.c, wl.c_hat, E1, P1)
        resE[i] = ((E1 - E0).abs() / Es).max()
        dP = (P1 - P0).pow(2).sum(0).sqrt()
        resP[i] = torch.where(Ps > 0, dP / Ps, dP).max()
        del Es, Ps, dP
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms = [a.elapsed_time(b) for a, b in evs]
    stats = ctx.get_stats()
    if calls > 1:                              # (the statistics were reset around the instrumented pass of the last call)
        for k in ("newton_evals_total", "outer_trips_total", "n_newton_unconverged", "n_outer_unconverged"):
            stats[k] += st_stats[k]
    total_s = sum(ms) * 1e-3
    dfma = binding.measure_dfma_peak(1 << 22)
    peak_tflops = 2.0 * dfma / 1e12
    fl = flops_last if calls > 1 else flops_first
    roofline = {"bound": "alu", "achieved": fl / (ms[-1] * 1e-3) / 1e12, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": fl / (ms[-1] * 1e-3) / 1e12 / peak_tflops, "traffic": None,
                "peak_source": "FP64 FMA rate measured in this run by mgrhd_measure_dfma_peak (x2 flop/FMA)",
                "which_call": "last call (iteration counts fall from call to call); first call alongside",
                "first_call": {"algorithmic_flops_per_cell_group": flops_first / (n * Nq),
                               "frac": flops_first / (ms[0] * 1e-3) / 1e12 / peak_tflops},
                "algorithmic_flops_per_cell_group": fl / (n * Nq)}
    cpu, parity = run_cpu_baseline(args, wl, keep0, keep1, wl.dt_of_call(0))
    line = {
        "metric": METRIC, "value": n * Nq * calls / total_s, "unit": UNIT, "n_gpus": 1, "steps": calls, "warmup": 0,
        "ms_per_step": 1e3 * total_s / calls, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_label(wl) + " (sustained: successive calls, no restore)", "cells_per_gpu": n,
                   "Nq": Nq, "c": wl.c, "c_hat": wl.c_hat, "l2": "state larger than L2"},
        "clocks": clocks, "gpu_launches": (ctx.launch_count() - launches0 - 2 * calls), "roofline": roofline,
        "cpu_baseline": cpu, "parity_sample": dict(parity, which="call 0"),
        "call_ms": {"first": ms[0], "min": min(ms), "max": max(ms), "last": ms[-1]},
        "iterations": {"newton_evals_per_cell_call": stats["newton_evals_total"] / (n * calls),
                       "outer_trips_per_cell_call": stats["outer_trips_total"] / (n * calls),
                       "n_newton_unconverged": stats["n_newton_unconverged"],
                       "n_outer_unconverged": stats["n_outer_unconverged"]},
        "conservation": {"energy_residual_max_over_calls": float(resE.max()),
                         "momentum_residual_max_over_calls": float(resP.max()),
                         "all_finite": all(bool(torch.isfinite(st[k]).all()) for k in ("mom", "Egas", "Erad", "Frad"))},
    }
    ctx.free()
    print(json.dumps(line))


def spawn_ranks(args) -> int:
    """`python bench.py --gpus N` without a launcher: start the N ranks ourselves, exactly as the driver does."""
    import socket
    import subprocess

    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_imex(args) -> None:
    """The transport kernel by itself (HBM-bound: 96 algorithmic bytes per cell-group) and the IMEX step around it."""
    import torch

    from paper_2407_18304_b200 import binding, build, workloads as W

    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    build.build()
    wl = W.workload(args.workload, ncells=args.cells)
    n, Nq = wl.ncells, wl.Nq
    pristine = wl.make_state(device="cuda")
    U, Wk = W.clone_state(pristine), W.clone_state(pristine)
    ctx = binding.Context.from_workload(wl)
    stream = torch.cuda.current_stream()
    dx = 1.0
    dt = 0.5 * dx / wl.c_hat                      # radiation CFL 0.5

    def timed(fn, reps, warm):
        for _ in range(warm):
            fn()
        torch.cuda.synchronize()
        evs = []
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream); fn(); e1.record(stream)
            evs.append((e0, e1))
        torch.cuda.synchronize()
        return [a.elapsed_time(b) for a, b in evs]

    sampler = ClockSampler(0)
    sampler.start()
    t_ms = timed(lambda: ctx.transport_add(pristine, Wk, dx, dt, wl.c, wl.c_hat, 0), max(args.steps, 5), max(args.warmup, 3))

    def step():
        copy_state(U, pristine)
        ctx.imex_step_1d(U, Wk, dx, dt, wl.c, wl.c_hat, 0)

    launches0 = ctx.launch_count()
    s_ms = timed(step, args.steps, args.warmup)
    gpu_launches = (ctx.launch_count() - launches0) * args.steps // (args.steps + args.warmup)
    clocks = sampler.stop()
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        peaks = {}
    hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
    tb = 96.0 * n * Nq                            # read u of src (4), read + write u of dst (4 + 4) doubles per cell-group
    t_avg = sum(t_ms) / len(t_ms) * 1e-3
    restore_ms = timed(lambda: copy_state(U, pristine), 3, 1)
    step_s = (sum(s_ms) / len(s_ms) - sum(restore_ms) / len(restore_ms)) * 1e-3
    line = {
        "metric": "IMEX-step cell-groups/sec (FP64; two transport sweeps + two implicit source updates, Eq. 35-36)",
        "value": n * Nq / step_s, "unit": "cell-group steps/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * step_s, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": workload_label(wl) + " as one periodic row (1-D)", "cells_per_gpu": n, "Nq": Nq,
                   "radiation_cfl": 0.5, "l2": "state larger than L2" if state_nbytes(pristine) > (512 << 20) else "state near L2 size"},
        "clocks": clocks, "gpu_launches": gpu_launches,
        "roofline": {"kernel": "transport_add_kernel", "bound": "hbm", "achieved": tb / t_avg / 1e9, "peak": hbm_peak, "unit": "GB/s",
                     "frac": tb / t_avg / 1e9 / hbm_peak, "traffic": None, "algorithmic_bytes_per_cell_group": 96,
                     "ms_per_launch": 1e3 * t_avg,
                     "peak_source": "MEASURED_PEAKS.json hbm_gbs" if peaks else "fallback 6650 GB/s"},
    }
    ctx.free()
    print(json.dumps(line))


def main():
    args = parse_args()
    if args.imex and args.impl == "ours":
        return run_imex(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours" and args.sustained == 0:
        raise SystemExit(spawn_ranks(args))
    if args.impl == "reference":
        run_reference(args)
    elif args.sustained > 0:
        run_sustained(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
