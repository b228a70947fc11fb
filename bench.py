"""bench.py -- throughput of the MacCormack-TVD step (Eqs. 30-39) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C5|C3|C4|C2|C1] [--impl ours|reference]

One "step" is one pass of the whole hot path over the whole grid: the CFL time step (fused max-reduction
+ dt kernel) and the 4 (2-D) or 6 (3-D) operators L_z L_y L_x L_z L_y L_x, each predictor + boundary
values + corrector + TVD term + average in one kernel.  Metric (BASELINE.json): cell-updates/s, with the
achieved HBM bandwidth of the dominant kernel as a fraction of the measured copy bandwidth.

Default workload: BASELINE config C5 (3-D 1024x1024x256, 268M cells, 10.7 GB per state), the largest
3-D case and the one the north-star roofline claim is made on; --workload C3 is the largest 2-D case.
Both are far larger than the 126 MB L2, so no L2 flush is needed between steps.

Prints ONE JSON line (rank 0).  N > 1 (torchrun): one independent replica of the workload per GPU
(the north-star path is single-GPU; replicas only), weak scaling, no collective
on the data path; time = max over ranks.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2411_10372_b200 import inputs  # noqa: E402

METRIC = "cell-updates/sec per MacCormack-TVD step (achieved HBM GB/s as fraction of roofline in `roofline`)"
UNIT = "cell-updates/s"
ORACLE_RATE_EST = 2.5e5          # cell-updates/s of the single-thread oracle, used only to SIZE its sample


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C5", choices=sorted(inputs.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg")
    ap.add_argument("--no-2d", action="store_true", help="skip the extra 2-D roofline leg (C3 at its 200 steps) of the default C5 run")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--slabs", action="store_true",
                    help="N > 1 only: ONE box cut into N slabs (paper_2411_10372_b200/slab.py, halo exchange over NCCL) instead "
                         "of N replicas; strong scaling.  Built and parity-tested, never timed on more than one GPU")
    ap.add_argument("--fused-halo", action="store_true",
                    help="with --slabs: the sweep kernels push their boundary rows into the neighbours' halos themselves "
                         "(CUDA-IPC-mapped peer buffers) instead of NCCL send/recv between the launches (3-D, even nx)")
    return ap.parse_args()


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md, MEASURED_PEAKS.json absent)"


class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU every 100 ms while the timed region runs."""

    def __init__(self, index: int):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "sw_power_cap": 0x4, "hw_power_brake_slowdown": 0x80, "sync_boost": 0x10}
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for n, bit in names.items():
                    if r & bit:
                        self.reasons.add(n)
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": int(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------------
# the CPU oracle on a bounded sample of the workload (cpu_baseline leg and --impl reference)
# ---------------------------------------------------------------------------------------------------
def oracle_sample(name: str, target_cells: float):
    """A full-height window of the workload's seeded initial state holding about target_cells nodes:
    the first w columns (2-D) or w x w columns (3-D), treated as a periodic box of the same spacing."""
    grid, params, _ = inputs.config(name)
    nz = grid["nz"]
    if grid["ndim"] == 2:
        w = int(min(grid["nx"], max(16, round(target_cells / nz / 8) * 8)))
        gw = dict(grid, nx=w, lx=grid["lx"] * w / grid["nx"])
        desc = f"{name} periodic window {w}x{nz} (same spacing, recipe and seed; full height)"
    else:
        w = int(min(grid["nx"], grid["ny"], max(16, round((target_cells / nz) ** 0.5 / 8) * 8)))
        gw = dict(grid, nx=w, ny=w, lx=grid["lx"] * w / grid["nx"], ly=grid["ly"] * w / grid["ny"])
        desc = f"{name} periodic window {w}x{w}x{nz} (same spacing, recipe and seed; full height)"
    X = inputs.conduction_state(gw, params)      # same recipe, same seed; window of the same spacing
    return gw, params, X, desc


def time_oracle(name: str, steps: int, warmup: int, target_cells: float):
    """Times the oracle, as it stands (single thread), step by step.  Returns (cells/s, s/step, desc)."""
    import oracle
    oracle.build()
    gw, params, X, desc = oracle_sample(name, target_cells)
    prob = oracle.Problem(gw, params)
    cells = inputs.num_nodes(gw)
    for _ in range(warmup):
        X, _, _ = oracle.step(prob, X, 1)
    t0 = time.perf_counter()
    for _ in range(steps):
        X, _, _ = oracle.step(prob, X, 1)
    el = time.perf_counter() - t0
    assert np.all(np.isfinite(X))
    return cells * steps / el, el / steps, desc, cells


def run_reference(args):
    """--impl reference: the oracle (kind "oracle", one host core) on this arm's config and metric."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    name = args.workload
    total = max(1, args.steps + args.warmup)
    target = max(2.0e4, ORACLE_RATE_EST * 90.0 / total)       # whole run ~1.5 minutes
    value, s_per_step, desc, cells = time_oracle(name, args.steps, args.warmup, target)
    grid, params, _ = inputs.config(name)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": s_per_step * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic (seeded hydrostatic conduction state + T noise, DESIGN.md input recipe)",
        "config": workload_config(name, grid, params),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": f"{desc}; {args.steps} timed steps of {cells} cells after {args.warmup} warm-up"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def workload_config(name, grid, params):
    dims = f"{grid['nx']}x{grid['nz']}" if grid["ndim"] == 2 else f"{grid['nx']}x{grid['ny']}x{grid['nz']}"
    return {"workload": f"{name}: {grid['ndim']}-D {dims} fp64, gamma=5/3, Pr=1, Ra={params['Ra']:g}, eps=0.1, D=0.4, CFL 0.5",
            "cells": inputs.num_nodes(grid), "fields": inputs.num_fields(grid),
            "operators_per_step": 4 if grid["ndim"] == 2 else 6,
            "l2": "state (>= 2 GB) far larger than the 126 MB L2; no flush needed" if inputs.num_nodes(grid) > 3e7
                  else "state comparable to L2: cache-resident case, not a roofline claim",
            "seed": inputs.SEED}


# ---------------------------------------------------------------------------------------------------
# our arm: the CUDA path through the C ABI
# ---------------------------------------------------------------------------------------------------
def kernel_names(ndim, nx=0):
    """Kernel behind each operator (csrc/mc_tvd.cu launch_sweep): the 3-D box has its own pair, and a 2-D box
    with an even nx runs the x-sweep with two nodes per thread (k_lane2)."""
    lane, march = (("k_lane2" if nx % 2 == 0 else "k_lane"), "k_march") if ndim == 2 else ("k_lane3", "k_march3")
    return {"Lx+": f"{lane} (L_x, dir +1)", "Lx-": f"{lane} (L_x, dir -1)",
            "Ly+": f"{march} (L_y, dir +1)", "Ly-": f"{march} (L_y, dir -1)",
            "Lz+": f"{march} (L_z, dir +1)", "Lz-": f"{march} (L_z, dir -1)"}


def ncu_counters(name: str, kernel_key: str):
    """(DRAM bytes, fp64 thread instructions) per launch of ONE kernel instance -- operator and direction, e.g.
    "Lx-" (the dir -1 x-sweep is the instance that carries the fused CFL reduction) -- from the committed
    ncu --set full capture (profiles/traffic.json, copied from profiles/*_ncu_full.txt), or (None, None)."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(path):
        return None, None
    try:
        with open(path) as f:
            rec = json.load(f).get(name, {}).get(kernel_key, {})
        return rec.get("dram_bytes"), rec.get("fp64_thread_insts")
    except Exception:
        return None, None


def max_over_ranks(x: float, world: int, device: str) -> float:
    """Slowest rank's value (replicas only: the job is as slow as its slowest replica)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(world: int, cells_per_rank: int, steps: int, ms: float) -> float:
    """Whole-job cell-updates/s: every rank advanced its own replica `steps` steps in `ms` milliseconds."""
    return world * cells_per_rank * steps / (ms * 1e-3)


def roofline_of(name, grid, per_kernel, ms, steps, sm_mhz):
    """The `roofline` object of one timed run: the slowest operator kernel against the measured HBM peak, the
    whole step, every kernel's share, and the fp64-pipe view of each kernel instance from the committed ncu capture."""
    nf, N = inputs.num_fields(grid), inputs.num_nodes(grid)
    peak, peak_src = measured_peaks()
    alg_bytes = 2 * nf * 8 * N                                       # read nf + write nf doubles per node per operator
    names = kernel_names(grid["ndim"], grid["nx"])
    fp64_peak = 148 * 64 * (sm_mhz or 1965) * 1e6                    # fp64 instructions/s: 64 lanes per SM per clock
    kernels = {}
    for k, (ms_sum, cnt) in per_kernel.items():
        avg = ms_sum / cnt
        traffic, insts = ncu_counters(name, k)
        kernels[names[k]] = {"avg_ms": avg, "launches": cnt, "share_of_step": ms_sum / ms,
                             "achieved_GBps": alg_bytes / (avg * 1e-3) / 1e9,
                             "frac": alg_bytes / (avg * 1e-3) / 1e9 / peak, "traffic": traffic,
                             "fp64_per_cell": insts / N if insts else None,
                             "fp64_pipe_frac": insts / (avg * 1e-3) / fp64_peak if insts else None}
    dom = max(per_kernel, key=lambda k: per_kernel[k][0] / per_kernel[k][1])
    d = kernels[names[dom]]
    fp64 = None
    if d["fp64_per_cell"]:
        fp64 = {"thread_insts_per_launch": d["fp64_per_cell"] * N, "per_cell": d["fp64_per_cell"],
                "peak_Ginst_s": fp64_peak / 1e9, "frac": d["fp64_pipe_frac"],
                "note": "co-bound: the fp64 pipe time of this kernel is close to its HBM time (DESIGN.md 8)"}
    step_gbps = (4 if grid["ndim"] == 2 else 6) * alg_bytes * steps / (ms * 1e-3) / 1e9
    return {"bound": "hbm", "kernel": names[dom], "achieved": d["achieved_GBps"], "peak": peak, "unit": "GB/s",
            "frac": d["frac"], "traffic": d["traffic"], "fp64_pipe": fp64, "peak_source": peak_src,
            "algorithmic_bytes_per_launch": alg_bytes, "algorithmic_bytes_per_cell_per_operator": 2 * nf * 8,
            "whole_step_achieved_GBps": step_gbps, "whole_step_frac": step_gbps / peak, "kernels": kernels}


def timed_run(binding, torch, name, steps, warmup, local, barrier, h_in=None):
    """W warm-up steps, then exactly K timed steps of workload `name` with the state resident in HBM; CUDA events on
    the library's stream around the region and around every operator launch; clocks sampled meanwhile."""
    grid, params, _ = inputs.config(name)
    if h_in is None:
        h_in = torch.from_numpy(inputs.conduction_state(grid, params).reshape(-1))
    solver = binding.MCTVD(grid, params, h_in, device=f"cuda:{local}")
    solver.step(warmup)
    barrier()
    l0 = solver.launch_count()
    solver.timing_enable(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clocks:
        barrier()
        e0.record(solver.stream)
        solver.step(steps)
        e1.record(solver.stream)
        barrier()
    ms = e0.elapsed_time(e1)
    launches = solver.launch_count() - l0
    per_kernel = solver.timing_read()
    solver.timing_enable(False)
    return solver, grid, params, ms, launches, per_kernel, clocks.summary()


def _oracle_worker(job):
    name, steps, warmup, target = job
    return time_oracle(name, steps, warmup, target)


def oracle_all_cores(name, steps, warmup, target):
    """The oracle as it stands (single-threaded C), one independent instance per host core on the same sample,
    started together: whole-host cell-updates/s = instances x cells x steps / slowest instance's time."""
    import multiprocessing as mp
    cores = os.cpu_count() or 1
    with mp.get_context("spawn").Pool(cores) as pool:
        res = pool.map(_oracle_worker, [(name, steps, warmup, target)] * cores)
    s_per_step = max(r[1] for r in res)
    return cores * res[0][3] / s_per_step, cores, res[0][2], res[0][3], s_per_step


def run_ours(args):
    import torch
    import torch.distributed as dist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (sm_100a); there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    from paper_2411_10372_b200 import binding
    name = args.workload
    grid, params, _ = inputs.config(name)
    nf, N = inputs.num_fields(grid), inputs.num_nodes(grid)
    state_bytes = nf * N * 8
    X0 = inputs.conduction_state(grid, params)                       # host, seeded (identical on every rank)
    h_in = torch.from_numpy(X0.reshape(-1))
    del X0
    try:
        h_in = h_in.pin_memory()
        h_out = torch.empty_like(h_in).pin_memory()
        pinned = True
    except Exception:
        h_out = torch.empty_like(h_in)
        pinned = False

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput: W warm-up steps, then exactly K timed steps ------------------
    solver, grid, params, ms, launches, per_kernel, clock_sum = timed_run(binding, torch, name, args.steps, args.warmup,
                                                                           local, barrier, h_in)
    dt_now = solver.dt()                                             # raises if the state went non-finite
    diag, *_ = solver.diagnostics()
    torch.cuda.synchronize()
    t_d = time.perf_counter()
    diag, *_ = solver.diagnostics()                                  # synchronises: plane sums + finish + D2H
    diag_ms = (time.perf_counter() - t_d) * 1e3

    ms_max = max_over_ranks(ms, world, f"cuda:{local}")
    value = job_value(world, N, args.steps, ms_max)

    # ---- end to end through the public host-buffer call (H2D + steps + D2H inside the timed region) --
    e2e = None
    if not args.no_e2e:
        n_e2e = max(1, args.e2e_steps)
        solver.step_host(h_in, h_out, 1)                             # warm-up of the copy path
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            solver.step_host(h_in, h_out, 1)                         # synchronises internally
        barrier()
        el = time.perf_counter() - t0
        el_max = max_over_ranks(el, world, f"cuda:{local}")
        e2e = {"value": job_value(world, N, n_e2e, el_max * 1e3), "unit": UNIT,
               "h2d_bytes_per_step": state_bytes, "d2h_bytes_per_step": state_bytes,
               "steps": n_e2e, "ms_per_step": el_max / n_e2e * 1e3,
               "call": "mc_tvd_step_host(h_in, h_out, 1): H2D of the state, dt reduction, 1 step, D2H of the state",
               "host_memory": "pinned" if pinned else "pageable"}
    solver.close()
    del solver, h_in, h_out
    torch.cuda.empty_cache()

    # ---- the other roofline case of north_star: the largest 2-D grid (C3) at the config's own step count ----
    roofline_2d = None
    if world == 1 and name == "C5" and not args.no_2d:
        s2, g2, p2, ms2, l2, pk2, clk2 = timed_run(binding, torch, "C3", inputs.CONFIGS["C3"]["steps"], max(3, args.warmup),
                                                    local, barrier)
        dt2 = s2.dt()
        s2.close()
        del s2
        torch.cuda.empty_cache()
        st2 = inputs.CONFIGS["C3"]["steps"]
        roofline_2d = {"config": workload_config("C3", g2, p2), "steps": st2, "ms_per_step": ms2 / st2,
                       "value": inputs.num_nodes(g2) * st2 / (ms2 * 1e-3), "unit": UNIT, "gpu_launches": int(l2),
                       "clocks": clk2, "roofline": roofline_of("C3", g2, pk2, ms2, st2, clk2.get("sm_mhz")),
                       "state_check": {"dt": dt2}}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic (seeded hydrostatic conduction state + T noise, DESIGN.md input recipe)",
        "config": workload_config(name, grid, params),
        "clocks": clock_sum, "gpu_launches": int(launches),
        "roofline": roofline_of(name, grid, per_kernel, ms, args.steps, clock_sum.get("sm_mhz")),
        "diagnostics_ms": diag_ms,
        "state_check": {"dt": dt_now, "nu_bar": diag["nu_bar"], "min_rho": diag["min_rho"], "min_T": diag["min_T"],
                        "steps_taken": diag["step"]},
    }
    if roofline_2d is not None:
        line["roofline_2d"] = roofline_2d
    if e2e is not None:
        line["e2e"] = e2e
    if world == 1 and not args.no_cpu_baseline:
        target = ORACLE_RATE_EST * 6.0                                # ~6 s per oracle step, 1 warm-up + 2 timed
        v, s_per_step, desc, cells = time_oracle(name, 2, 1, target)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"{desc}; 2 timed steps of {cells} cells after 1 warm-up, {s_per_step:.1f} s/step"}
        va, cores, desc, cells, sps = oracle_all_cores(name, 2, 1, target)
        line["cpu_baseline_all_cores"] = {"value": va, "unit": UNIT, "cores": cores, "kind": "oracle, one independent instance per core",
                                          "sample": f"{cores} x ({desc}); 2 timed steps after 1 warm-up, slowest instance {sps:.1f} s/step"}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_slabs(args):
    """--slabs under torchrun: the workload's ONE box as N slabs, one per GPU, halo exchange and the dt
    all-reduce inside the timed region.  value = cells of the whole box x steps / slowest rank's device time."""
    import torch
    import torch.distributed as dist

    world, rank, local = int(os.environ["WORLD_SIZE"]), int(os.environ["RANK"]), int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2411_10372_b200 import binding, slab
    name = args.workload
    grid, params, _ = inputs.config(name)
    X0 = inputs.conduction_state(grid, params)
    drv = slab.make_dist_driver(binding, grid, params, X0, device=f"cuda:{local}", fused=args.fused_halo)
    del X0
    drv.step(args.warmup)
    dist.barrier(); torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clocks:
        e0.record(drv.ranks[0].stream)
        drv.step(args.steps)
        e1.record(drv.ranks[0].stream)
        dist.barrier(); torch.cuda.synchronize()
    ms = max_over_ranks(e0.elapsed_time(e1), world, f"cuda:{local}")
    dt_now = drv.dt()
    if rank == 0:
        N = inputs.num_nodes(grid)
        print(json.dumps({
            "metric": METRIC, "value": N * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64",
            "data": "synthetic (seeded hydrostatic conduction state + T noise, DESIGN.md input recipe)",
            "config": dict(workload_config(name, grid, params), decomposition=f"{world} slabs along {slab.slab_axis(grid)}, halo 2, "
                           + ("halo rows pushed by the sweep kernels into the neighbours' buffers (CUDA IPC), a barrier per operator"
                              if args.fused_halo else "exchange after every operator (NCCL send/recv)") + ", dt all-reduce"),
            "clocks": clocks.summary(), "gpu_launches": int(drv.ranks[0].launch_count()), "state_check": {"dt": dt_now}}), flush=True)
    dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.slabs and "WORLD_SIZE" in os.environ:            # under torchrun (any world size, 1 included)
        run_slabs(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
