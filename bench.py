#!/usr/bin/env python
"""bench.py -- cell-updates/s of one implicit chemistry step (kr_thermochem_step) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--mode fp64|mixed] [--impl reference]

A "step" is one pass of the whole hot path (layout-in, thermo, rate constants, rates of progress,
Jacobian, LU + substitution, Newton loop, sub-step controller, finalise, layout-out: DESIGN.md a1-a9)
over every cell of the workload, i.e. one kr_thermochem_step call.  Default workload: BASELINE.json
configs[1] (combustion-like, S = 9, R = 21, N = 10, 2^20 cells, fp64, early-exit Newton), seeded synthetic.

One JSON line is printed by rank 0.  ``value`` is device-timed (CUDA events around each call, state
restored and L2 flushed before each timed call, outside the events); ``e2e`` goes through
kr_thermochem_step_host with pinned HOST buffers (copies inside the timed region).  ``roofline`` is the
algorithmic FP64 work (paper_2504_04941_b200/flops.py, from the solver's own counters) over the kernel's
event-timed duration, against the FP64 FMA peak measured in this run by kr_measure_fp64_peak.
``--impl reference`` times the CPU oracle (oracle/, test infrastructure) on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2504_04941_b200 import flops as F          # noqa: E402
from paper_2504_04941_b200 import workloads as w      # noqa: E402

METRIC = "cell-updates/s for one implicit chem step"
UNIT = "cell-updates/s"

# DRAM traffic of the step kernel per cell-update, from the ncu --set full captures summarised under profiles/
# (dram__bytes_read.sum + dram__bytes_write.sum of one launch / cells of that launch).  It is BELOW the algorithmic
# bytes because the results of the last cells are still in the 126 MB L2 when the kernel ends.
NCU_DRAM_BYTES_PER_CELL = {("c1", "fp64"): 130.2, ("c3", "fp64"): 285.8}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period: float = 0.05):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._halt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20,
                 "hw_power_brake_slowdown": 0x80, "applications_clocks_setting": 0x2}
        while not self._halt.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self) -> dict:
        self._halt.set()
        if self.is_alive():
            self.join(timeout=2.0)
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def oracle_sample_rate(net, cells, opts, target_seconds: float, cores: int):
    """Time the oracle as it stands on a bounded prefix of the workload; returns (cells/s, n_sample, seconds)."""
    from oracle import build as obuild
    obuild.build_oracle()
    from oracle import oracle as O
    on = O.OracleNetwork(net, opts)
    n = min(cells.n_cells, 64 * cores)
    t0 = time.perf_counter()
    on.step(cells.take(slice(0, n)), n_threads=cores)
    t = max(time.perf_counter() - t0, 1e-6)
    n2 = int(min(cells.n_cells, max(n, n / t * target_seconds)))
    t0 = time.perf_counter()
    on.step(cells.take(slice(0, n2)), n_threads=cores)
    t2 = time.perf_counter() - t0
    return n2 / t2, n2, t2


def run_reference(args, rank: int, world: int) -> None:
    """--impl reference: the CPU oracle on the host cores, bounded sample per step (rank 0 only)."""
    if rank != 0:
        return
    cores = os.cpu_count() or 1
    net, cells, opts = w.make_config(args.config, min(w.FULL_CELLS[args.config], 1 << 16))
    from oracle import build as obuild
    obuild.build_oracle()
    from oracle import oracle as O
    on = O.OracleNetwork(net, opts)
    n = min(cells.n_cells, 64 * cores)
    t0 = time.perf_counter()
    on.step(cells.take(slice(0, n)), n_threads=cores)
    rate = n / max(time.perf_counter() - t0, 1e-6)
    budget = 120.0 / max(args.steps + args.warmup, 1)                 # whole run within a few minutes
    n_s = int(max(cores, min(cells.n_cells, rate * min(budget, 10.0))))
    sample = cells.take(slice(0, n_s))
    for _ in range(args.warmup):
        on.step(sample, n_threads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        on.step(sample, n_threads=cores)
    dt = time.perf_counter() - t0
    value = n_s * args.steps / dt
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.CONFIG_NAMES[args.config], "cells_per_step": n_s, "newton": "early-exit",
                       "note": "CPU oracle (oracle/kr_oracle.cpp, -O2, std::thread over disjoint cell ranges)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"first {n_s} cells of the seeded workload per step"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--mode", default="fp64", choices=["fp64", "mixed"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cells", type=int, default=0, help="override the cell count (testing only)")
    ap.add_argument("--mapping", type=int, default=0, help="override the per-cell mapping (KR_MAP_*; mapping study only)")
    ap.add_argument("--threads-per-cell", type=int, default=0)
    ap.add_argument("--retry", action="store_true", help="enable the retry procedure (PAPER.md:218; study only, default options have it off)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_2504_04941_b200 import binding as B
    from paper_2504_04941_b200 import parallel as par

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    B.load()

    idx = args.config
    mode = B.KR_FP64 if args.mode == "fp64" else B.KR_MIXED
    n_cells = args.cells or w.FULL_CELLS[idx]
    net = w.make_network(idx)
    # weak scaling: every rank integrates a full-size, differently seeded batch (cells are independent:
    # no data-path collective)
    cells = w.make_cells(idx, net, n_cells, seed=w.BASE_SEED + 1000 + idx + 7919 * rank)
    opts = w.default_opts(idx, fixed_newton=0)
    if args.retry:
        opts.retry = 1
    gn = B.Network(net, opts)
    if args.mapping:
        gn.set_mapping(args.mapping, args.threads_per_cell)
    stream = torch.cuda.current_stream()
    gn.set_stream(stream.cuda_stream)

    rho = torch.tensor(cells.rho, device=dev)
    T0 = torch.tensor(cells.T, device=dev)
    y0 = torch.tensor(cells.y, device=dev)
    aux = None if cells.aux is None else torch.tensor(cells.aux, device=dev)
    T = T0.clone(); y = y0.clone()
    status = torch.zeros(n_cells, dtype=torch.int32, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)       # > 126 MB L2

    def restore():
        T.copy_(T0); y.copy_(y0)
        flush.zero_()

    def step(want_stats=False):
        return gn.thermochem_step_ex(n_cells, rho, T, y, cells.dt, mode, aux=aux, status=status, want_stats=want_stats)

    peak_tf = B.measure_fp64_peak(8192)
    for _ in range(max(args.warmup, 3)):
        restore(); step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    torch.cuda.synchronize()
    wall0 = time.perf_counter()
    launches = 0
    for k in range(args.steps):
        restore()
        ev[k][0].record(stream)
        step()
        ev[k][1].record(stream)
        launches += gn.last_launch_count()
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    clocks = sampler.stop()
    if world > 1:
        dist.barrier()
    ms_each = [a.elapsed_time(b) for a, b in ev]
    ms_total = par.max_over_ranks(float(sum(ms_each)))
    cells_total = par.sum_over_ranks(float(n_cells)) if world > 1 else float(n_cells)
    ms_per_step = ms_total / args.steps
    value = cells_total / (ms_per_step * 1e-3)

    # counters of one (untimed) step -> algorithmic flops
    restore()
    stats = step(want_stats=True)
    n_failed = stats["n_failed"]
    mixed_stats = None
    if mode == B.KR_MIXED:
        ms = gn.last_mixed_stats()
        mixed_stats = {"refinements_per_newton": ms["n_refine"] / max(stats["n_newton"], 1),
                       "fp64_fallback_cell_fraction": ms["n_fp64_cells"] / n_cells,
                       "fp64_kernel": "register-tile fp64 kernel on the listed cells (second launch)"}
    flops_step = F.step_flops(net, stats)
    kern_ms = float(np.mean(ms_each))                     # this rank's kernel: one launch per step
    achieved_tf = flops_step / (kern_ms * 1e-3) / 1e12
    bytes_step = F.step_bytes(net, n_cells, 0 if cells.aux is None else cells.aux.shape[0])

    # end to end: pinned host buffers through kr_thermochem_step_host
    e2e = None
    if not args.no_e2e:
        hp = dict(rho=torch.tensor(cells.rho).pin_memory(), T=torch.tensor(cells.T).pin_memory(),
                  y=torch.tensor(cells.y).pin_memory(), st=torch.zeros(n_cells, dtype=torch.int32).pin_memory(),
                  aux=None if cells.aux is None else torch.tensor(cells.aux).pin_memory())
        T_h0 = torch.tensor(cells.T); y_h0 = torch.tensor(cells.y)
        n_e2e = max(1, min(args.steps, 3))
        t_e2e = 0.0
        for k in range(1 + n_e2e):
            hp["T"].copy_(T_h0); hp["y"].copy_(y_h0)
            torch.cuda.synchronize()
            if world > 1:
                dist.barrier()
            t0 = time.perf_counter()
            gn.thermochem_step_host(n_cells, hp["rho"], hp["T"], hp["y"], cells.dt, mode, aux=hp["aux"], status=hp["st"])
            if k > 0:
                t_e2e += time.perf_counter() - t0
        t_e2e = par.max_over_ranks(t_e2e)
        n_aux = 0 if cells.aux is None else cells.aux.shape[0]
        h2d = n_cells * 8 * (2 + net.n_species + n_aux)
        d2h = n_cells * (8 * (net.n_species + net.energy_equation) + 4)
        e2e = {"value": cells_total * n_e2e / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "steps": n_e2e}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cores = os.cpu_count() or 1
        rate, n_s, secs = oracle_sample_rate(net, cells, opts, 12.0, cores)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {n_s} cells of the same seeded workload, {secs:.1f} s, {cores} threads"}

    if rank == 0:
        info = gn.info()
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if mode == B.KR_FP64 else "f32+f64", "data": "synthetic",
            "config": {"workload": w.CONFIG_NAMES[idx], "cells_per_gpu": n_cells, "S": net.n_species, "R": net.n_reac,
                       "N": net.n_unknowns, "dt": cells.dt, "newton": "early-exit, K<=8", "precision_mode": args.mode, "retry": int(bool(args.retry)),
                       "mapping": {1: "thread-per-cell", 2: "warp-per-cell", 3: "cta-per-cell", 4: "thread-per-cell (table)",
                                   5: "group-per-cell (table)"}[info["mapping"]],
                       "kernel": gn.kernel_desc(),
                       "threads_per_cell": info["threads_per_cell"], "smem_bytes_per_block": info["smem_bytes"],
                       "l2": "state restored from a pristine copy and a 256 MiB buffer written before every timed call",
                       "parallelism": f"cells sharded, {world} rank(s), no data-path collective"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
            "roofline": {"bound": "alu", "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s",
                         "frac": achieved_tf / peak_tf,
                         "traffic": (NCU_DRAM_BYTES_PER_CELL[(f"c{idx}", args.mode)] * n_cells
                                     if (f"c{idx}", args.mode) in NCU_DRAM_BYTES_PER_CELL else None),
                         "peak_source": "FP64 FMA peak measured in this run (kr_measure_fp64_peak); nominal 148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2",
                         "flops_per_launch": flops_step, "kernel_ms": kern_ms,
                         "hbm_bytes_per_launch": bytes_step, "hbm_gbs": bytes_step / (kern_ms * 1e-3) / 1e9},
            "cpu_baseline": cpu,
            "solver": {k: v / n_cells for k, v in stats.items()}, "n_failed": n_failed, "wall_s_timed_region": wall,
            "mixed": mixed_stats,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
