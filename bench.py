#!/usr/bin/env python
"""bench.py -- cell-updates/s of one implicit chemistry step (kr_thermochem_step) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--mode fp64|mixed] [--scaling weak|strong]
                  [--impl reference]

A "step" is one pass of the whole hot path (layout-in, thermo, rate constants, rates of progress,
Jacobian, LU + substitution, Newton loop, sub-step controller, finalise, layout-out: DESIGN.md a1-a9)
over every cell of the workload, i.e. one kr_thermochem_step call.

ONE JSON line is printed by rank 0.  Its top-level fields are the headline workload -- BASELINE.json configs[1]
(combustion-like, S = 9, R = 21, N = 10, 2^20 cells, fp64, early-exit Newton; the configuration the metric is quoted on
that fits one GPU) -- and, when no --config is given, ``"configs"`` lists the same measurements for ALL five BASELINE
configs in fp64 and for configs 3 and 4 in mixed precision (BASELINE.json: "cell-updates/s ... (fp64, mixed) and % of
FP64/HBM roofline", per config).  ``--config C [--mode M]`` measures that one workload only.

``value`` is device-timed (CUDA events around each call on the stream the library launches on, state restored and L2
flushed before each timed call, outside the events); ``e2e`` goes through kr_thermochem_step_host with pinned HOST
buffers (copies inside the timed region).  ``roofline`` is the algorithmic FP64 work (paper_2504_04941_b200/flops.py,
from the solver's own counters) over the event-timed duration, against the FP64 FMA peak measured in this run by
kr_measure_fp64_peak.  ``cpu_baseline`` / ``--impl reference`` time the CPU oracle (oracle/, test infrastructure) on a
bounded sample, on all host cores and on one thread.

``--gpus N`` with N > 1 and no torchrun environment starts N ranks itself (one process per GPU, NCCL for the counter and
time reductions only: cells are independent).  ``--scaling weak`` (default) gives every rank a
full-size, differently seeded batch; ``--scaling strong`` shards ONE full-size batch block-cyclically over the ranks
(paper_2504_04941_b200/parallel.py, shard_indices).
"""
from __future__ import annotations

import argparse
import json
import os
import socket
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
HEADLINE = 1
# every (config, precision) BASELINE.json asks for
ALL_RUNS = [(0, "fp64"), (1, "fp64"), (2, "fp64"), (3, "fp64"), (4, "fp64"), (3, "mixed"), (4, "mixed")]
MAPPING_NAMES = {1: "thread-per-cell", 2: "warp-per-cell", 3: "cta-per-cell", 4: "thread-per-cell (table)", 5: "group-per-cell (table)"}
TRAFFIC_NOTE = ("null: DRAM bytes are not measurable inside the run; the ncu --set full captures of the step kernels "
                "(dram__bytes_read.sum + dram__bytes_write.sum per launch) are under profiles/, each with its command")


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


def _oracle():
    from oracle import build as obuild
    obuild.build_oracle()
    from oracle import oracle as O
    return O


def oracle_rates(net, cells, opts, target_seconds: float, cores: int) -> dict:
    """The oracle as it stands on a bounded prefix of the workload: all host cores, then one thread."""
    O = _oracle()
    on = O.OracleNetwork(net, opts)
    n = min(cells.n_cells, 64 * cores)
    t0 = time.perf_counter()
    on.step(cells.take(slice(0, n)), n_threads=cores)
    t = max(time.perf_counter() - t0, 1e-6)
    n2 = int(min(cells.n_cells, max(n, n / t * target_seconds)))
    t0 = time.perf_counter()
    on.step(cells.take(slice(0, n2)), n_threads=cores)
    t2 = time.perf_counter() - t0
    rate_all = n2 / t2
    n1 = int(max(8, min(n2, rate_all / cores * 0.35 * target_seconds)))      # ~a third of the budget on one thread
    t0 = time.perf_counter()
    on.step(cells.take(slice(0, n1)), n_threads=1)
    t1 = time.perf_counter() - t0
    return {"value": rate_all, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {n2} cells of the same seeded workload, {t2:.1f} s, {cores} threads",
            "one_thread": {"value": n1 / t1, "unit": UNIT, "cores": 1, "sample": f"first {n1} cells, {t1:.1f} s"}}


def run_reference(args) -> None:
    """--impl reference: the CPU oracle on the host cores, bounded sample per step (rank 0 only)."""
    idx = HEADLINE if args.config is None else args.config
    cores = os.cpu_count() or 1
    net, cells, opts = w.make_config(idx, min(w.FULL_CELLS[idx], 1 << 16))
    O = _oracle()
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
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": args.scaling,
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.CONFIG_NAMES[idx], "cells_per_step": n_s, "newton": "early-exit",
                       "note": "CPU oracle (oracle/kr_oracle.cpp, -O2, std::thread over disjoint cell ranges)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"first {n_s} cells of the seeded workload per step"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def bench_one(idx: int, mode_name: str, args, ctx) -> dict:
    """Measure one (config, precision) on this rank's GPU; returns the result dict (rank 0's is printed)."""
    import torch
    import torch.distributed as dist
    from paper_2504_04941_b200 import binding as B
    from paper_2504_04941_b200 import parallel as par

    rank, world, dev = ctx["rank"], ctx["world"], ctx["dev"]
    mode = B.KR_FP64 if mode_name == "fp64" else B.KR_MIXED
    full = args.cells or w.FULL_CELLS[idx]
    net = w.make_network(idx)
    if args.scaling == "strong" and world > 1:
        # ONE full-size batch (the rank-0 seed), sharded block-cyclically: every rank draws the same batch and keeps its share
        cells = par.shard_cells(w.make_cells(idx, net, full, seed=w.BASE_SEED + 1000 + idx), rank, world)
    else:
        # weak scaling: every rank integrates a full-size, differently seeded batch (no data-path collective)
        cells = w.make_cells(idx, net, full, seed=w.BASE_SEED + 1000 + idx + 7919 * rank)
    n_cells = cells.n_cells
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
    flush = ctx["flush"]

    def restore():
        T.copy_(T0); y.copy_(y0)
        flush.zero_()

    def step(want_stats=False):
        return gn.thermochem_step_ex(n_cells, rho, T, y, cells.dt, mode, aux=aux, status=status, want_stats=want_stats)

    warm = max(args.warmup, 3)
    for _ in range(warm):
        restore(); step()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(ctx["local_rank"])
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
                       "fp64_fallback_cell_fraction": ms["n_fp64_cells"] / max(n_cells, 1),
                       "discarded_newton_per_cell": ms["n_discarded_newton"] / max(n_cells, 1),
                       "fp64_kernel": "fp64 warp-per-cell kernel on the listed cells (second launch)"}
    flops_step = F.step_flops(net, stats)
    kern_ms = float(np.mean(ms_each))                     # this rank's step
    achieved_tf = flops_step / (kern_ms * 1e-3) / 1e12
    n_aux = 0 if cells.aux is None else cells.aux.shape[0]
    bytes_step = F.step_bytes(net, n_cells, n_aux)

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
        h2d = n_cells * 8 * (2 + net.n_species + n_aux)
        d2h = n_cells * (8 * (net.n_species + net.energy_equation) + 4)
        e2e = {"value": cells_total * n_e2e / t_e2e, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "steps": n_e2e}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = oracle_rates(net, cells, opts, args.cpu_seconds, os.cpu_count() or 1)

    info = gn.info()
    peak_tf = ctx["peak_tf"]
    notes = []
    if n_cells <= 65536:
        notes.append("launch bound: two kernel launches per step on 4 096 cells (a correctness config)")
    if idx in (3, 4) or info["mapping"] in (2, 3):
        notes.append("the timed step includes the stiffest-first scheduling: cost pass, iota and a CUB radix sort (library kernels, ~0.3 % of the step)")
    if idx == 3:
        notes.append("workload deviation D2 (DESIGN.md section 4): the 140 two-body reactions are one-way, so this config has no reverse-rate exponentials")
    if idx == 4:
        notes.append("workload deviation D2 (DESIGN.md section 4): associations use A x 1e-6 and bond-like formation enthalpies")
    return {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": args.scaling, "vs_baseline": None,
        "dtype": "f64" if mode == B.KR_FP64 else "f32+f64", "data": "synthetic",
        "config": {"workload": w.CONFIG_NAMES[idx], "cells_per_gpu": n_cells, "S": net.n_species, "R": net.n_reac,
                   "N": net.n_unknowns, "dt": cells.dt, "newton": "early-exit, K<=8", "precision_mode": mode_name,
                   "retry": int(bool(args.retry)), "mapping": MAPPING_NAMES[info["mapping"]], "kernel": gn.kernel_desc(),
                   "threads_per_cell": info["threads_per_cell"], "smem_bytes_per_block": info["smem_bytes"],
                   "l2": "state restored from a pristine copy and a 256 MiB buffer written before every timed call",
                   "parallelism": f"cells sharded ({args.scaling} scaling), {world} rank(s), no data-path collective",
                   "notes": notes},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
        "roofline": {"bound": "alu", "achieved": achieved_tf, "peak": peak_tf, "unit": "TFLOP/s",
                     "frac": achieved_tf / peak_tf, "traffic": None, "traffic_note": TRAFFIC_NOTE,
                     "peak_source": "FP64 FMA peak measured in this run (kr_measure_fp64_peak); nominal 148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2",
                     "flops_per_launch": flops_step, "kernel_ms": kern_ms,
                     "hbm_bytes_per_launch": bytes_step, "hbm_gbs": bytes_step / (kern_ms * 1e-3) / 1e9},
        "cpu_baseline": cpu,
        "solver": {k: v / max(n_cells, 1) for k, v in stats.items()}, "n_failed": n_failed, "wall_s_timed_region": wall,
        "mixed": mixed_stats,
    }


def hbm_peak():
    """(GB/s, source): MEASURED_PEAKS.json's copy bandwidth (driver-written), else the profiling guide's fallback."""
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        return 6650.0, "fallback 6.65 TB/s of /opt/skills/guides/B200_PROFILING.md (MEASURED_PEAKS.json absent)"


def bench_advection(args, ctx) -> dict:
    """one stage of kr_advect_species_1d (projected PLM, eqs. 9-14) on a seeded synthetic
    1-D field with config 1's composition matrix; HBM-bound: algorithmic bytes 16 S + 24 per cell (read y, rho, mass flux;
    write y, rho) over the event-timed launch, against the measured copy bandwidth."""
    import torch
    from paper_2504_04941_b200 import binding as B
    dev = ctx["dev"]
    n = args.advect_cells
    comp = w.make_network(1).composition
    S = comp.shape[1]
    _, yb, rb, fb = w.make_advection_batch(S, comp.shape[0], 1 << 16, seed=w.BASE_SEED + 2001)
    reps = (n + yb.shape[0] - 1) // yb.shape[0]
    y = torch.tensor(yb, device=dev).repeat(reps, 1)[:n].contiguous()
    rho = torch.tensor(rb, device=dev).repeat(reps)[:n].contiguous()
    flux = torch.tensor(fb, device=dev).repeat(reps)[:n].contiguous()
    y_out = torch.empty_like(y); rho_out = torch.empty_like(rho)
    rc = B.Recon(comp)
    stream = torch.cuda.current_stream()
    dx, lam = 1.0 / n, 0.2
    run = lambda: rc.advect_species_1d(n, y, rho, flux, lam, dx, B.Recon.SCHEME_PLM_PROJECTED, True, y_out, rho_out,
                                       stream=stream.cuda_stream)
    for _ in range(3):
        run()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        ctx["flush"].zero_()
        a.record(stream); run(); b.record(stream)
    torch.cuda.synchronize()
    ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
    bytes_launch = float(n) * (16 * S + 24)
    peak, src = hbm_peak()
    gbs = bytes_launch / (ms * 1e-3) / 1e9
    return {"workload": f"advection_1d_S{S}_projected_plm", "dtype": "f64", "cells": n, "value": n / (ms * 1e-3), "unit": "cell-updates/s",
            "ms_per_launch": ms, "gpu_launches": args.steps,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": None,
                         "traffic_note": TRAFFIC_NOTE, "peak_source": src, "bytes_per_launch": bytes_launch},
            "note": "the step before the chemistry step in the paper's cycle (PAPER.md section 2.1); input larger than L2 and L2 flushed between launches"}


def bench_raytrace(args, ctx) -> dict:
    """kr_raytrace_cartesian (section 3, eqs. 24, 29-31) on config 2's mesh (256^3 cells): one
    plane-parallel ray along +x through every (y, z) column (the plane-parallel source of PAPER.md Fig. 2), two absorbers,
    four energy bins.  Algorithmic bytes: every cell's absorber densities read once and its rate coefficients written once
    (16 B per absorber and cell) plus the rays; the call also zeroes the rate field first (inside the timed region)."""
    import torch
    from paper_2504_04941_b200 import binding as B
    dev = ctx["dev"]
    nx = ny = nz = args.ray_mesh
    n_abs, n_bins = 2, 4
    case = w.make_ray_case(shape=(nx, ny, nz), n_oblique=0, n_abs=n_abs, n_bins=n_bins, seed=w.BASE_SEED + 3001, columns=True)
    t = lambda a: torch.tensor(np.ascontiguousarray(a), device=dev)
    nd = t(case["n_dens"].reshape(n_abs, -1)); k = torch.empty_like(nd)
    org, drc, L = t(case["origins"]), t(case["directions"]), t(case["L"])
    Lo = torch.empty_like(L); path = torch.empty(org.shape[0], dtype=torch.float64, device=dev)
    n_rays, n_cells = int(org.shape[0]), nx * ny * nz
    stream = torch.cuda.current_stream()
    run = lambda: B.raytrace_cartesian(case["shape"], case["spacing"], n_rays, org, drc, L, case["sigma"], nd, k, Lo, path,
                                       stream=stream.cuda_stream)
    for _ in range(3):
        run()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        ctx["flush"].zero_()
        a.record(stream); run(); b.record(stream)
    torch.cuda.synchronize()
    ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
    assert abs(float(path.min().item()) - nx * case["spacing"][0]) < 1e-9          # every ray crossed the whole mesh
    bytes_launch = float(n_cells) * 16 * n_abs + float(n_rays) * 8 * (6 + 2 * n_bins + 1)
    peak, src = hbm_peak()
    gbs = bytes_launch / (ms * 1e-3) / 1e9
    return {"workload": f"raytrace_cartesian_{nx}x{ny}x{nz}_abs{n_abs}_bins{n_bins}", "dtype": "f64", "cells": n_cells, "rays": n_rays,
            "value": n_cells / (ms * 1e-3), "unit": "cell-crossings/s", "ms_per_launch": ms, "gpu_launches": args.steps,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": None,
                         "traffic_note": TRAFFIC_NOTE, "peak_source": src, "bytes_per_launch": bytes_launch},
            "note": "the photo-reaction rate field that feeds config 2's chemistry step (PAPER.md section 3); per cell crossing "
                    "and energy bin one exp() and one expm1() in FP64, three FP64 divides per crossing (eq. 24 un-contracted, so "
                    "that the visited cells equal the oracle's); mesh larger than L2 and L2 flushed between launches"}


def bench_table_rates(args, ctx) -> dict:
    """kr_table_rates for config 2's six thermal rate laws read from tables (n_rho = 1,
    4 097 temperature nodes: 197 KB of table, resident in L2), on 2^24 cells with config 2's temperature and density
    distributions.  Algorithmic bytes: 16 in (rho, T) + 8 per table out = 64 per cell."""
    import torch
    from paper_2504_04941_b200 import binding as B
    dev = ctx["dev"]
    n = args.advect_cells
    net, cells, _ = w.make_config(2, 1 << 16)
    table = w.make_rate_table(net, [0, 1, 3, 4, 6, 7], T_range=(50.0, 2.0e5), n_T=4097)
    reps = (n + cells.n_cells - 1) // cells.n_cells
    rho = torch.tensor(cells.rho, device=dev).repeat(reps)[:n].contiguous()
    T = torch.tensor(cells.T, device=dev).repeat(reps)[:n].contiguous()
    lnk = torch.tensor(table.ln_k, device=dev)
    n_tab = int(lnk.shape[0])
    out = torch.empty((n_tab, n), dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream()
    run = lambda: B.table_rates(lnk, table.ln_rho0, table.d_ln_rho, table.ln_T0, table.d_ln_T, rho, T, out, stream=stream.cuda_stream)
    for _ in range(3):
        run()
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for a, b in ev:
        ctx["flush"].zero_()
        a.record(stream); run(); b.record(stream)
    torch.cuda.synchronize()
    ms = float(np.mean([a.elapsed_time(b) for a, b in ev]))
    bytes_launch = float(n) * (16 + 8 * n_tab)
    peak, src = hbm_peak()
    gbs = bytes_launch / (ms * 1e-3) / 1e9
    return {"workload": f"table_rates_{n_tab}x4097", "dtype": "f64", "cells": n, "value": n / (ms * 1e-3), "unit": "cells/s",
            "ms_per_launch": ms, "gpu_launches": args.steps,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak, "traffic": None,
                         "traffic_note": TRAFFIC_NOTE, "peak_source": src, "bytes_per_launch": bytes_launch},
            "note": "tabulated reaction rates at the start of the chemistry step (PAPER.md:171); two log(), six exp() and two divides "
                    "in FP64 per cell beside 64 B of traffic; input larger than L2 and L2 flushed between launches"}


def worker(args, rank: int, local_rank: int, world: int) -> None:
    import torch
    import torch.distributed as dist
    from paper_2504_04941_b200 import binding as B

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the library has no CPU path")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    B.load()
    ctx = dict(rank=rank, local_rank=local_rank, world=world, dev=dev,
               flush=torch.empty(256 << 20, dtype=torch.uint8, device=dev),       # > 126 MB L2
               peak_tf=B.measure_fp64_peak(8192))
    if args.advection_only:
        if rank == 0:
            print(json.dumps({"next": {"advection": bench_advection(args, ctx), "raytrace": bench_raytrace(args, ctx), "table_rates": bench_table_rates(args, ctx)}}), flush=True)
        return
    if args.config is not None:
        runs = [(args.config, args.mode)]
    elif world > 1 and not args.all_configs:
        runs = [(HEADLINE, "fp64")]              # scaling runs time the headline workload; --all-configs for the rest
    else:
        runs = ALL_RUNS
    results = []
    for idx, mode_name in runs:
        results.append(bench_one(idx, mode_name, args, ctx))
        torch.cuda.empty_cache()
    advection = None
    if rank == 0 and world == 1 and args.config is None and not args.no_advection:
        advection = bench_advection(args, ctx)
        raytrace = bench_raytrace(args, ctx)
        table_rates = bench_table_rates(args, ctx)
    if rank == 0:
        head = next((r for r, (i, m) in zip(results, runs) if i == HEADLINE and m == "fp64"), results[0])
        line = dict(head)
        if len(results) > 1:
            line["config"] = dict(head["config"])
            line["config"]["headline"] = ("BASELINE.json configs[1]: the configuration the base contract names for N = 1; every other "
                                          "config and both precisions are measured in the same run under \"configs\" (lowest "
                                          "roofline fraction at S >= 9: see there)")
            line["configs"] = [{"workload": r["config"]["workload"], "dtype": r["dtype"], "value": r["value"],
                                "ms_per_step": r["ms_per_step"], "roofline": r["roofline"], "e2e": r["e2e"],
                                "cpu_baseline": r["cpu_baseline"], "n_failed": r["n_failed"], "solver": r["solver"],
                                "gpu_launches": r["gpu_launches"], "clocks": r["clocks"], "mixed": r["mixed"],
                                "kernel": r["config"]["kernel"], "cells_per_gpu": r["config"]["cells_per_gpu"],
                                "notes": r["config"]["notes"]} for r in results]
            line["gpu_launches"] = int(sum(r["gpu_launches"] for r in results))
        if advection is not None:
            line["next"] = {"advection": advection, "raytrace": raytrace, "table_rates": table_rates}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def _spawn_entry(local_rank: int, args, world: int, port: int) -> None:
    os.environ.update(RANK=str(local_rank), LOCAL_RANK=str(local_rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    worker(args, local_rank, local_rank, world)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=None, help="measure this BASELINE config only (default: all of them, headline = 1)")
    ap.add_argument("--mode", default="fp64", choices=["fp64", "mixed"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"])
    ap.add_argument("--all-configs", action="store_true", help="with --gpus N > 1: measure every config, not only the headline")
    ap.add_argument("--cells", type=int, default=0, help="override the cell count (testing only)")
    ap.add_argument("--mapping", type=int, default=0, help="override the per-cell mapping (KR_MAP_*; mapping study only)")
    ap.add_argument("--threads-per-cell", type=int, default=0)
    ap.add_argument("--retry", action="store_true", help="enable the retry procedure (PAPER.md:218; study only, default options have it off)")
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="budget of the oracle timing per config")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-advection", action="store_true", help="skip the NEXT-2 advection-stage bandwidth measurement")
    ap.add_argument("--advect-cells", type=int, default=1 << 24)
    ap.add_argument("--ray-mesh", type=int, default=256, help="cells per side of the NEXT-3 ray-tracing mesh (config 2's: 256)")
    ap.add_argument("--advection-only", action="store_true", help="measure only the NEXT-2 advection stage (profiling runs)")
    args = ap.parse_args()
    under_launcher = "RANK" in os.environ and "WORLD_SIZE" in os.environ
    rank = int(os.environ.get("RANK", "0"))
    if args.impl == "reference":
        if rank == 0:
            run_reference(args)
        return
    if under_launcher:
        worker(args, rank, int(os.environ.get("LOCAL_RANK", "0")), int(os.environ["WORLD_SIZE"]))
    elif args.gpus > 1:
        # no torchrun around us: start the ranks here, one process per GPU
        import torch
        import torch.multiprocessing as mp
        n_dev = torch.cuda.device_count()
        if n_dev < args.gpus:
            raise SystemExit(f"--gpus {args.gpus} asked for, {n_dev} CUDA device(s) visible")
        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
        mp.spawn(_spawn_entry, args=(args, args.gpus, port), nprocs=args.gpus, join=True)
    else:
        worker(args, 0, 0, 1)


if __name__ == "__main__":
    main()
