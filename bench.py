#!/usr/bin/env python
"""bench.py -- measures BASELINE.json's metric: FP64 grid-point RK4 updates/s of the fused CLTx hot path
(curl J1 + fused RHS/RK4 kernels) on config 4 (512 x 64 x 512), and the achieved fraction of the HBM roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 4]

One "step" = one classical RK4 step = 4 x (curl_J1 + fused RHS) over the whole grid = all rows of SURVEY 8(a).
Multi-GPU: the path does not shard in this round (north_star: one GPU, no halo exchange) -- "replicas only":
N ranks run N independent replicas, value = sum of the replicas' updates / max-over-ranks time.
--impl reference times the CPU oracle (oracle/) on the same configuration (whole RK4 steps of config 4; the number of
timed steps is cut if the box's cores would need more than a few minutes), rank 0 only.
Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "FP64 grid-point RK4 updates/sec"
UNIT = "updates/s"
# Algorithmic HBM traffic per grid point.  SURVEY 8(d) counts 164 doubles per RK4 step for the
# textbook accumulator schedule (27 + 43 + 43 + 27 through the fused kernel + 4 x 6 through the curl).  The library
# uses a reduced schedule that rebuilds the partial sums from stage states it reads anyway: 19 + 35 + 27 + 35 + 4 x 6
# = 140 doubles.  Roofline fractions use the bytes the launches REALLY have to move (the reduced schedule); the
# SURVEY-equivalent figure is reported next to them.
RHS_DOUBLES = {1: 19, 2: 35, 3: 27, 4: 35}   # per point per launch of the fused RHS+RK4 kernel
CURL_DOUBLES = 6
BYTES_PER_UPDATE = (sum(RHS_DOUBLES.values()) + 4 * CURL_DOUBLES) * 8      # 140 doubles = 1120 B
SURVEY_BYTES_PER_UPDATE = 164 * 8


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)).get("hbm_gbs"), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def profiled_pipes(kernel="rhs_tma"):
    """FP64-pipe and L1/shared-memory utilisation of the dominant kernel from the same committed ncu capture (mean over
    its launches), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        for line in open(p).read().splitlines()[1:]:
            f = line.split(",")
            if f[0] == kernel and len(f) >= 5:
                return {"fp64_pipe_pct": float(f[3]), "l1tex_throughput_pct": float(f[4]), "source": f[2]}
    except Exception:
        pass
    return None


def profiled_traffic(kernel="rhs_tma"):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed ncu --set full
    summary (profiles/traffic.csv names the source file); None if there is no capture."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        for line in open(p).read().splitlines()[1:]:
            f = line.split(",")
            if f[0] == kernel:
                return float(f[1])
    except Exception:
        pass
    return None


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def oracle_rate(index, steps, warmup=0, budget_seconds=0.0):
    """Times the CPU oracle as it stands on BASELINE.json config `index` (same seeded inputs as the GPU arm).
    budget_seconds > 0: the first step is timed alone and the number of timed steps is cut so that the whole call stays
    within the budget (the grid is never shrunk: the sample is whole RK4 steps of the named configuration)."""
    import oracle as orc
    from paper_1812_00525_b200 import inputs
    prob = inputs.make_problem(index)
    c = prob.cfg
    o = orc.Oracle(c.nR, c.nphi, c.nZ, c.Rmin, c.Rmax, c.Zmin, c.Zmax, c.phi_extent, gamma=c.gamma, eta=c.eta, nu=c.nu,
                   D=c.D, kappa=c.kappa, dt=prob.dt)
    o.set_equilibrium(prob.U0)
    o.set_state(prob.U)
    asked = steps
    if warmup:
        t0 = time.perf_counter()
        o.step(1)
        t1 = time.perf_counter() - t0
        if budget_seconds > 0:
            warmup = max(1, min(warmup, int(0.15 * budget_seconds / t1)))
        if warmup > 1:
            o.step(warmup - 1)
    t0 = time.perf_counter()
    o.step(1)
    first = time.perf_counter() - t0
    if budget_seconds > 0:
        steps = max(1, min(steps, int(0.8 * budget_seconds / first)))
    if steps > 1:
        o.step(steps - 1)
    dt = time.perf_counter() - t0
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    cut = "" if steps == asked else f" (of {asked} asked: cut to stay within {budget_seconds:.0f} s)"
    return {"value": c.interior * steps / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "config_index": index,
            "sample": f"{steps} RK4 step(s){cut} of config {index} itself, {c.nR}x{c.nphi}x{c.nZ} ({c.interior} interior nodes), "
                      f"oracle/clt_oracle.c as it stands (gcc -O2 -ffp-contract=off, OpenMP over nodes, {cores} thread(s))",
            "seconds": dt, "ms_per_step": 1e3 * dt / steps, "steps": steps}


def oracle_rate_single_thread(index, steps):
    """The same measurement with OMP_NUM_THREADS=1 (single-threaded on config 2), in a worker process
    because the OpenMP runtime reads the variable once."""
    env = dict(os.environ, OMP_NUM_THREADS="1")
    try:
        r = subprocess.run([sys.executable, os.path.abspath(__file__), "--oracle-worker", f"{index},{steps}"], env=env,
                           capture_output=True, text=True, timeout=600)
        return json.loads(r.stdout.strip().splitlines()[-1])
    except Exception as e:      # a baseline figure, never a reason to lose the bench line
        return {"error": repr(e)}


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the configuration the GPU arm measures (config 4 by default)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    r = oracle_rate(args.config, args.steps, args.warmup, budget_seconds=args.reference_budget)
    from paper_1812_00525_b200 import inputs
    cfg = inputs.CONFIGS[args.config]
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config {cfg.index}: {cfg.nR}x{cfg.nphi}x{cfg.nZ} (R x phi x Z), {cfg.interior} interior nodes, "
                                   f"seeded reference state + perturbations (BASELINE.json configs[{cfg.index - 1}])",
                       "timed_steps": r["steps"], "sample": r["sample"]},
            "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_slabs(args):
    """NEXT-4 measurement: the same workload cut into Z-slabs (paper_1812_00525_b200/slab.py).  --slabs K with one
    process = K sub-domain contexts on ONE GPU, a stream each (measures the cost of the decomposition itself:
    redundant ghost-row work, no link); under torchrun (--gpus N > 1) = one slab per rank, strong scaling,
    ghost rows over NCCL.  Not the contract's default (north_star: replicas only)."""
    import torch
    import torch.distributed as dist
    from paper_1812_00525_b200 import build as clt_build
    from paper_1812_00525_b200 import inputs, replicas, slab
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        clt_build.build()
    if world > 1:
        dist.barrier()
    prob = inputs.make_problem(args.config)
    cfg = prob.cfg
    nslabs = world if world > 1 else args.slabs
    grp = slab.SlabGroup(cfg, prob.dt, prob.U0, prob.U, nslabs, devices=(f"cuda:{local}",), dist=dist if world > 1 else None,
                         d_i=args.d_i, phi_scheme=args.phi_scheme)
    grp.step(args.warmup)
    replicas.barrier(f"cuda:{local}")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stream = grp.slabs[0].g.torch_stream
    grp.join()
    e0.record(stream)
    grp.step(args.steps)
    grp.join()               # in-process slabs run on a stream each: the first one's waits for the others
    e1.record(stream)
    replicas.barrier(f"cuda:{local}")
    ms = e0.elapsed_time(e1)
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device=f"cuda:{local}")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    d = grp.diagnostics()
    if rank == 0:
        line = {"metric": METRIC, "value": cfg.interior * args.steps / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": f"config {cfg.index}: {cfg.nR}x{cfg.nphi}x{cfg.nZ}, cut into {nslabs} Z-slabs with 4 ghost rows per cut",
                           "parallelism": f"{nslabs} slabs, " + ("one per GPU, ghost rows over NCCL" if world > 1 else "in one process on one GPU"),
                           "ghost_bytes_per_cut_per_step": 4 * 2 * 4 * 8 * cfg.nphi * cfg.nR * 8,
                           "state_finite_after_run": bool(np.isfinite(d["kinetic"]) and np.isfinite(d["magnetic"]))},
                "gpu_launches": sum(s.g.launch_count for s in grp.slabs)}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_1812_00525_b200 import build as clt_build
    from paper_1812_00525_b200 import clt, inputs, replicas

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        clt_build.build()
    if world > 1:
        dist.barrier()

    prob = inputs.make_problem(args.config)
    cfg = prob.cfg
    dt = prob.dt * args.dt_scale
    g = clt.Clt.from_config(cfg, dt, device=f"cuda:{local}", d_i=args.d_i)
    if args.phi_scheme:
        g.set_phi_scheme(args.phi_scheme)
    if args.tile_z or args.phi_chunks or args.graph:
        g.set_tuning(args.tile_z, args.phi_chunks, args.graph)
    hU0 = torch.from_numpy(prob.U0).pin_memory()
    hU = torch.from_numpy(prob.U).pin_memory()
    hOut = torch.empty_like(hU).pin_memory()
    g.set_equilibrium(hU0)
    g.set_state(hU)

    def barrier():
        replicas.barrier(f"cuda:{local}")

    # ---- device-resident throughput: the library's default path (clt_step replays the step as a CUDA graph) ---------
    g.step(args.warmup)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    launches0 = g.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(g.torch_stream)
    if args.adaptive:
        g.step_cfl(args.steps, cfg.cfl)      # NEXT-1: dt = SETDT per step, on the device
    else:
        g.step(args.steps)
    e1.record(g.torch_stream)
    barrier()
    ms = e0.elapsed_time(e1)
    launches = g.launch_count - launches0
    clocks = sampler.stop()
    # ---- second, separately reported region: the same steps with a CUDA event pair around every launch (no graph), for
    # the per-kernel roofline; `value` above never comes from it ----------------------------------------------------
    prof_steps = max(1, min(args.steps, args.profile_steps))
    g.set_profiling(True)
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record(g.torch_stream)
    if args.adaptive:
        g.step_cfl(prof_steps, cfg.cfl)
    else:
        g.step(prof_steps)
    p1.record(g.torch_stream)
    barrier()
    prof_ms_step = p0.elapsed_time(p1) / prof_steps
    prof = g.get_profile()
    g.set_profiling(False)
    total_updates, secs, value = replicas.aggregate(cfg.interior * args.steps, ms * 1e-3, device=f"cuda:{local}")
    ms = secs * 1e3
    d = g.diagnostics()
    finite = all(np.isfinite(d[k]) for k in ("kinetic", "magnetic", "max_divB"))

    # ---- end to end through the C ABI with host buffers -----------------------------------------
    e2e_steps = max(1, min(args.e2e_steps, args.steps))
    g.set_state(hU); g.step(1); g.get_state(hOut)        # warm-up of the copy path
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        g.set_state(hU)          # H2D of the step's input from pinned host memory
        g.step(1)
        g.get_state(hOut)        # D2H of the result (synchronous: host destination)
    barrier()
    e2e_s = time.perf_counter() - t0
    _, e2e_s, e2e_value = replicas.aggregate(cfg.interior * e2e_steps, e2e_s, device=f"cuda:{local}")
    state_bytes = int(np.prod(cfg.shape)) * 8
    e2e_serial = e2e_value
    e2e_how = "clt_set_state(pinned host) + clt_step(1) + clt_get_state(pinned host) per step, wall clock"
    # The same calls from two host threads, each with a context and a stream of its own (two independent copies of the
    # job): the H2D copy of one step overlaps the compute and the D2H copy of the other -- PCIe is full duplex and the
    # serial loop above leaves the GPU idle for 90 % of the time.  Every step still copies its input in and its result out.
    if args.e2e_pipeline > 1:
        import threading
        nw = args.e2e_pipeline
        workers, same = [(g, hU, hOut)], True
        for _ in range(nw - 1):
            g2 = clt.Clt.from_config(cfg, dt, device=f"cuda:{local}", d_i=args.d_i, stream=torch.cuda.Stream(f"cuda:{local}"))
            if args.phi_scheme:
                g2.set_phi_scheme(args.phi_scheme)
            if args.tile_z or args.phi_chunks or args.graph:
                g2.set_tuning(args.tile_z, args.phi_chunks, args.graph)
            g2.set_equilibrium(hU0)
            hU2, hOut2 = hU.clone().pin_memory(), torch.empty_like(hU).pin_memory()
            g2.set_state(hU2); g2.step(1); g2.get_state(hOut2)       # warm-up; also: every pipeline computes the same thing
            same = same and bool(torch.equal(hOut, hOut2))
            workers.append((g2, hU2, hOut2))
        start = threading.Barrier(nw + 1)

        def work(gg, hin, hout):
            torch.cuda.set_device(local)
            start.wait()
            for _ in range(e2e_steps):
                gg.set_state(hin)
                gg.step(1)
                gg.get_state(hout)

        th = [threading.Thread(target=work, args=w) for w in workers]
        for t in th:
            t.start()
        barrier()
        start.wait()
        t0 = time.perf_counter()
        for t in th:
            t.join()
        pipe_s = time.perf_counter() - t0
        barrier()
        _, pipe_s, e2e_value = replicas.aggregate(cfg.interior * e2e_steps * nw, pipe_s, device=f"cuda:{local}")
        e2e_how = (f"{nw} host threads, each with its own context and stream, each doing clt_set_state(pinned host) + clt_step(1) + "
                   "clt_get_state(pinned host) per step (the copies of one overlap the compute and the copies of the others), wall "
                   f"clock; `serial_value` is one thread alone; all pipelines return identical states: {same}")
        for w in workers[1:]:
            w[0].close()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    ms_step = ms / args.steps
    peak, peak_src = measured_peaks()
    # dominant kernel: the fused RHS + RK4 stage-combine kernel (its four stage variants pooled)
    n_rhs = sum(prof["n_rhs"][1:5])
    ms_rhs = sum(prof["ms_rhs"][1:5])
    roof = None
    if n_rhs:
        bytes_per_launch = sum(RHS_DOUBLES[s] * prof["n_rhs"][s] for s in (1, 2, 3, 4)) * 8.0 * cfg.interior / n_rhs
        dur = ms_rhs / n_rhs * 1e-3
        ach = bytes_per_launch / dur / 1e9
        per_stage = {f"stage{s}": {"ms": prof["ms_rhs"][s] / prof["n_rhs"][s],
                                   "GBps": RHS_DOUBLES[s] * 8.0 * cfg.interior / (prof["ms_rhs"][s] / prof["n_rhs"][s] * 1e-3) / 1e9}
                     for s in (1, 2, 3, 4) if prof["n_rhs"][s]}
        curl = None
        if prof["n_curl"]:
            cms = prof["ms_curl"] / prof["n_curl"]
            curl = {"ms": cms, "GBps": CURL_DOUBLES * 8.0 * cfg.interior / (cms * 1e-3) / 1e9}
        roof = {"bound": "hbm", "kernel": "rhs_tma_kernel (fused RHS + RK4 stage combine, its 4 stage variants pooled)",
                "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                "traffic": args.traffic if args.traffic is not None else (profiled_traffic() if cfg.index == 4 else None),
                "traffic_source": ("--traffic argument" if args.traffic is not None else
                                   ("committed ncu --set full capture, profiles/traffic.csv (not measured in this run)"
                                    if cfg.index == 4 else None)),
                "profiled_region": {"steps": prof_steps, "ms_per_step": prof_ms_step,
                                    "note": "per-kernel CUDA events, no graph; `value` is timed on the default graph path"},
                "ncu_pipes": profiled_pipes() if cfg.index == 4 else None,
                "peak_source": peak_src + ", burst figure", "avg_launch_ms": ms_rhs / n_rhs,
                "algorithmic_bytes_per_launch": bytes_per_launch, "share_of_step": ms_rhs / (ms_rhs + prof["ms_curl"] + prof.get("ms_phi", 0.0)),
                "per_stage": per_stage, "curl_kernel": curl,
                "phi_prepass": ({"ms": prof["ms_phi"] / prof["n_phi"], "launches_per_step": prof["n_phi"] / prof_steps}
                                if prof.get("n_phi") else None),
                "algorithmic_doubles_per_node": {"stage1": 19, "stage2": 35, "stage3": 27, "stage4": 35, "curl": 6,
                                                 "rk4_step": BYTES_PER_UPDATE // 8, "survey_textbook_schedule": 164},
                "whole_step": {"GBps": BYTES_PER_UPDATE * cfg.interior / (ms_step * 1e-3) / 1e9,
                               "frac": BYTES_PER_UPDATE * cfg.interior / (ms_step * 1e-3) / 1e9 / peak,
                               "survey_equivalent_GBps": SURVEY_BYTES_PER_UPDATE * cfg.interior / (ms_step * 1e-3) / 1e9}}
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        # the oracle on the measured configuration itself (>= 2 steps of config 4, about 10-30 s on the box's
        # cores) and once single-threaded on config 2
        r = oracle_rate(cfg.index, 2, budget_seconds=60.0)
        cpu = {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")}
        one = oracle_rate_single_thread(2, 2)
        cpu["single_thread_config2"] = {k: one[k] for k in ("value", "unit", "cores", "sample") if k in one} or one
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": f"config {cfg.index}: {cfg.nR}x{cfg.nphi}x{cfg.nZ} (R x phi x Z), {cfg.interior} interior nodes, "
                                   f"seeded reference state + perturbations (BASELINE.json configs[{cfg.index - 1}])",
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2": f"working set {g.workspace_bytes / 1e9:.2f} GB per replica, far larger than the 126 MB L2 (no flush needed)",
                       "dt": dt, "d_i": args.d_i, "phi_scheme": "pseudo-spectral" if args.phi_scheme else "fd4",
                       "time_step": "SETDT every step (clt_step_cfl)" if args.adaptive else "fixed",
                       "tile_z": args.tile_z, "phi_chunks": args.phi_chunks, "graph": args.graph,
                       "state_finite_after_run": bool(finite)},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": state_bytes,
                    "d2h_bytes_per_step": state_bytes, "steps": e2e_steps * max(1, args.e2e_pipeline),
                    "serial_value": e2e_serial, "how": e2e_how},
            "gpu_launches": launches,
            "roofline": roof, "cpu_baseline": cpu,
            "achieved_GBps_whole_step": BYTES_PER_UPDATE * cfg.interior / (ms_step * 1e-3) / 1e9}
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--tile-z", dest="tile_z", type=int, default=0)
    ap.add_argument("--phi-chunks", dest="phi_chunks", type=int, default=0)
    ap.add_argument("--graph", type=int, default=0, help="clt_set_tuning use_graph: 0 = library default (graph), 1 = always, 2 = never")
    ap.add_argument("--profile-steps", dest="profile_steps", type=int, default=10,
                    help="steps of the second, per-kernel-profiled region (roofline object)")
    ap.add_argument("--reference-budget", dest="reference_budget", type=float, default=280.0,
                    help="--impl reference: seconds of oracle time the run may take (timed steps are cut to fit)")
    ap.add_argument("--oracle-worker", dest="oracle_worker", default=None, help=argparse.SUPPRESS)
    ap.add_argument("--e2e-steps", dest="e2e_steps", type=int, default=3)
    ap.add_argument("--e2e-pipeline", dest="e2e_pipeline", type=int, default=2,
                    help="end-to-end figure from this many host threads with a context each; 1 = one serial loop only")
    ap.add_argument("--d-i", dest="d_i", type=float, default=0.0, help="Hall term of eq (5) (NEXT-3); 0 = the measured config")
    ap.add_argument("--phi-scheme", dest="phi_scheme", type=int, default=0, help="1 = pseudo-spectral phi scheme (NEXT-2)")
    ap.add_argument("--adaptive", action="store_true", help="NEXT-1: time clt_step_cfl (SETDT every step) instead of clt_step")
    ap.add_argument("--slabs", type=int, default=0, help="NEXT-4: cut the workload into K Z-slabs (see run_slabs)")
    ap.add_argument("--dt-scale", dest="dt_scale", type=float, default=1.0, help="scales the recipe's CFL time step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--traffic", type=float, default=None,
                    help="dram bytes per launch of the dominant kernel from an ncu --set full capture (profiles/)")
    args = ap.parse_args()
    if args.oracle_worker:
        idx, n = (int(x) for x in args.oracle_worker.split(","))
        print(json.dumps(oracle_rate(idx, n)), flush=True)
        return
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        run_reference(args)
    elif args.slabs > 1:
        run_slabs(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
