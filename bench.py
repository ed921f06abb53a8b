#!/usr/bin/env python
"""bench.py -- geodesic RK4 steps/s (FP64) of the hot path on B200, and the fraction of the FP64 roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload config4|...]

A "step" is one pass of the whole hot path (load+init, RHS, RK4, stop rules, work queue, final record)
over one batch: by default BASELINE.json configs[3], the configuration the metric's roofline target is
quoted on -- Kerr a=0.5, 2^22 timelike bound particles, h=0.01, 10^4 RK4 steps each, no snapshots.
Inputs are seeded and synthetic (paper_1803_08320_b200/workloads.py).  One JSON line on stdout (rank 0).

  value     whole-job geodesic-steps/s with inputs resident in HBM (CUDA events on the launch stream)
  e2e       the same through geo_integrate_host: pinned HOST buffers, H2D + D2H inside the timed region
  roofline  bound "alu": achieved FP64 TFLOP/s = steps/s x flop/step (static SASS count of the hot loop,
            paper_1803_08320_b200/sass_count.py) against 148 SM x 64 FP64 lanes x 2 x 1.965 GHz; the
            live register-only DFMA probe is reported beside it
  cpu_baseline  the oracle as it stands on the box's host cores, on a bounded sample

N > 1 (torchrun): independent geodesics are sharded by rank, no data-path collective, weak scaling
(every rank integrates its own 2^22-particle batch, seed + rank); value = all ranks' steps / max time.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_1803_08320_b200 import workloads as W  # noqa: E402

METRIC = "geodesic RK4 steps/sec (FP64, 1xB200)"
UNIT = "geodesic-steps/s"
# EXECUTED FP64 instructions per RK4 step of one geodesic (per thread): dynamic counts from ncu's
# per-instruction "Instructions Executed" of the hot kernel divided by the warp-steps of the launch
# (profiles/r01_config4_v3.md: DFMA 140, DMUL 143, DADD 42, DSETP 6 for Kerr).  flop = 2*DFMA + DMUL + DADD;
# pipe = all four.  The static SASS count of the loop (sass_count.py, an upper bound that includes the
# rarely executed blocks inside the loop's address range) is printed beside them as a cross-check.
FLOP_PER_STEP = {"kerr": 465.0, "schwarzschild": 397.0, "tabulated": 2218.0}
PIPE_INSTR_PER_STEP = {"kerr": 331.0, "schwarzschild": 273.0, "tabulated": 1300.0}
OTHER_INSTR_PER_STEP = {"kerr": 99.0}     # non-FP64 instructions per step, same ncu capture
FLOP_COUNT_SOURCE = {"kerr": "ncu dynamic count (profiles/r01_config4_v3.md)", "schwarzschild": "static SASS count",
                     "tabulated": "ncu dynamic thread-level count (profiles/r01_tab4.md): 918 DFMA + 323 DMUL + 58 DADD per step"}
SM_COUNT, FP64_LANES_PER_SM = 148, 64
# adaptive RK5(4) kernel, per step ATTEMPT of one Kerr geodesic, executed (ncu, thread level)
ADAPTIVE_FLOP_PER_ATTEMPT, ADAPTIVE_PIPE_PER_ATTEMPT = 1045.0, 684.0
ADAPTIVE_SOURCE = "ncu dynamic thread-level count (profiles/r01_config3a_rk45.md): 361 DFMA + 271 DMUL + 52 DADD per attempt"
# declared algorithmic work of one Kerr RK4 step (4 RHS + compensated update).
F_ALG_SURVEY = {"kerr": 800.0}
# dram__bytes_read.sum + dram__bytes_write.sum of one geo_rk4_kernel launch from the committed
# `ncu --set full` capture of that workload (profiles/), bytes; None where no capture exists.
TRAFFIC_NCU_BYTES = {"config3a": 103_028_736, "tab4": 657_377_536, "config4": 664_555_776, "snapbench": 69_562_443_296}      # profiles/r01_config4_final.md, r01_snapbench_v3.md, r01_config3a_rk45.md, r01_tab4.md (full-size capture of v2: particle I/O only)


def workload(name: str, rank: int, n_override: int | None, nthreads: int) -> dict:
    """The five BASELINE.json configs as concrete inputs."""
    if name == "config1":
        n = n_override or 256
        return dict(name="configs[0] Schwarzschild circular", metric="schwarzschild", a=0.0, st=W.circular_schwarzschild(n, W.SEED_BASE + 1 + 1000 * rank),
                    h=0.01, nsteps=2000, snapshot_every=100, snap_mask=0xFF, kind=0, r_capture=-np.inf, r_escape=np.inf)
    if name in ("config2", "config4"):
        a = 0.9 if name == "config2" else 0.5
        n = n_override or (65536 if name == "config2" else 1 << 22)
        k = 2 if name == "config2" else 4
        st = W.kerr_bound(n, a, W.SEED_BASE + k + 1000 * rank, nthreads=nthreads, chunk=1 << 20)
        return dict(name=f"configs[{k - 1}] Kerr a={a} bound timelike", metric="kerr", a=a, st=st, h=0.01,
                    nsteps=100000 if name == "config2" else 10000, snapshot_every=1000 if name == "config2" else 0,
                    snap_mask=0xFF, kind=0, r_capture=-np.inf, r_escape=np.inf)
    if name in ("paper_t4", "paper_t3"):
        # the paper's own performance test (section 6.4): "random" timelike geodesics around
        # Kerr a = 0.5, t_f = 1000, h = 0.1 (10^4 RK4 steps); its initial conditions are unpublished, the
        # bound-orbit generator of configs 2/4 stands in.  Table 4: 10 000 geodesics, no
        # output, 27.066675 s on a GTX 960M.  Table 3: 50 000 geodesics with the solution
        # of EVERY step copied to the host and written out (t, x, y, z per step), 35.6253648 min.
        n = n_override or (10000 if name == "paper_t4" else 50000)
        st = W.kerr_bound(n, 0.5, W.SEED_BASE + 8 + 1000 * rank, nthreads=nthreads)
        t3 = name == "paper_t3"
        return dict(name=("paper Table 3: 50 000 Kerr a=0.5 geodesics, every step output in the paper's format" if t3 else
                          "paper Table 4: 10 000 Kerr a=0.5 geodesics, no output"), metric="kerr", a=0.5, st=st, h=0.1,
                    nsteps=10000, snapshot_every=1 if t3 else 0, snap_mask=0x0F, kind=0, r_capture=-np.inf, r_escape=np.inf,
                    flags=8 if t3 else 0,      # GEO_FLAG_CARTESIAN_SNAP
                    paper_steps_per_s=(50000 * 1e4 / (35.6253648 * 60.0)) if t3 else (10000 * 1e4 / 27.066675))
    if name == "snapbench":
        # SURVEY.md 8(d) snapshot-writer microbenchmark: cheap RHS, a record of all 8 components EVERY step
        n = n_override or (1 << 22)
        return dict(name="snapshot microbenchmark: Schwarzschild circular, snapshot every step, 8 comps", metric="schwarzschild", a=0.0,
                    st=W.circular_schwarzschild(n, W.SEED_BASE + 6 + 1000 * rank), h=0.01, nsteps=256, snapshot_every=1,
                    snap_mask=0xFF, kind=0, r_capture=-np.inf, r_escape=np.inf)
    if name in ("snapkerr", "snapkerr_xyz"):
        # round-1 verdict, kernel item 9: the paper's own output mode (a record EVERY step) on the Kerr
        # kernel at a size that fills the machine: the configs[3] particles, 256 steps, all 8 BL components (snapkerr,
        # 69 GB) or the paper's (t, x, y, z) record of eq.(7) (snapkerr_xyz, 34 GB)
        n = n_override or (1 << 22)
        st = W.kerr_bound(n, 0.5, W.SEED_BASE + 4 + 1000 * rank, nthreads=nthreads, chunk=1 << 20)
        xyz = name == "snapkerr_xyz"
        return dict(name="Kerr a=0.5 bound particles, a record every step: " + ("(t, x, y, z) of eq.(7)" if xyz else "8 BL components"),
                    metric="kerr", a=0.5, st=st, h=0.01, nsteps=256, snapshot_every=1, snap_mask=0x0F if xyz else 0xFF, kind=0,
                    r_capture=-np.inf, r_escape=np.inf, flags=8 if xyz else 0)
    if name == "config3s":
        # configs[2] with the pixels in a seeded random order: every warp holds a captured/escaped mix
        wl = workload("config3", rank, n_override, nthreads)
        perm = np.random.default_rng(W.SEED_BASE + 3).permutation(wl["st"].shape[1])
        wl["st"] = np.ascontiguousarray(wl["st"][:, perm])
        wl["name"] += " (pixels shuffled)"
        return wl
    if name == "tab4":
        # the particles of configs[3] through a TABULATED Kerr a = 0.5 metric (eq.(8) sampled on a
        # 2049 x 513 Boyer-Lindquist grid + ghosts, 42 MB in the kernel's layout: L2-resident), 1000 RK4 steps
        wl = workload("config4", rank, n_override, nthreads)
        wl["name"] = "configs[3] particles on a tabulated Kerr a=0.5 metric (2049x513 nodes, cubic convolution)"
        wl["metric"] = "tabulated"
        wl["table"] = W.kerr_metric_table(1.0, 0.5, 2049, 513, 2.0, 45.0, 0.1, math.pi - 0.1)
        wl["nsteps"] = 1000
        return wl
    if name == "config3a":
        # the rays of configs[2] with the adaptive Dormand-Prince 5(4) stepper (per-ray step control);
        # unit = one step ATTEMPT (accepted or rejected: 6 new RHS evaluations + error estimate)
        wl = workload("config3", rank, n_override, nthreads)
        wl["name"] += " -- adaptive RK5(4), rtol = atol = 1e-9"
        wl["adaptive"] = dict(h0=wl["h"], rtol=1e-9, atol=1e-9, max_attempts=wl["nsteps"])
        return wl
    if name in ("config3", "config5"):
        N = n_override or (1024 if name == "config3" else 4096)
        incl = 60.0 if name == "config3" else 85.0
        rows = N if name == "config3" else min(N, 256)      # config 5 is tiled (S3): one tile
        st = W.camera_rays(N, 0.998, incl, row0=(N - rows) // 2 if name == "config5" else 0, rows=rows)
        return dict(name=f"configs[{2 if name == 'config3' else 4}] Kerr a=0.998 camera {N}x{rows} i={incl}", metric="kerr", a=0.998, st=st,
                    h=0.02, nsteps=200000, snapshot_every=0 if name == "config3" else 500, snap_mask=0x0F, kind=1,
                    r_capture=W.horizon_radius(1.0, 0.998) + 0.01, r_escape=1100.0)
    raise SystemExit(f"unknown workload {name}")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def stop(self, t0: float, t1: float) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 and len(r) >= 7] or [r for (_, r) in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [nm for k, nm in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "reasons": reasons,
                "power_w_max": max(float(r[2]) for r in rows), "samples": len(rows)}


def oracle_time(wl: dict, steps: int, warmup: int, budget_s: float = 12.0) -> dict:
    """Time the oracle, as it stands, on the host cores on a bounded sample of the workload."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import geo_oracle
    cores = os.cpu_count() or 1
    st = wl["st"]
    # sample: a prefix of the batch sized for ~budget_s of wall time at ~3e6 steps/s/core
    ad = wl.get("adaptive")
    per = max(1, int(budget_s * 3.0e6 * cores / max(1, 300 * 2 if ad else wl["nsteps"])))   # adaptive: ~300 attempts/ray, 2x cost
    m = min(st.shape[1], max(cores, per))
    sub = np.ascontiguousarray(st[:, :m])
    metric = geo_oracle.KERR if wl["metric"] == "kerr" else geo_oracle.SCHWARZSCHILD
    if wl["metric"] == "tabulated":
        import geo_tab_oracle
        per = max(1, per // 4)          # ~4x the analytic RHS cost
    kw = dict(r_capture=wl["r_capture"], r_escape=wl["r_escape"], kind=wl["kind"], nthreads=cores,
              snapshot_every=wl["snapshot_every"], snap_mask=wl["snap_mask"], flags=wl.get("flags", 0))
    times, done = [], 0
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        if wl["metric"] == "tabulated":
            o = geo_tab_oracle.integrate(wl["table"], sub, wl["h"], wl["nsteps"], r_capture=wl["r_capture"],
                                         r_escape=wl["r_escape"], kind=wl["kind"], nthreads=cores)
        elif ad:
            o = geo_oracle.integrate_adaptive(metric, 1.0, wl["a"], sub, ad["h0"], ad["rtol"], ad["atol"], ad["max_attempts"],
                                              r_capture=wl["r_capture"], r_escape=wl["r_escape"], kind=wl["kind"], nthreads=cores)
        else:
            o = geo_oracle.integrate(metric, 1.0, wl["a"], sub, wl["h"], wl["nsteps"], **kw)
        dt = time.perf_counter() - t0
        if i >= warmup:
            times.append(dt)
            done += int(o["steps_done"].sum()) + (int(o["rejected"].sum()) if ad else 0)
    return {"value": done / sum(times), "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {m} of {st.shape[1]} particles x up to {wl['nsteps']} steps, {steps} pass(es)",
            "ms_per_step": 1e3 * sum(times) / len(times)}


def run_reference(args, rank: int, world: int) -> None:
    """--impl reference: the oracle on the host cores (this tier has no reference implementation)."""
    if rank != 0:
        return
    n_gen = args.n
    if n_gen is None and args.workload in ("config2", "config4"):
        # the sample is a prefix of the batch and kerr_bound(n)[:m] == kerr_bound(m): generate only the prefix
        nsteps = 100000 if args.workload == "config2" else 10000
        n_gen = min(65536 if args.workload == "config2" else 1 << 22,
                    max(os.cpu_count() or 1, int(8.0 * 3.0e6 * (os.cpu_count() or 1) / nsteps)))
    wl = workload(args.workload, 0, n_gen, os.cpu_count() or 1)
    r = oracle_time(wl, args.steps, min(args.warmup, 1), budget_s=8.0)
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": r["ms_per_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl["name"], "n_sample": int(wl["st"].shape[1]), "h": wl["h"], "nsteps": wl["nsteps"]},
            "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def flop_counts(metric: str) -> tuple[float, float, str, dict | None]:
    static = None
    try:
        from paper_1803_08320_b200 import sass_count
        c = sass_count.count({"kerr": "rk4_kernelILb1ELi0ELb0", "schwarzschild": "rk4_kernelILb0ELi0ELb0",
                              "tabulated": "geo_tab_rk4_kernelILb0ELb1E"}[metric])
        static = {"flop": c["flop"], "fp64_pipe": c["fp64_pipe"]}
    except Exception:
        pass
    return FLOP_PER_STEP[metric], PIPE_INSTR_PER_STEP[metric], FLOP_COUNT_SOURCE[metric], static


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config4", choices=["config1", "config2", "config3", "config4", "config5", "config3s", "config3a", "tab4", "snapbench", "snapkerr", "snapkerr_xyz", "paper_t3", "paper_t4"])
    ap.add_argument("--n", type=int, default=None, help="override particle count / image size (development)")
    ap.add_argument("--flags", type=int, default=0, help="GEO_FLAG_* bits (2 = static mapping, 4 = shared-memory-staged snapshots, 16 = tabulated metric: gather instead of the stencil cache)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_1803_08320_b200 import geo

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    if not os.environ.get("GEO_LIB"):
        from paper_1803_08320_b200 import build as geo_build
        geo_build.build()      # in-tree (re)build if libgeo.so is missing or stale; raises if nvcc fails
    geo.lib()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    ncpu = max(1, (os.cpu_count() or 1) // max(1, world))
    wl = workload(args.workload, rank, args.n, ncpu)
    st = wl["st"]
    n = st.shape[1]
    if wl["metric"] == "tabulated":
        tb = wl["table"]
        ctx = geo.geo_create_tabulated(tb["tab"], tb["x1_0"], tb["d1"], tb["x2_0"], tb["d2"])
    else:
        ctx = geo.geo_create(geo.KERR if wl["metric"] == "kerr" else geo.SCHWARZSCHILD, 1.0, wl["a"])
    d_in = torch.from_numpy(st).to(dev)
    out = geo.alloc_outputs(n, dev, wl["nsteps"], wl["snapshot_every"], None, wl["snap_mask"])
    kw = dict(r_capture=wl["r_capture"], r_escape=wl["r_escape"], kind=wl["kind"], flags=args.flags | wl.get("flags", 0),
              snapshot_every=wl["snapshot_every"])
    stream = torch.cuda.current_stream(dev)

    ad = wl.get("adaptive")
    d_rej = torch.zeros(n, dtype=torch.int32, device=dev) if ad else None

    def one_pass():
        if ad:
            geo.geo_integrate_adaptive(ctx, d_in, ad["h0"], ad["rtol"], ad["atol"], ad["max_attempts"], out, r_capture=wl["r_capture"],
                                       r_escape=wl["r_escape"], kind=wl["kind"], rejected=d_rej, stream=stream)
        else:
            geo.geo_integrate(ctx, d_in, wl["h"], wl["nsteps"], out, stream=stream, **kw)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(args.warmup):
        one_pass()
    barrier()

    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    barrier()
    t0 = time.time()
    ev[0].record(stream)
    for i in range(args.steps):
        one_pass()
        ev[i + 1].record(stream)
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    steps_per_pass = int(out["steps_done"].sum().item())    # every pass integrates the same batch
    if ad:
        steps_per_pass += int(d_rej.sum().item())           # adaptive: unit = step attempt (accepted + rejected)
    total_ms = ev[0].elapsed_time(ev[-1])
    per_launch_ms = [ev[i].elapsed_time(ev[i + 1]) for i in range(args.steps)]
    tmax = torch.tensor([total_ms], dtype=torch.float64, device=dev)
    tot_steps = torch.tensor([float(steps_per_pass) * args.steps], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot_steps, op=dist.ReduceOp.SUM)
    value = tot_steps.item() / (tmax.item() * 1e-3)

    # ---- e2e: host buffers through geo_integrate_host (pinned), H2D + D2H inside the timed region ----
    e2e = None
    snap_bytes = out["snapshots"].numel() * 8 if out["snapshots"] is not None else 0
    if ad and not args.no_e2e:
        h_in = torch.from_numpy(st).pin_memory()
        h_out = geo.alloc_outputs_host(n, pinned=True)
        h_rej = torch.zeros(n, dtype=torch.int32).pin_memory()
        akw = dict(r_capture=wl["r_capture"], r_escape=wl["r_escape"], kind=wl["kind"], rejected=h_rej)
        geo.geo_integrate_adaptive_host(ctx, h_in, ad["h0"], ad["rtol"], ad["atol"], ad["max_attempts"], h_out, **akw)   # warm-up
        ke = max(1, min(args.steps, 2))
        barrier()
        te0 = time.perf_counter()
        for _ in range(ke):
            geo.geo_integrate_adaptive_host(ctx, h_in, ad["h0"], ad["rtol"], ad["atol"], ad["max_attempts"], h_out, **akw)
        torch.cuda.synchronize(dev)
        te = torch.tensor([time.perf_counter() - te0], dtype=torch.float64, device=dev)
        es = torch.tensor([float(h_out["steps_done"].sum().item() + h_rej.sum().item()) * ke], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
            dist.all_reduce(es, op=dist.ReduceOp.SUM)
        bo = sum(v.numel() * v.element_size() for k, v in h_out.items() if hasattr(v, "numel")) + h_rej.numel() * 4
        e2e = {"value": es.item() / te.item(), "unit": UNIT, "h2d_bytes_per_step": int(h_in.numel() * 8),
               "d2h_bytes_per_step": int(bo), "passes": ke, "api": "geo_integrate_adaptive_host (pinned host buffers)"}
    elif not args.no_e2e and snap_bytes <= (16 << 30):      # larger trajectory buffers stay device-resident
        h_in = torch.from_numpy(st).pin_memory()
        h_out = geo.alloc_outputs_host(n, wl["nsteps"], wl["snapshot_every"], None, wl["snap_mask"], pinned=True)
        geo.geo_integrate_host(ctx, h_in, wl["h"], wl["nsteps"], h_out, **kw)    # warm-up (allocates scratch)
        ke = max(1, min(args.steps, 2))
        barrier()
        te0 = time.perf_counter()
        for _ in range(ke):
            geo.geo_integrate_host(ctx, h_in, wl["h"], wl["nsteps"], h_out, **kw)
        torch.cuda.synchronize(dev)
        te = torch.tensor([time.perf_counter() - te0], dtype=torch.float64, device=dev)
        es = torch.tensor([float(h_out["steps_done"].sum().item()) * ke], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
            dist.all_reduce(es, op=dist.ReduceOp.SUM)
        bo = sum(v.numel() * v.element_size() for k, v in h_out.items() if hasattr(v, "numel"))
        bi = h_in.numel() * 8
        e2e = {"value": es.item() / te.item(), "unit": UNIT, "h2d_bytes_per_step": int(bi), "d2h_bytes_per_step": int(bo),
               "passes": ke, "api": "geo_integrate_host (pinned host buffers)"}

    if rank != 0:
        if world > 1:
            dist.barrier()
            dist.destroy_process_group()
        return

    # ---- roofline: FP64 ALU (DFMA pipe) ----
    flop, pipe, how, static_count = flop_counts(wl["metric"])
    if ad:
        # unit = one step attempt of the RK5(4) kernel; executed FP64 instructions per attempt from the ncu capture
        flop, pipe, how = ADAPTIVE_FLOP_PER_ATTEMPT, ADAPTIVE_PIPE_PER_ATTEMPT, ADAPTIVE_SOURCE
        try:
            from paper_1803_08320_b200 import sass_count
            c = sass_count.count("geo_rk45_kernelILb1E")
            static_count = {"flop": c["flop"], "fp64_pipe": c["fp64_pipe"]}
        except Exception:
            static_count = None
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    sm_max = float(clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0)
    peak_tf = SM_COUNT * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    kernel_ms = sum(per_launch_ms) / len(per_launch_ms)
    ach_tf = steps_per_pass * flop / (kernel_ms * 1e-3) / 1e12
    # live DFMA probe (register-only FMA chains over a full-chip grid)
    sink = torch.zeros(1, dtype=torch.float64, device=dev)
    geo.geo_probe_dfma(ctx, 2000, sink, stream)
    torch.cuda.synchronize(dev)
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record(stream)
    nf = geo.geo_probe_dfma(ctx, 400000, sink, stream)
    p1.record(stream)
    torch.cuda.synchronize(dev)
    probe_tf = 2.0 * nf / (p0.elapsed_time(p1) * 1e-3) / 1e12
    info = geo.geo_launch_info(ctx, n, args.flags, wl["snapshot_every"])
    if ad:
        info = {"grid": SM_COUNT * 3, "block": 128, "regs": 168, "ctas_per_sm": 3}     # geo_rk45_kernel (profiles/r01_config3a_rk45.md)
    # Algorithmic work per unit: the flop of one RK4 step in the formulation built here,
    # 465 for Kerr = what the kernel executes (ncu counts) -- so `achieved` is also what ncu's
    # dadd + dmul + 2 dfma counters give, the quantity the north_star's ">= 50 % of FP64 peak in ncu" is about.
    # SURVEY.md 8(d) had declared F_alg = 800 flop from a hand count before any kernel existed and asked for
    # that figure too ("so neither padding nor trimming arithmetic can game the fraction"): it is reported as
    # frac_survey_f_alg.  fp64_pipe_util counts every FP64 instruction as one pipe slot (a DMUL occupies the
    # pipe like a DFMA); ncu's sm__pipe_fp64_cycles_active agrees with it.
    f_alg = F_ALG_SURVEY.get(wl["metric"], flop)
    sps = steps_per_pass / (kernel_ms * 1e-3)
    roofline = {"bound": "alu", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                "frac": ach_tf / peak_tf, "traffic": TRAFFIC_NCU_BYTES.get(args.workload),
                "kernel": "geo_rk45_kernel" if ad else ("geo_tab_rk4_kernel" if wl["metric"] == "tabulated" else "geo_rk4_kernel"),
                "kernel_ms": kernel_ms,
                "flop_per_step": flop, "fp64_pipe_instr_per_step": pipe,
                "flop_count_source": how, "static_sass_count_of_loop": static_count,
                "flop_per_step_survey_f_alg": f_alg, "frac_survey_f_alg": sps * f_alg / 1e12 / peak_tf,
                "peak_source": f"derived: {SM_COUNT} SM x {FP64_LANES_PER_SM} FP64 lanes x 2 flop x {sm_max:.0f} MHz (nominal clock; MEASURED_PEAKS.json has no FP64 entry)",
                "fp64_pipe_util": sps * pipe / (SM_COUNT * FP64_LANES_PER_SM * sm_max * 1e6),
                "dfma_probe_tflops": probe_tf, "frac_of_dfma_probe": ach_tf / probe_tf}
    if wl["metric"] == "tabulated":
        # SURVEY 8(f).3 expected this path to be memory- rather than FP64-bound: the table reads are reported beside
        # the ALU figure.  Algorithmic bytes: 4 stencil evaluations per step x 640 B (16 x 40-B nodes), served by L1/L2.
        roofline.pop("frac_survey_f_alg")
        roofline.pop("flop_per_step_survey_f_alg")
        roofline["table_bytes_per_step"] = 4 * 640
        roofline["table_read_gbs"] = sps * 4 * 640 / 1e9
        tbl = wl["table"]["tab"]
        roofline["table_mb_on_device"] = tbl.shape[1] * tbl.shape[2] * 40 / 1e6
    if ad:
        roofline.pop("flop_per_step_survey_f_alg"), roofline.pop("frac_survey_f_alg")
        roofline["unit_of_work"] = "one RK5(4) step attempt (accepted or rejected)"
    elif wl["metric"] == "kerr":
        # measured bound: a warp-level FP64 instruction holds the scheduler's issue port
        # for 2 cycles (16 FP64 lanes per scheduler), any other instruction for 1
        slots = 2.0 * pipe + OTHER_INSTR_PER_STEP["kerr"]
        roofline["other_instr_per_step"] = OTHER_INSTR_PER_STEP["kerr"]
        roofline["issue_slot_util"] = sps * slots / (SM_COUNT * 4 * 32 * sm_max * 1e6)

    if args.workload == "snapbench":
        # snapshot-heavy run: the bound is HBM write bandwidth.  Algorithmic bytes per launch = every
        # record written once (n x slots x ncomp x 8 B) + inputs read + final records written.
        ncomp = bin(wl["snap_mask"] & 0xFF).count("1")
        slots = 1 + wl["nsteps"] // wl["snapshot_every"]
        alg_bytes = n * (slots * ncomp * 8 + 48 + 100)
        hbm = float(peaks.get("hbm_gbs") or 6459.6)
        gbs = alg_bytes / (kernel_ms * 1e-3) / 1e9
        roofline = {"bound": "hbm", "achieved": gbs, "peak": hbm, "unit": "GB/s", "frac": gbs / hbm,
                    "traffic": TRAFFIC_NCU_BYTES.get(args.workload), "kernel": "geo_rk4_kernel", "kernel_ms": kernel_ms,
                    "algorithmic_bytes_per_launch": alg_bytes,
                    "peak_source": "MEASURED_PEAKS.json hbm_gbs (copy, read+write)" if peaks.get("hbm_gbs") else "fallback 6459.6 GB/s (MEASURED_PEAKS.json absent)",
                    "alu_view": roofline}

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        r = oracle_time(wl, 1, 0)
        cpu = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": tmax.item() / args.steps, "higher_is_better": True, "scaling": "weak",
            # only the paper's own workloads have a published number (GTX 960M, another machine: context)
            "vs_baseline": (value / wl["paper_steps_per_s"]) if wl.get("paper_steps_per_s") else None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl["name"], "n_per_gpu": n, "h": wl["h"], "nsteps": wl["nsteps"], "adaptive": ad,
                       "geodesics_per_s": (n * world * args.steps / (tmax.item() * 1e-3)),
                       "snapshot_every": wl["snapshot_every"], "geodesic_steps_per_pass_per_gpu": steps_per_pass,
                       "parallelism": f"independent geodesics sharded by rank x{world}, no collective",
                       "launch": info, "flags": args.flags | wl.get("flags", 0),
                       "paper": ({"steps_per_s": wl["paper_steps_per_s"], "hardware": "GeForce GTX 960M, CUDA 7.5 (PAPER.md:446)",
                                  "e2e_over_paper": (e2e["value"] / wl["paper_steps_per_s"]) if e2e else None}
                                 if wl.get("paper_steps_per_s") else None),
                       "l2": f"inputs+outputs {(d_in.numel() * 8 + out['final_state'].numel() * 8) / 1e6:.0f} MB vs 126 MB L2; state lives in registers"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": args.steps, "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(line), flush=True)
    geo.geo_destroy(ctx)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
