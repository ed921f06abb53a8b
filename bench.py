#!/usr/bin/env python
"""bench.py -- geodesic RK4 steps/s (FP64) of the hot path on B200, and the fraction of the FP64 roofline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload config4|...]
                    [--scaling weak|strong] [--no-secondary]

A "step" is one pass of the whole hot path (load+init, RHS, RK4, stop rules, work queue, final record)
over one batch: by default BASELINE.json configs[3], the configuration the metric's roofline target is
quoted on -- Kerr a=0.5, 2^22 timelike bound particles, h=0.01, 10^4 RK4 steps each, no snapshots.
Inputs are seeded and synthetic (paper_1803_08320_b200/workloads.py).  One JSON line on stdout (rank 0).

  value     whole-job geodesic-steps/s with inputs resident in HBM (CUDA events on the launch stream)
  e2e       the same through geo_integrate_host: pinned HOST buffers, H2D + D2H inside the timed region
  roofline  bound "alu": achieved FP64 TFLOP/s = steps/s x EXECUTED flop per step (ncu per-instruction counts of the
            committed capture, profiles/; cross-checked at run time against the static SASS count of the hot loop
            in the library that is loaded -- the run FAILS if they differ by more than 5 %) against
            148 SM x 64 FP64 lanes x 2 x SM clock; the live register-only DFMA probe is reported beside it
  secondary one pass each of the other configs / kernels (config 2, 3, 3 shuffled queue-vs-static, 5 central tile,
            snapshot microbenchmarks, adaptive RK5(4), tabulated metric, the paper's own Table 3/4 workloads)
  cpu_baseline  the oracle as it stands on the box's host cores, on a bounded sample

--workload config5 runs configs[4] WHOLE: the 4096^2 image as 16 tiles of 256 rows (the dense trajectory buffer
would be 215 GB), total steps / total kernel time, records actually written.

N > 1 (torchrun): independent geodesics are sharded by rank, no data-path collective.  --scaling weak (default):
every rank integrates its own 2^22-particle batch (seed + 1000 rank).  --scaling strong: ONE configs[2] image,
interleaved row tiles (tile t -> rank t mod N).  value = all ranks' steps / max time over ranks.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import re
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
SM_COUNT, FP64_LANES_PER_SM = 148, 64
# declared algorithmic work of one Kerr RK4 step (4 RHS + compensated update), a hand count made
# before any kernel existed; reported beside the executed count (frac_survey_f_alg), never used for `frac`.
F_ALG_SURVEY = {"kerr": 800.0}

# EXECUTED instructions per unit of work (per thread), from ncu's per-instruction "Instructions Executed" of the
# committed `ncu --set full` capture divided by the launch's warp-units.  flop = 2 DFMA + DMUL + DADD; pipe = all FP64
# instructions incl. DSETP; other = everything else.  Cross-check at run time (kernel_counts): the hot loop of `sym` in
# the LOADED library is counted statically (cuobjdump); that count must (a) equal `static_at_capture` -- the static count of the
# build the capture was made from -- within 1 %, i.e. the kernel has not changed since its instruction mix was
# measured, and (b) lie within 8 % of the executed count (the static count also contains the rarely executed blocks
# inside the loop's address range).  A kernel edit without a new capture makes bench.py FAIL instead of reporting
# stale numbers.
KERNEL_COUNTS = {
    "kerr": dict(sym="geo_rk4_kernelILb1ELi0ELb0ELb0ELb0E", units_per_loop=2, flop=461.0, pipe=326.0, other=68.0, tol=0.08, static_at_capture=(964, 686),
                 source="ncu per-instruction counts, profiles/r02_config4.md: 140 DFMA + 141 DMUL + 40 DADD + 5 DSETP per step",
                 kernel="geo_rk4_kernel"),
    "schwarzschild": dict(sym="geo_rk4_kernelILb0ELi0ELb0ELb0ELb0E", units_per_loop=2, flop=342.0, pipe=245.0, other=None, tol=0.0,
                          source="static SASS count of the hot loop (no ncu capture of this instantiation)", kernel="geo_rk4_kernel"),
    "adaptive": dict(sym="geo_rk45_kernelILi1ELb0E", units_per_loop=1, flop=1039.0, pipe=678.0, other=None, tol=0.15, static_at_capture=(1135, 778),
                     source="ncu thread-level counts, profiles/r02_config3a_rk45.md: 361 DFMA + 264 DMUL + 52 DADD per attempt "
                            "(incl. predicated-on work of lanes waiting for a refill)", kernel="geo_rk45_kernel"),
    "kerr_schild": dict(sym="geo_ks_rk4_kernelILi0ELb0EE", units_per_loop=2, flop=561.0, pipe=393.8, other=57.6, tol=0.08, static_at_capture=(1161, 821),
                        source="ncu per-instruction counts, profiles/r02_ks4.md: 172.2 DFMA + 160.6 DMUL + 56.0 DADD + 5.0 DSETP per step",
                        kernel="geo_ks_rk4_kernel"),
    "adaptive_ks": dict(sym="geo_ks_rk45_kernelILb0EE", units_per_loop=1, flop=0.0, pipe=0.0, other=None, tol=0.0,
                        source="static SASS count of the attempt loop (no ncu capture of this kernel; counts include predicated-off work)",
                        kernel="geo_ks_rk45_kernel"),
    "tabulated_general": dict(sym="geo_tabg_rk4_kernelILb0ELb1ELb0E", units_per_loop=None, flop=4073.0, pipe=2376.0, other=None, tol=None,
                              source="ncu per-instruction counts, profiles/r02_tab4_tabg4.md: 1735 DFMA + 550 DMUL + 52 DADD + 38 DSETP per step "
                                     "(4 evaluations through one rolled copy of the evaluator: no static cross-check)", kernel="geo_tabg_rk4_kernel"),
    "tabulated": dict(sym="geo_tab_rk4_kernelILb0ELb1ELb0E", units_per_loop=None, flop=2224.0, pipe=1300.0, other=None, tol=None,
                      source="ncu thread-level counts, profiles/r02_tab4_tabg4.md: 924.5 DFMA + 323 DMUL + 52 DADD per step (4 evaluations "
                             "through one rolled copy of the evaluator: no static cross-check)", kernel="geo_tab_rk4_kernel"),
}
# dram__bytes_read.sum + dram__bytes_write.sum of one launch from the committed `ncu --set full` capture of that
# workload (profiles/), bytes; None where no capture exists.
TRAFFIC_NCU_BYTES = {"config3a": 103_264_512, "tab4": 651_665_920, "tabg4": 1_225_114_112, "config4": 600_256_000, "snapbench": 69_562_443_296,
                     "snapkerr": 70_775_029_960, "paper_t3": 16_144_486_488, "ks4": 556_309_504}     # profiles/r02_*.md (snapbench: r01_snapbench_v3.md)


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
    if name == "tabg4":
        # SURVEY 8(f).3, general form (reading T6): the particles of configs[3] in ingoing KERR-SCHILD coordinates through
        # the ten-field table of the Kerr a = 0.5 metric (2049 x 513 nodes + ghosts, 102 MB of 96-byte node records), 250 steps
        n = n_override or (1 << 22)
        st, consts = W.kerr_bound(n, 0.5, W.SEED_BASE + 4 + 1000 * rank, nthreads=nthreads, chunk=1 << 20, return_constants=True)
        return dict(name="configs[3] particles in Kerr-Schild coordinates on a GENERAL tabulated metric (10 fields, 2049x513 nodes)",
                    metric="tabulated_general", a=0.5, st=W.to_kerr_schild(st, consts[0], 1.0, 0.5), h=0.01, nsteps=250,
                    snapshot_every=0, snap_mask=0xFF, kind=0, r_capture=-np.inf, r_escape=np.inf,
                    table=W.kerr_schild_metric_table(1.0, 0.5, 2049, 513, 2.0, 45.0, 0.1, math.pi - 0.1))
    if name == "ks4":
        # SURVEY 8(f).3, second clause (readings K1-K5): the particles of configs[3] in CARTESIAN Kerr-Schild coordinates on the
        # analytic horizon-penetrating, axis-regular path (geo_ks_rk4_kernel), 2500 RK4 steps
        n = n_override or (1 << 22)
        st, consts = W.kerr_bound(n, 0.5, W.SEED_BASE + 4 + 1000 * rank, nthreads=nthreads, chunk=1 << 20, return_constants=True)
        return dict(name="configs[3] particles in Cartesian Kerr-Schild coordinates (analytic, horizon-penetrating, axis-regular)",
                    metric="kerr_schild", a=0.5, st=W.to_cartesian_kerr_schild(st, consts[0], 1.0, 0.5), h=0.01, nsteps=2500,
                    snapshot_every=0, snap_mask=0xFF, kind=0, r_capture=-np.inf, r_escape=np.inf)
    if name == "config3ks":
        # the rays of configs[2] on the Cartesian Kerr-Schild path: the image without the polar-axis artefacts of eq.(8)
        wl = workload("config3", rank, n_override, nthreads)
        wl["name"] += " -- in Cartesian Kerr-Schild coordinates"
        wl["metric"] = "kerr_schild"
        wl["st"] = W.to_cartesian_kerr_schild(wl["st"], np.ones(wl["st"].shape[1]), 1.0, wl["a"])
        return wl
    if name == "config3aks":
        # reading K6: the rays of configs[2] with the adaptive stepper in Cartesian Kerr-Schild coordinates
        wl = workload("config3ks", rank, n_override, nthreads)
        wl["name"] += ", adaptive RK5(4), rtol = atol = 1e-9"
        wl["adaptive"] = dict(h0=wl["h"], rtol=1e-9, atol=1e-9, max_attempts=wl["nsteps"])
        return wl
    if name == "config3a":
        # the rays of configs[2] with the adaptive Dormand-Prince 5(4) stepper (per-ray step control);
        # unit = one step ATTEMPT (accepted or rejected: 6 new RHS evaluations + error estimate)
        wl = workload("config3", rank, n_override, nthreads)
        wl["name"] += " -- adaptive RK5(4), rtol = atol = 1e-9"
        wl["adaptive"] = dict(h0=wl["h"], rtol=1e-9, atol=1e-9, max_attempts=wl["nsteps"])
        return wl
    if name in ("config3", "config5", "config5tile"):
        N = n_override or (1024 if name == "config3" else 4096)
        incl = 60.0 if name == "config3" else 85.0
        rows = N if name == "config3" else min(N, 256)      # config 5 is tiled (S3): 16 tiles of 256 rows
        wl = dict(metric="kerr", a=0.998, h=0.02, nsteps=200000, snapshot_every=0 if name == "config3" else 500, snap_mask=0x0F,
                  kind=1, r_capture=W.horizon_radius(1.0, 0.998) + 0.01, r_escape=1100.0)
        if name == "config5":
            # the WHOLE image: every tile's rays (805 MB in all) stay resident, one trajectory buffer is reused
            wl["tiles"] = [W.camera_rays(N, 0.998, incl, row0=r0, rows=rows) for r0 in range(0, N, rows)]
            wl["st"] = wl["tiles"][len(wl["tiles"]) // 2]
            wl["name"] = f"configs[4] Kerr a=0.998 camera {N}x{N} i={incl}, WHOLE image in {len(wl['tiles'])} tiles of {rows} rows"
            return wl
        wl["st"] = W.camera_rays(N, 0.998, incl, row0=(N - rows) // 2 if name == "config5tile" else 0, rows=rows)
        wl["name"] = (f"configs[2] Kerr a=0.998 camera {N}x{rows} i={incl}" if name == "config3" else
                      f"configs[4] Kerr a=0.998 camera, central tile {N}x{rows} of {N}x{N}, i={incl}")
        return wl
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




_SASS_CACHE: dict = {}


def static_sass_count(sym_part: str) -> dict | None:
    """FP64 instructions in the hot loop of a kernel of the LOADED library: the backward branch that spans the most
    DFMA.  Static count: it includes the rarely executed blocks inside the loop's address range (an upper bound)."""
    from paper_1803_08320_b200 import geo
    key = (geo.LIB_PATH, os.path.getmtime(geo.LIB_PATH) if os.path.exists(geo.LIB_PATH) else 0)
    if key not in _SASS_CACHE:
        try:
            _SASS_CACHE[key] = subprocess.run(["cuobjdump", "-sass", geo.LIB_PATH], capture_output=True, text=True, check=True).stdout
        except (OSError, subprocess.CalledProcessError):
            _SASS_CACHE[key] = None
    out = _SASS_CACHE[key]
    if out is None:
        return None
    ins_re = re.compile(r"^\s+/\*([0-9a-f]{4,})\*/\s+(?:@!?U?P\d+\s+)?([A-Z0-9_.]+)(.*?);")
    ins, on = [], False
    for line in out.splitlines():
        m = re.search(r"Function : (\S+)", line)
        if m:
            if on:
                break
            on = sym_part in m.group(1)
            continue
        m = ins_re.match(line) if on else None
        if m:
            ins.append((int(m.group(1), 16), m.group(2), m.group(3)))
    best = (0, 0, -1)
    for addr, op, rest in ins:
        m = re.search(r"0x([0-9a-f]+)", rest) if op.startswith("BRA") else None
        if m and int(m.group(1), 16) < addr:
            tgt = int(m.group(1), 16)
            nf = sum(1 for a, o, _ in ins if tgt <= a <= addr and o.startswith("DFMA"))
            if nf > best[2]:
                best = (tgt, addr, nf)
    if best[2] < 0:
        return None
    body = [o for a, o, _ in ins if best[0] <= a <= best[1]]
    c = {k: sum(1 for o in body if o.startswith(k)) for k in ("DFMA", "DMUL", "DADD", "DSETP")}
    return {"flop": 2 * c["DFMA"] + c["DMUL"] + c["DADD"], "fp64_pipe": sum(c.values()), "instructions": len(body), **c}


def kernel_counts(key: str) -> dict:
    """KERNEL_COUNTS[key] checked against the static count of the loaded library (fails loudly on disagreement)."""
    kc = dict(KERNEL_COUNTS[key])
    st = static_sass_count(kc["sym"])
    kc["static"] = st
    if st and kc["units_per_loop"]:
        per = {k: st[k] / kc["units_per_loop"] for k in ("flop", "fp64_pipe")}
        kc["static_per_unit"] = per
        if kc["tol"] == 0.0:                      # no capture: the static count IS the source
            kc["flop"], kc["pipe"] = per["flop"], per["fp64_pipe"]
        elif kc["tol"]:
            rec = kc.get("static_at_capture")
            if rec and (abs(st["flop"] - rec[0]) > 0.01 * rec[0] or abs(st["fp64_pipe"] - rec[1]) > 0.01 * rec[1]):
                raise SystemExit(f"bench.py: the hot loop of {kc['kernel']} in the loaded library has {st['flop']} flop / {st['fp64_pipe']} "
                                 f"FP64 instructions (static), the build its ncu counts come from had {rec[0]} / {rec[1]}: the kernel "
                                 f"changed -- re-capture it (profiles/) and update KERNEL_COUNTS")
            for mine, theirs, what in ((kc["flop"], per["flop"], "flop"), (kc["pipe"], per["fp64_pipe"], "FP64 instructions")):
                if abs(theirs - mine) > kc["tol"] * mine:
                    raise SystemExit(f"bench.py: the {what} per unit of {kc['kernel']} in the loaded library (static {theirs:.1f}) "
                                     f"differs from the committed ncu count ({mine:.1f}) by more than {100 * kc['tol']:.0f} %: "
                                     f"re-capture the kernel (profiles/) and update KERNEL_COUNTS")
    return kc


def oracle_time(wl: dict, steps: int, warmup: int, budget_s: float = 12.0) -> dict:
    """Time the oracle, as it stands, on the host cores on a bounded sample of the workload."""
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import geo_oracle
    cores = os.cpu_count() or 1
    st = wl["st"]
    # sample: a prefix of the batch sized for ~budget_s of wall time at ~3e6 steps/s/core
    ad = wl.get("adaptive")
    per = max(1, int(budget_s * 3.0e6 * cores / max(1, 300 * 2 if ad else wl["nsteps"])))   # adaptive: ~300 attempts/ray, 2x cost
    if wl["metric"] in ("tabulated", "tabulated_general"):
        import geo_tab_oracle
        per = max(1, per // (4 if wl["metric"] == "tabulated" else 10))          # ~4x / ~10x the analytic RHS cost
    m = min(st.shape[1], max(cores, per))
    sub = np.ascontiguousarray(st[:, :m])
    metric = geo_oracle.KERR if wl["metric"] == "kerr" else geo_oracle.SCHWARZSCHILD
    kw = dict(r_capture=wl["r_capture"], r_escape=wl["r_escape"], kind=wl["kind"], nthreads=cores,
              snapshot_every=wl["snapshot_every"], snap_mask=wl["snap_mask"], flags=wl.get("flags", 0))
    times, done = [], 0
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        if wl["metric"] in ("tabulated", "tabulated_general"):
            fn = geo_tab_oracle.integrate if wl["metric"] == "tabulated" else geo_tab_oracle.integrate_general
            o = fn(wl["table"], sub, wl["h"], wl["nsteps"], r_capture=wl["r_capture"],
                   r_escape=wl["r_escape"], kind=wl["kind"], nthreads=cores)
        elif wl["metric"] == "kerr_schild" and ad:
            import geo_ks_oracle
            o = geo_ks_oracle.integrate_adaptive(1.0, wl["a"], sub, ad["h0"], ad["rtol"], ad["atol"], ad["max_attempts"],
                                                 r_capture=wl["r_capture"], r_escape=wl["r_escape"], kind=wl["kind"], nthreads=cores)
        elif wl["metric"] == "kerr_schild":
            import geo_ks_oracle
            o = geo_ks_oracle.integrate(1.0, wl["a"], sub, wl["h"], wl["nsteps"], r_capture=wl["r_capture"], r_escape=wl["r_escape"],
                                        kind=wl["kind"], nthreads=cores)
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
    if args.workload == "config5":
        args.workload = "config5tile"          # the sample is a prefix of the central tile
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


# ---------------------------------------------------------------------------------------------------------------
# N > 1: the only collectives of the path are the bench's own reductions (geodesics are independent).
# Factored out so that tests/test_multirank_gloo.py drives exactly this code with world_size 2 on gloo.
# ---------------------------------------------------------------------------------------------------------------
def dist_init(world: int, backend: str, device=None):
    """Returns torch.distributed (initialised) or None for a single process.  MASTER_ADDR/PORT, RANK, WORLD_SIZE come
    from the environment (torchrun)."""
    if world <= 1:
        return None
    import torch.distributed as dist
    if backend == "nccl":
        dist.init_process_group("nccl", device_id=device)
    else:
        dist.init_process_group(backend)
    return dist


def dist_barrier(dist, sync=None) -> None:
    if dist is not None:
        dist.barrier()
    if sync is not None:
        sync()


def reduce_time_and_units(dist, device, local_ms: float, local_units: float) -> tuple[float, float]:
    """(max over ranks of the device-timed milliseconds, sum over ranks of the units processed)."""
    import torch
    tmax = torch.tensor([local_ms], dtype=torch.float64, device=device)
    tot = torch.tensor([local_units], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    return tmax.item(), tot.item()


def dist_finish(dist) -> None:
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def make_line(args, world: int, value: float, ms_per_step: float, scaling: str, config: dict, clocks: dict, e2e, launches: int,
              roofline: dict, cpu, secondary=None, vs_baseline=None) -> dict:
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": scaling, "vs_baseline": vs_baseline,
            "dtype": "f64", "data": "synthetic", "config": config, "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
            "roofline": roofline, "cpu_baseline": cpu}
    if secondary is not None:
        line["secondary"] = secondary
    return line


def shard_for_rank(wl: dict, rank: int, world: int, scaling: str) -> dict:
    """--scaling strong: this rank's share of ONE image -- interleaved row tiles: tile t -> rank t mod world,
    so every rank gets the same captured/escaped mix.  Weak scaling shards nothing (each rank has its own batch)."""
    if scaling != "strong" or world == 1:
        return wl
    st = wl["st"]
    n = st.shape[1]
    N = int(round(math.sqrt(n)))
    if N * N != n:
        raise SystemExit("--scaling strong needs an image workload (config3)")
    rows = max(1, N // 16)
    tiles = W.interleaved_tiles(N // rows, rank, world)
    idx = np.concatenate([np.arange(t * rows * N, (t + 1) * rows * N) for t in tiles]) if tiles else np.zeros(0, dtype=np.int64)
    out = dict(wl)
    out["st"] = np.ascontiguousarray(st[:, idx])
    out["name"] = wl["name"] + f" -- strong scaling: rank {rank} of {world} holds tiles {tiles} of {N // rows}"
    return out


# ---------------------------------------------------------------------------------------------------------------
# GPU legs
# ---------------------------------------------------------------------------------------------------------------
class GpuRun:
    """One workload resident on the device: context, inputs, outputs, and timed passes through the C ABI."""

    def __init__(self, torch, geo, dev, wl: dict, flags: int):
        self.torch, self.geo, self.dev, self.wl = torch, geo, dev, wl
        self.flags = flags | wl.get("flags", 0)
        self.stream = torch.cuda.current_stream(dev)
        if wl["metric"] in ("tabulated", "tabulated_general"):
            tb = wl["table"]
            mk = geo.geo_create_tabulated if wl["metric"] == "tabulated" else geo.geo_create_tabulated_general
            self.ctx = mk(tb["tab"], tb["x1_0"], tb["d1"], tb["x2_0"], tb["d2"])
        else:
            self.ctx = geo.geo_create({"kerr": geo.KERR, "kerr_schild": geo.KERR_SCHILD}.get(wl["metric"], geo.SCHWARZSCHILD), 1.0, wl["a"])
        tiles = wl.get("tiles") or [wl["st"]]
        self.d_in = [torch.from_numpy(t).to(dev) for t in tiles]
        self.n = tiles[0].shape[1]
        self.n_total = sum(t.shape[1] for t in tiles)
        self.out = geo.alloc_outputs(self.n, dev, wl["nsteps"], wl["snapshot_every"], None, wl["snap_mask"])
        self.ad = wl.get("adaptive")
        self.d_rej = torch.zeros(self.n, dtype=torch.int32, device=dev) if self.ad else None
        self.kw = dict(r_capture=wl["r_capture"], r_escape=wl["r_escape"], kind=wl["kind"], flags=self.flags,
                       snapshot_every=wl["snapshot_every"])
        self.units_per_pass = None
        self.records_per_pass = None

    def launch(self, d_in) -> None:
        wl, ad = self.wl, self.ad
        if ad:
            self.geo.geo_integrate_adaptive(self.ctx, d_in, ad["h0"], ad["rtol"], ad["atol"], ad["max_attempts"], self.out,
                                            r_capture=wl["r_capture"], r_escape=wl["r_escape"], kind=wl["kind"],
                                            rejected=self.d_rej, stream=self.stream)
        else:
            self.geo.geo_integrate(self.ctx, d_in, wl["h"], wl["nsteps"], self.out, stream=self.stream, **self.kw)

    def count_pass(self) -> None:
        """One untimed pass that also counts the units of work (accepted steps; adaptive: attempts) and the trajectory
        records of every launch -- the work of a pass is the same every time."""
        units, records = 0, 0
        for d in self.d_in:
            self.launch(d)
            self.torch.cuda.synchronize(self.dev)
            units += int(self.out["steps_done"].sum().item())
            if self.ad:
                units += int(self.d_rej.sum().item())
            if self.out["snap_count"] is not None:
                records += int(self.out["snap_count"].sum().item())
        self.units_per_pass, self.records_per_pass = units, records

    def timed(self, steps: int, warmup: int, barrier) -> dict:
        torch = self.torch
        self.count_pass()                                   # first warm-up pass
        for _ in range(max(0, warmup - 1)):
            for d in self.d_in:
                self.launch(d)
        barrier()
        nl = len(self.d_in)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps * nl + 1)]
        t0 = time.time()
        ev[0].record(self.stream)
        k = 0
        for _ in range(steps):
            for d in self.d_in:
                self.launch(d)
                k += 1
                ev[k].record(self.stream)
        barrier()
        t1 = time.time()
        per_launch = [ev[i].elapsed_time(ev[i + 1]) for i in range(steps * nl)]
        return {"total_ms": ev[0].elapsed_time(ev[-1]), "per_launch_ms": per_launch, "launches": steps * nl,
                "kernel_ms_per_pass": sum(per_launch) / steps, "wall": (t0, t1)}

    def e2e(self, passes: int, barrier) -> dict:
        """The same work through the host-buffer entry points: pinned host memory, H2D + D2H inside the timed region."""
        torch, geo, wl, ad = self.torch, self.geo, self.wl, self.ad
        tiles = wl.get("tiles") or [wl["st"]]
        h_in = [torch.from_numpy(t).pin_memory() for t in tiles]
        h_out = geo.alloc_outputs_host(self.n, wl["nsteps"], wl["snapshot_every"], None, wl["snap_mask"], pinned=True)
        h_rej = torch.zeros(self.n, dtype=torch.int32).pin_memory() if ad else None

        def one(h):
            if ad:
                geo.geo_integrate_adaptive_host(self.ctx, h, ad["h0"], ad["rtol"], ad["atol"], ad["max_attempts"], h_out,
                                                r_capture=wl["r_capture"], r_escape=wl["r_escape"], kind=wl["kind"], rejected=h_rej)
                return int(h_out["steps_done"].sum().item() + h_rej.sum().item())
            geo.geo_integrate_host(self.ctx, h, wl["h"], wl["nsteps"], h_out, **self.kw)
            return int(h_out["steps_done"].sum().item())
        one(h_in[0])                                        # warm-up (allocates the ctx's device scratch)
        barrier()
        t0 = time.perf_counter()
        units = 0
        for _ in range(passes):
            for h in h_in:
                units += one(h)
        torch.cuda.synchronize(self.dev)
        dt = time.perf_counter() - t0
        bo = sum(v.numel() * v.element_size() for v in h_out.values() if hasattr(v, "numel")) + (h_rej.numel() * 4 if ad else 0)
        return {"seconds": dt, "units": units, "h2d_bytes_per_step": int(sum(h.numel() * 8 for h in h_in)),
                "d2h_bytes_per_step": int(bo * len(h_in)), "passes": passes,
                "api": ("geo_integrate_adaptive_host" if ad else "geo_integrate_host") + " (pinned host buffers)"}

    def close(self) -> None:
        self.geo.geo_destroy(self.ctx)
        self.d_in, self.out = None, None


def counts_key(wl: dict) -> str:
    if wl.get("adaptive"):
        return "adaptive_ks" if wl["metric"] == "kerr_schild" else "adaptive"
    return wl["metric"]


def alu_roofline(kc: dict, units_per_s: float, sm_max_mhz: float) -> dict:
    peak_tf = SM_COUNT * FP64_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
    ach = units_per_s * kc["flop"] / 1e12
    r = {"bound": "alu", "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s", "frac": ach / peak_tf,
         "fp64_pipe_util": units_per_s * kc["pipe"] / (SM_COUNT * FP64_LANES_PER_SM * sm_max_mhz * 1e6)}
    return r


# one pass each in the default run (driver-measured): (key in the JSON, workload, extra flags, e2e too?)
SECONDARY = [("config2", "config2", 0, True), ("config3", "config3", 0, True), ("config3_shuffled_queue", "config3s", 0, False),
             ("config3_shuffled_static", "config3s", 2, False), ("config5_central_tile", "config5tile", 0, False),
             ("snapbench_schwarzschild_every_step", "snapbench", 0, False), ("snapkerr_every_step_8comp", "snapkerr", 0, False),
             ("snapkerr_every_step_txyz", "snapkerr_xyz", 0, False), ("config3_adaptive_rk45", "config3a", 0, True),
             ("tab4_tabulated_metric", "tab4", 0, False), ("tabg4_general_tabulated_metric_kerr_schild", "tabg4", 0, False),
             ("ks4_cartesian_kerr_schild", "ks4", 0, True), ("config3_cartesian_kerr_schild", "config3ks", 0, False),
             ("config3_adaptive_rk45_cartesian_kerr_schild", "config3aks", 0, True), ("paper_table3", "paper_t3", 0, False), ("paper_table4", "paper_t4", 0, False)]


def run_secondary(torch, geo, dev, sm_max: float, ncpu: int, peaks: dict, reuse_config4) -> dict:
    """One warm-up + one timed pass of every other workload / kernel; kernel time by CUDA events."""
    res = {}
    for key, wname, flags, want_e2e in SECONDARY:
        try:
            if wname in ("tab4", "snapkerr", "snapkerr_xyz") and reuse_config4 is not None:
                # these use the configs[3] particles: reuse the batch already generated for the headline
                wl = _derive_from_config4(wname, reuse_config4)
            else:
                wl = workload(wname, 0, None, ncpu)
            run = GpuRun(torch, geo, dev, wl, flags)
            t = run.timed(1, 1, lambda: torch.cuda.synchronize(dev))
            ms = t["kernel_ms_per_pass"]
            ups = run.units_per_pass / (ms * 1e-3)
            kc = kernel_counts(counts_key(wl))
            rf = alu_roofline(kc, ups, sm_max)
            info = geo.geo_launch_info(run.ctx, run.n, run.flags, wl["snapshot_every"]) if not wl.get("adaptive") else None
            r = {"workload": wl["name"], "value": ups, "unit": UNIT + (" (unit = step attempt)" if wl.get("adaptive") else ""),
                 "ms": ms, "units_per_pass": run.units_per_pass, "frac": rf["frac"], "fp64_pipe_util": rf["fp64_pipe_util"],
                 "launch": info, "flags": run.flags}
            if run.records_per_pass:
                ncomp = bin(wl["snap_mask"] & 0xFF).count("1")
                wb = run.records_per_pass * ncomp * 8
                r["record_bytes_written"] = wb
                r["record_write_gbs"] = wb / (ms * 1e-3) / 1e9
                if wl["snapshot_every"] == 1:
                    r["hbm_frac"] = (wb + run.n * 148) / (ms * 1e-3) / 1e9 / float(peaks.get("hbm_gbs") or 6459.6)
            if wl.get("paper_steps_per_s"):
                r["paper_steps_per_s"] = wl["paper_steps_per_s"]
                r["vs_paper_gtx960m"] = ups / wl["paper_steps_per_s"]
            if want_e2e:
                e = run.e2e(1, lambda: torch.cuda.synchronize(dev))
                r["e2e"] = {"value": e["units"] / e["seconds"], "h2d_bytes_per_step": e["h2d_bytes_per_step"],
                            "d2h_bytes_per_step": e["d2h_bytes_per_step"], "api": e["api"]}
            run.close()
            del run
            torch.cuda.empty_cache()
            res[key] = r
        except Exception as ex:      # a secondary leg must not take the headline down; it is reported as failed
            res[key] = {"error": f"{type(ex).__name__}: {ex}"}
    q, s = res.get("config3_shuffled_queue", {}).get("value"), res.get("config3_shuffled_static", {}).get("value")
    if q and s:
        res["queue_vs_static_on_shuffled_pixels"] = q / s
    return res


def _derive_from_config4(wname: str, c4: dict) -> dict:
    wl = dict(c4)
    if wname == "tab4":
        wl["name"] = "configs[3] particles on a tabulated Kerr a=0.5 metric (2049x513 nodes, cubic convolution)"
        wl["metric"] = "tabulated"
        wl["table"] = W.kerr_metric_table(1.0, 0.5, 2049, 513, 2.0, 45.0, 0.1, math.pi - 0.1)
        wl["nsteps"] = 1000
        return wl
    xyz = wname == "snapkerr_xyz"
    wl.update(name="Kerr a=0.5 bound particles, a record every step: " + ("(t, x, y, z) of eq.(7)" if xyz else "8 BL components"),
              nsteps=256, snapshot_every=1, snap_mask=0x0F if xyz else 0xFF, flags=8 if xyz else 0)
    return wl


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config4",
                    choices=["config1", "config2", "config3", "config4", "config5", "config5tile", "config3s", "config3a", "tab4", "tabg4", "ks4", "config3ks", "config3aks",
                             "snapbench", "snapkerr", "snapkerr_xyz", "paper_t3", "paper_t4"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank its own batch; strong = one image (config3) split into interleaved row tiles")
    ap.add_argument("--n", type=int, default=None, help="override particle count / image size (development)")
    ap.add_argument("--flags", type=int, default=0, help="GEO_FLAG_* bits (2 = static mapping, 4 = shared-memory-staged snapshots, 16 = tabulated metric: gather instead of the stencil cache)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-secondary", action="store_true", help="skip the one-pass legs of the other workloads (default run, N = 1 only)")
    ap.add_argument("--dist-backend", default="nccl", help=argparse.SUPPRESS)
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    from paper_1803_08320_b200 import geo

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    if not os.environ.get("GEO_LIB"):
        from paper_1803_08320_b200 import build as geo_build
        geo_build.build()      # in-tree (re)build if libgeo.so is missing or stale; raises if nvcc fails
    geo.lib()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = dist_init(world, args.dist_backend, dev)

    def barrier():
        dist_barrier(dist, lambda: torch.cuda.synchronize(dev))

    if args.scaling == "strong" and args.workload == "config4":
        args.workload = "config3"
    ncpu = max(1, (os.cpu_count() or 1) // max(1, world))
    wl = workload(args.workload, rank if args.scaling == "weak" else 0, args.n, ncpu)
    wl = shard_for_rank(wl, rank, world, args.scaling)
    kc = kernel_counts(counts_key(wl))                       # fails loudly on a stale instruction count
    run = GpuRun(torch, geo, dev, wl, args.flags)
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    t = run.timed(args.steps, args.warmup, barrier)
    clocks = sampler.stop(*t["wall"])
    tmax_ms, tot_units = reduce_time_and_units(dist, dev, t["total_ms"], float(run.units_per_pass) * args.steps)
    value = tot_units / (tmax_ms * 1e-3)

    e2e = None
    snap_bytes = run.out["snapshots"].numel() * 8 if run.out["snapshots"] is not None else 0
    if not args.no_e2e and (snap_bytes <= (16 << 30)):
        e = run.e2e(1 if wl.get("tiles") else max(1, min(args.steps, 2)), barrier)
        te_ms, eu = reduce_time_and_units(dist, dev, e["seconds"] * 1e3, float(e["units"]))
        e2e = {"value": eu / (te_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": e["h2d_bytes_per_step"],
               "d2h_bytes_per_step": e["d2h_bytes_per_step"], "passes": e["passes"], "api": e["api"]}

    if rank != 0:
        run.close()
        dist_finish(dist)
        return

    # ---- roofline: FP64 ALU (DFMA pipe) of the dominant (only) kernel, this rank's launches ----
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    sm_max = float(clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0)
    kernel_ms = sum(t["per_launch_ms"]) / len(t["per_launch_ms"])            # average launch duration
    units_per_launch = run.units_per_pass / len(run.d_in)
    ups = run.units_per_pass / (t["kernel_ms_per_pass"] * 1e-3)
    roofline = alu_roofline(kc, ups, sm_max)
    sink = torch.zeros(1, dtype=torch.float64, device=dev)
    geo.geo_probe_dfma(run.ctx, 2000, sink, run.stream)                      # live register-only DFMA probe
    torch.cuda.synchronize(dev)
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record(run.stream)
    nf = geo.geo_probe_dfma(run.ctx, 400000, sink, run.stream)
    p1.record(run.stream)
    torch.cuda.synchronize(dev)
    probe_tf = 2.0 * nf / (p0.elapsed_time(p1) * 1e-3) / 1e12
    ad = wl.get("adaptive")
    info = geo.geo_launch_info(run.ctx, run.n, run.flags, wl["snapshot_every"]) if not ad else \
        {"grid": SM_COUNT * 3, "block": 128, "regs": 168, "ctas_per_sm": 3}
    roofline.update({
        "traffic": TRAFFIC_NCU_BYTES.get(args.workload), "kernel": kc["kernel"], "kernel_ms": kernel_ms,
        "units_per_launch": units_per_launch, "flop_per_step": kc["flop"], "fp64_pipe_instr_per_step": kc["pipe"],
        "flop_count_source": kc["source"], "static_sass_count_of_loop": kc.get("static"),
        "static_per_unit": kc.get("static_per_unit"),
        "peak_source": f"derived: {SM_COUNT} SM x {FP64_LANES_PER_SM} FP64 lanes x 2 flop x {sm_max:.0f} MHz (nominal clock; MEASURED_PEAKS.json has no FP64 entry)",
        "dfma_probe_tflops": probe_tf, "frac_of_dfma_probe": roofline["achieved"] / probe_tf})
    if wl["metric"] == "kerr" and not ad:
        # SURVEY 8(d)'s pre-kernel hand estimate, reported so that trimming arithmetic cannot hide in `frac`
        roofline["flop_per_step_survey_f_alg"] = F_ALG_SURVEY["kerr"]
        roofline["frac_survey_f_alg"] = ups * F_ALG_SURVEY["kerr"] / 1e12 / roofline["peak"]
        if kc.get("other"):
            # measured law of this kernel: an FP64 instruction holds the issue port 2 cycles, any other 1
            roofline["other_instr_per_step"] = kc["other"]
            roofline["issue_slot_util"] = ups * (2.0 * kc["pipe"] + kc["other"]) / (SM_COUNT * 4 * 32 * sm_max * 1e6)
    if wl["metric"] in ("tabulated", "tabulated_general"):
        node_b = 40 if wl["metric"] == "tabulated" else 96        # bytes per node record on the device
        roofline["table_bytes_per_step"] = 4 * 16 * node_b
        roofline["table_read_gbs"] = ups * 4 * 16 * node_b / 1e9
        tbl = wl["table"]["tab"]
        roofline["table_mb_on_device"] = tbl.shape[1] * tbl.shape[2] * node_b / 1e6
    if ad:
        roofline["unit_of_work"] = "one RK5(4) step attempt (accepted or rejected)"
    ncomp = bin(wl["snap_mask"] & 0xFF).count("1")
    rec_bytes = (run.records_per_pass or 0) * ncomp * 8
    if wl["snapshot_every"] == 1:
        # record-every-step runs: the bound to quote is HBM write bandwidth.  Algorithmic bytes per launch = every
        # record written once + inputs read + final records written.
        alg_bytes = rec_bytes + run.n * (48 + 100)
        hbm = float(peaks.get("hbm_gbs") or 6459.6)
        gbs = alg_bytes / (kernel_ms * 1e-3) / 1e9
        roofline = {"bound": "hbm", "achieved": gbs, "peak": hbm, "unit": "GB/s", "frac": gbs / hbm,
                    "traffic": TRAFFIC_NCU_BYTES.get(args.workload), "kernel": kc["kernel"], "kernel_ms": kernel_ms,
                    "algorithmic_bytes_per_launch": alg_bytes,
                    "peak_source": "MEASURED_PEAKS.json hbm_gbs (copy, read+write)" if peaks.get("hbm_gbs") else "fallback 6459.6 GB/s (MEASURED_PEAKS.json absent)",
                    "alu_view": roofline}

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        r = oracle_time(wl, 1, 0)
        cpu = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]}

    secondary = None
    if world == 1 and args.workload == "config4" and not args.no_secondary and args.n is None and args.flags == 0:
        c4 = dict(wl)
        run.close()
        del run
        torch.cuda.empty_cache()
        secondary = run_secondary(torch, geo, dev, sm_max, ncpu, peaks, c4)
        run = None

    config = {"workload": wl["name"], "n_per_gpu": int(sum(x.shape[1] for x in (wl.get("tiles") or [wl["st"]]))), "h": wl["h"],
              "nsteps": wl["nsteps"], "adaptive": ad,
              "geodesics_per_s": value / (tot_units / args.steps / max(1, world)) * int(sum(x.shape[1] for x in (wl.get("tiles") or [wl["st"]]))),
              "snapshot_every": wl["snapshot_every"], "geodesic_steps_per_pass_per_gpu": int(tot_units / args.steps / max(1, world)),
              "launches_per_pass": len(wl.get("tiles") or [1]), "record_bytes_written_per_pass": rec_bytes or None,
              "parallelism": (f"independent geodesics sharded by rank x{world}, no collective" if args.scaling == "weak" else
                              f"one image, interleaved row tiles over {world} rank(s), no collective"),
              "launch": info, "flags": args.flags | wl.get("flags", 0),
              "paper": ({"steps_per_s": wl["paper_steps_per_s"], "hardware": "GeForce GTX 960M, CUDA 7.5 (PAPER.md:446)",
                         "e2e_over_paper": (e2e["value"] / wl["paper_steps_per_s"]) if e2e else None}
                        if wl.get("paper_steps_per_s") else None),
              "l2": "inputs + final records exceed the 126 MB L2 at the full sizes; the state lives in registers (0 B/step)"}
    line = make_line(args, world, value, tmax_ms / args.steps, args.scaling, config, clocks, e2e, t["launches"], roofline, cpu,
                     secondary, vs_baseline=(value / wl["paper_steps_per_s"]) if wl.get("paper_steps_per_s") else None)
    print(json.dumps(line), flush=True)
    if run is not None:
        run.close()
    dist_finish(dist)


if __name__ == "__main__":
    main()
