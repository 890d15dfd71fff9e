#!/usr/bin/env python
"""bench.py -- LJ NVE particle-steps/s at N = 256,000 (BASELINE.json metric), B200.

One bench "step" = `--md-steps` (default 100) velocity-Verlet steps of config 3 through ONE
md_nve_step call: the whole hot path (kick/drift/rebuild test, conditional cell list + re-sort
+ neighbor list, LJ force + second kick), rebuilds amortised.  Defaults: 3 warm-up steps (the
jittered lattice melts), 20 timed steps = twice the config's 1000 MD steps.

  value      device-resident state, CUDA events per bench step on the launching stream,
             L2 flushed between bench steps (not timed), max over ranks
  e2e        the same metric through md_nve_run_host: pinned HOST buffers in, host buffers
             out, H2D + list build + steps + D2H all inside the timed region
  roofline   the force kernel (dominant) in the variant the step loop runs (no energy, second
             half-kick in the epilogue: md_force_half_kick): algorithmic bytes (4*Kbar + 68) * N
             per launch (SURVEY 8d / DESIGN.md §6) over its median duration, L2 flushed before
             every launch, against MEASURED_PEAKS.json's hbm_gbs; `traffic` = DRAM bytes per
             launch read from profiles/r2_traffic.json (one ncu --set full capture; the file
             names the capture and the build it was taken on), null when there is none for the config
  survey_timing  SURVEY 8(d)'s protocol beside the contract's: initial state restored, 50 warm-up
             steps, the config's own step count in ONE md_nve_step call, 5 repeats, median
  cpu_baseline  the fp64 oracle's own list-based loop on the host cores, bounded sample

`--impl reference` times the oracle (this tier's reference arm) instead.
N > 1 (torchrun): independent replicas, one per GPU, different seeds; no collective on the
data path ("replicas only").
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

METRIC = "LJ NVE particle-steps/sec at N=256k (incl. amortised rebuilds)"
UNIT = "particle-steps/s"
FALLBACK_HBM_GBS = 6650.0      # /opt/skills/guides/B200_PROFILING.md fallback
CONFIG_STEPS = {0: 100, 1: 1000, 2: 1000, 3: 1000, 4: 500}      # BASELINE.json: each config's own run length


def measured_traffic(config):
    """DRAM bytes per launch of the force kernel from the committed ncu capture, with its source."""
    p = os.path.join(ROOT, "profiles", "r2_traffic.json")
    try:
        t = json.load(open(p))[str(config)]
        return float(t["dram_bytes_per_launch"]), t["source"]
    except Exception:
        return None, None


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index")
    ap.add_argument("--md-steps", type=int, default=100, help="MD steps per bench step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--decompose", action="store_true",
                    help="time the split-list multi-GPU loop (SURVEY 8f-f1) instead: ONE system over all ranks, "
                         "strong scaling; not the contract line")
    ap.add_argument("--slabs", type=int, default=0,
                    help="time the slab decomposition (SURVEY 8f-f1, second version) with this many ranks stepped in "
                         "lockstep on ONE GPU: what the protocol costs, not a multi-GPU number; not the contract line")
    ap.add_argument("--next-rows", action="store_true",
                    help="time the SURVEY 8(f) rows instead (one JSON line per row; not the contract line)")
    ap.add_argument("--no-graph", action="store_true",
                    help="run md_nve_step as plain launches (same kernels, rebuild kernels return at once on a zero "
                         "flag): what a profiler can list kernel by kernel; not the contract line")
    ap.add_argument("--no-survey-timing", action="store_true")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """SM clocks and throttle reasons DURING the timed region (B200_PROFILING.md).  Two sources: the recipe's
    `nvidia-smi --query-gpu=... -lms 20`, started before the warm-up (start() waits for its first line, so the
    tool is already printing when the timed region begins), and the same counters read through NVML in this
    process every 10 ms.  nvidia-smi can take hundreds of ms per query on a busy box, which leaves a 160 ms timed
    region without a sample; the NVML samples then carry the numbers ("source" says which).  stop(t0, t1) keeps
    the samples whose timestamp falls inside [t0, t1] (host wall clock)."""
    Q = ("timestamp,index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []
        self.nvml, self.nvml_samples, self._run = None, [], False

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "20"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
            t_end = time.time() + 3.0
            while not self.lines and time.time() < t_end and self.proc.poll() is None:
                time.sleep(0.01)
        except Exception:
            self.proc = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nvml = pynvml
            self.handle = pynvml.nvmlDeviceGetHandleByIndex(self.index)
            self._run = True
            self.t2 = threading.Thread(target=self._poll, daemon=True)
            self.t2.start()
        except Exception:
            self.nvml = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def _poll(self):
        N = self.nvml
        bits = [("hw_slowdown", "nvmlClocksThrottleReasonHwSlowdown"),
                ("hw_thermal_slowdown", "nvmlClocksThrottleReasonHwThermalSlowdown"),
                ("sw_thermal_slowdown", "nvmlClocksThrottleReasonSwThermalSlowdown"),
                ("sw_power_cap", "nvmlClocksThrottleReasonSwPowerCap")]
        bits = [(n, getattr(N, a)) for n, a in bits if hasattr(N, a)]
        try:
            cmax = float(N.nvmlDeviceGetMaxClockInfo(self.handle, N.NVML_CLOCK_SM))
        except Exception:
            cmax = None
        while self._run:
            try:
                clk = float(N.nvmlDeviceGetClockInfo(self.handle, N.NVML_CLOCK_SM))
                mask = int(N.nvmlDeviceGetCurrentClocksThrottleReasons(self.handle))
                self.nvml_samples.append((time.time(), clk, cmax, [n for n, b in bits if mask & b]))
            except Exception:
                pass
            time.sleep(0.01)

    def stop(self, t0=None, t1=None):
        import datetime
        self._run = False
        if not self.proc and not self.nvml:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
        sm, mx, reasons, allsm = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 10:
                continue
            try:
                ts = datetime.datetime.strptime(f[0], "%Y/%m/%d %H:%M:%S.%f").timestamp()
                clk, cmax = float(f[2]), float(f[3])
            except ValueError:
                continue
            allsm.append(clk)
            if t0 is not None and not (t0 <= ts <= t1):
                continue
            sm.append(clk); mx.append(cmax)
            for name, v in zip(names, f[6:10]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        source = "nvidia-smi -lms 20"
        inside = [q for q in self.nvml_samples if t0 is None or t0 <= q[0] <= t1]
        if inside and len(inside) > len(sm):
            # the in-process NVML samples cover the region better: they carry the numbers, reasons are merged
            source = "NVML in process every 10 ms (nvidia-smi -lms 20 gave %d samples inside the region, %d in all)" % (len(sm), len(allsm))
            sm = [q[1] for q in inside]
            mx = [q[2] for q in inside if q[2] is not None] or mx
            for q in inside:
                reasons.update(q[3])
            allsm = [q[1] for q in self.nvml_samples]
        if self.nvml:
            try:
                self.nvml.nvmlShutdown()
            except Exception:
                pass
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "samples": len(sm),
                "samples_total": len(allsm), "reasons": sorted(reasons), "source": source}


def oracle_sample(w, md_steps):
    """The oracle's own list-based fp64 loop (build + force + velocity Verlet + half-skin
    rebuilds) on the host cores for `md_steps` steps of workload w. Returns seconds, threads."""
    from oracle import md_oracle as orc
    orc.build()
    diam = w.pos[:, 3].astype(np.float64)
    t0 = time.perf_counter()
    idx, cnt, _ = orc.neighbor_list(w.pos, w.box, w.dim, w.r_cut, w.skin, w.capacity, predicate=1, method=1)
    f0, _, _ = orc.energy_force(w.pos, diam, w.box, w.dim, w.kind, w.epsilon, w.sigma, w.r_cut, w.shift, idx, cnt)
    orc.nve_run(w.pos, w.vel, f0, diam, w.box, w.dim, w.kind, w.epsilon, w.sigma, w.r_cut, w.shift,
                w.dt, w.mass, md_steps, use_list=1, skin=w.skin, capacity=w.capacity, want_energies=False)
    return time.perf_counter() - t0, orc.num_threads()


def run_reference(args):
    """This tier's reference arm: the oracle as it stands, timed on the host cores; each
    bench step is a bounded sample of the same workload (about 1 s of wall time: the initial
    list build, then MD steps with the half-skin rebuilds they trigger)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1912_04232_b200 import workloads as W
    w = W.config(args.config)
    sample = {0: 2000, 1: 500, 2: 200, 3: 20, 4: 5}[args.config]
    for _ in range(min(args.warmup, 1)):
        oracle_sample(w, 1)
    times = []
    cores = 1
    for _ in range(args.steps):
        t, cores = oracle_sample(w, sample)
        times.append(t)
    total = sum(times)
    value = w.n * sample * args.steps / total
    desc = f"{sample} MD steps of config {args.config} (N={w.n}) per bench step incl. the initial list build and half-skin rebuilds"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": w.name, "n": w.n, "md_steps_per_step": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def run_next_rows(args):
    """SURVEY 8(f) rows on the headline geometry (config 3's particles and box unless stated):
    the pair force per launch (L2 flushed before each) for the other potentials, and us per step
    of the other update rules through their graph-captured loops (rebuilds amortised)."""
    import dataclasses
    import torch
    from paper_1912_04232_b200 import binding as B
    from paper_1912_04232_b200 import workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    base = W.config(args.config)
    n = base.n
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def emit(row, what, us, **kw):
        print(json.dumps({"row": row, "what": what, "n": kw.pop("n", n), "us": us, **kw}), flush=True)

    def time_force(S, reps=10):
        S.build(); S.compute_force()
        ts = []
        for _ in range(reps):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(); S.compute_force(want_energy=False); b.record()
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b) * 1e3)
        return statistics.median(ts)

    def time_rule(call, nsteps):
        call(nsteps)                                    # warm-up: graph capture, first rebuilds
        torch.cuda.synchronize()
        flush.fill_(1)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); call(nsteps); b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b) * 1e3 / nsteps

    # f2: the pair force of every potential on two states of the same particles, the lattice as generated
    # and the liquid it melts into; LJ, Morse and Buckingham on the fp32 fast path with fp64 re-evaluation
    # (their default) and on the fp64 pair chain ("fast32" = 0), species LJ and BKS on the chain only
    S = B.System(base)
    S.build(); S.compute_force(); S.step(400)
    torch.cuda.synchronize()
    liquid = np.empty_like(base.pos)
    liquid[S.id.cpu().numpy()] = S.pos.cpu().numpy()
    S.close()
    states = [("lattice as generated", base.pos), ("liquid, after 400 LJ steps", liquid)]
    eps = np.array([[1.0, 1.5], [1.5, 0.5]], np.float32)
    sig = np.array([[1.0, 0.8], [0.8, 0.88]], np.float32)
    one = np.ones((2, 2), np.float32)
    potentials = [
        ("LJ (the headline kernel)", dict(), True, None),
        ("Morse (D=1, alpha=5, r0=1.12)", dict(kind=W.KIND_MORSE, epsilon=1.0, sigma=1.12, alpha=5.0), True, None),
        ("Buckingham exp-6", dict(kind=W.KIND_BUCKINGHAM, epsilon=float(np.float32(9.02e5)),
                                  sigma=float(np.float32(3.454)), alpha=12.5), True, None),
        ("species x species LJ (80:20 binary mixture)", dict(kind=W.KIND_LJ_SPECIES), False,
         lambda S: B.md_set_species_lj(S.sys, eps, sig, (2.5 * sig).astype(np.float32))),
        ("BKS-type (exp-6 + damped shifted-force Coulomb, 2 species)", dict(kind=W.KIND_BKS, r_cut=2.5), False,
         lambda S: B.md_set_species_bks(S.sys, 9.02e5 * one, 12.5 * one, 3.454 * one,
                                        np.array([0.6, -0.6], np.float32), 0.3, 1.0)),
    ]
    for what, over, fast, setup in potentials:
        for sname, spos in states:
            pos = spos.copy()
            if setup is not None:
                pos[:, 3] = (np.arange(n) % 5 == 0).astype(np.float32)
            S = B.System(dataclasses.replace(base, pos=pos, **over))
            if setup is not None:
                setup(S)
            if fast:
                emit("f2", f"{what} force, fp32 fast path with fp64 re-evaluation", time_force(S), state=sname)
                B.md_set_option(S.sys, "fast32", 0)
            emit("f2", f"{what} force, fp64 pair chain", time_force(S), state=sname)
            S.close()

    # f3: update rules, LJ fast path, 200 steps each
    steps = 200
    S = B.System(base); S.build(); S.compute_force()
    emit("f3", "NVE (fused graph; for scale)", time_rule(lambda k: S.step(k), steps), steps=steps); S.close()
    S = B.System(base); S.build(); S.compute_force()
    emit("f3", "Brownian dynamics kT=0.8 gamma=1", time_rule(lambda k: B.md_brownian_step(
        S.sys, S.pot, S.pos, S.force, S.id, S.nbr_idx, S.nbr_count, 1e-4, 1.0, 0.8, 7, 0, k, S.stats), steps),
        steps=steps); S.close()
    S = B.System(base); S.build(); S.compute_force()
    emit("f3", "Langevin (BAOAB) kT=1 gamma=1", time_rule(lambda k: B.md_langevin_step(
        S.sys, S.pot, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, base.dt, base.mass, 1.0, 1.0, 7, 0, k,
        S.stats), steps), steps=steps); S.close()
    S = B.System(base); S.build(); S.compute_force()
    nh = torch.zeros(2, dtype=torch.float64, device=dev)
    emit("f3", "Nose-Hoover kT=1 tau=0.2", time_rule(lambda k: B.md_nose_hoover_step(
        S.sys, S.pot, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, base.dt, base.mass, 1.0, 0.2, nh, k,
        S.stats), steps), steps=steps); S.close()
    w = dataclasses.replace(base, vel=np.zeros_like(base.vel))
    S = B.System(w); S.build(); S.compute_force()
    fs = torch.zeros(4, dtype=torch.float32, device=dev)
    fp = B.md_fire_params(0.002, 0.02, 5, 1.1, 0.5, 0.1, 0.99)
    emit("f3", "FIRE minimisation", time_rule(lambda k: B.md_fire_minimize(
        S.sys, S.pot, fp, S.pos, S.vel, S.force, S.id, S.nbr_idx, S.nbr_count, fs, k, S.stats), steps),
        steps=steps); S.close()

    # f4: flocking, 2-D, 262,144 boids on a strongly jittered square lattice, spacing 1.26 (~24 neighbors in
    # R + skin).  Jitter 0.4: with a weak jitter every boid is surrounded evenly, the cohesion term of eq. 10
    # is singular (|Delta R| -> 0) and some boid jumps past skin / 2 every step (a rebuild per step: round 1)
    m = 512
    nb = m * m
    L = np.float32(m * 1.26 + 0.37)
    rng = np.random.default_rng(5)
    g = (np.arange(m) + 0.5) * (float(L) / m)
    box = np.array([L, L, 1.0], np.float32)
    p = np.zeros((nb, 4), np.float32)
    p[:, :2] = W.into_box_f32(np.stack(np.meshgrid(g, g, indexing="ij"), -1).reshape(-1, 2)
                              + rng.normal(0, 0.4, (nb, 2)), box)
    p[:, 3] = rng.uniform(-np.pi, np.pi, nb).astype(np.float32)
    w = dataclasses.replace(base, name="flock2d", n=nb, dim=2, box=box, pos=p, vel=np.zeros((nb, 4), np.float32),
                            kind=W.KIND_SOFT, r_cut=3.0, skin=0.5, capacity=64)
    # (a) alignment + avoidance: the well-conditioned part of the model (rebuilds amortised over many steps);
    # (b) with the cohesion term of eq. 10, whose gradient ~ J / |Delta R| is unbounded: among 262,144 boids
    #     one is always surrounded evenly enough to jump past skin / 2 in a step, so the list is rebuilt every
    #     step whatever the initial state -- that line times flocking pass + rebuild, and says so
    par_aa = B.md_flock_params(1.0, 3.0, 10.0, 1.0, 0.0, 3.0, 3.0, 0.5)
    par = B.md_flock_params(1.0, 3.0, 10.0, 1.0, 0.5, 3.0, 3.0, 0.5)
    for what, pr in (("flocking (align + avoid), forward Euler", par_aa),
                     ("flocking (align + avoid + cohesion: singular gradient, a rebuild per step), forward Euler", par)):
        S = B.System(w); S.build()
        us = time_rule(lambda k: B.md_flock_step(S.sys, pr, S.pos, S.id, S.nbr_idx, S.nbr_count, 0.01, k, S.stats), steps)
        emit("f4", what, us, steps=steps, n=nb, rebuilds=int(S.stats[1]), mean_neighbors=float(S.nbr_count.float().mean()))
        S.close()
    S = B.System(w); S.build()
    cen = rng.uniform(5.0, float(L) - 5.0, (16, 2)).astype(np.float32)
    B.md_flock_obstacles(S.sys, cen, np.full(16, 4.0, np.float32), 4.0)
    pred = torch.zeros(16, 4, dtype=torch.float32, device=dev)
    pred[:, :2] = torch.from_numpy(rng.uniform(5.0, float(L) - 5.0, (16, 2)).astype(np.float32)).to(dev)
    B.md_flock_predators(S.sys, pred, B.md_predator_params(5.0, 4.0, 3.0, 12.0, 0.8))
    us = time_rule(lambda k: B.md_flock_step(S.sys, par, S.pos, S.id, S.nbr_idx, S.nbr_count, 0.01, k, S.stats), steps)
    emit("f4", "flocking + 16 disk obstacles + 16 predators", us, steps=steps, n=nb, rebuilds=int(S.stats[1]))
    S.close()


def run_slabs(args):
    """SURVEY 8(f)-f1, second version: `--slabs P` ranks (slabs along x with halos; paper_1912_04232_b200/slabs.py)
    of config `--config`, all in this process on one GPU, stepped in lockstep.  One GPU executes the work of P
    ranks one after the other, so us_per_md_step is (sum over ranks) and says what the decomposition costs in
    total work -- halo copies, per-step exchange, host-driven phases -- against md_nve_step on one context."""
    import torch
    from paper_1912_04232_b200 import binding as B
    from paper_1912_04232_b200 import slabs as SL
    from paper_1912_04232_b200 import workloads as W
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    w = W.config(args.config)
    run = SL.SlabRun(B, w, args.slabs)
    for _ in range(args.warmup):
        run.step(args.md_steps)
    torch.cuda.synchronize()
    r0 = run.rebuilds
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    for _ in range(args.steps):
        run.step(args.md_steps)
    b.record()
    torch.cuda.synchronize()
    ms = a.elapsed_time(b)
    total = args.steps * args.md_steps
    owned = [int((S.id[: S.n] >= 0).sum()) for S in run.ranks]
    print(json.dumps({
        "mode": "slabs", "metric": METRIC, "value": w.n * total / (ms * 1e-3), "unit": UNIT, "n_gpus": 1,
        "ranks_on_this_gpu": args.slabs, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
        "us_per_md_step_all_ranks": 1e3 * ms / total, "higher_is_better": True, "dtype": "f32", "data": "synthetic",
        "config": {"workload": w.name, "n": w.n, "md_steps_per_step": args.md_steps,
                   "parallelism": f"{args.slabs} slabs along x with halos of width r_cut + skin, in lockstep on one GPU"},
        "rebuilds": run.rebuilds - r0, "owned_per_rank": owned, "local_per_rank": [S.n for S in run.ranks],
        "rows_per_step_per_link": run.exchange_plan()}))
    run.close()


def run_decomposed(args):
    """one system of config `--config` over all ranks (replicated positions, split list;
    paper_1912_04232_b200/decomposition.py).  A bench step is `--md-steps` MD steps; device time by CUDA
    events on the current stream, max over ranks; value = N * md_steps / that time (strong scaling).  With
    one rank it measures what the host-driven step costs against md_nve_step's graph."""
    import torch
    import torch.distributed as dist
    from paper_1912_04232_b200 import binding as B
    from paper_1912_04232_b200 import decomposition as D
    from paper_1912_04232_b200 import replicas as R
    from paper_1912_04232_b200 import workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
        exchange = D.DistExchange()
    else:
        class Solo:
            def all_gather(self, slot):
                return slot.unsqueeze(0)
        exchange = Solo()
    w = W.config(args.config)                       # the SAME system on every rank
    S = B.System(w, device=dev)
    loop = D.RankLoop(S, rank, world)
    loop.start()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(args.warmup):
        D.run(loop, exchange, args.md_steps)
    barrier()
    r0 = loop.rebuilds
    ms = 0.0
    for _ in range(args.steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        D.run(loop, exchange, args.md_steps)
        b.record()
        torch.cuda.synchronize(dev)
        ms += a.elapsed_time(b)
    barrier()
    ms = R.max_over_ranks(ms, dev) if world > 1 else ms
    if rank == 0:
        total = args.steps * args.md_steps
        print(json.dumps({
            "mode": "decompose", "metric": METRIC, "value": w.n * total / (ms * 1e-3), "unit": UNIT,
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
            "us_per_md_step": 1e3 * ms / total, "higher_is_better": True, "scaling": "strong",
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "n": w.n, "md_steps_per_step": args.md_steps,
                       "parallelism": f"split list x{world} (replicated positions, one all-gather per step)"},
            "rebuilds": loop.rebuilds - r0, "range_rank0": list(loop.range)}))
    if world > 1:
        dist.destroy_process_group()


def respawn_under_torchrun(args):
    """`python bench.py --gpus N` without torchrun: start N ranks on this node ourselves."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    raise SystemExit(subprocess.call(cmd))


def main():
    args = parse()
    if args.gpus < 1:
        raise SystemExit("--gpus must be >= 1")
    if "WORLD_SIZE" not in os.environ and args.gpus > 1:
        return respawn_under_torchrun(args)
    if int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={os.environ.get('WORLD_SIZE', '1')}: launch one rank per GPU")
    if args.impl == "reference":
        return run_reference(args)
    if args.next_rows:
        return run_next_rows(args)
    if args.decompose:
        return run_decomposed(args)
    if args.slabs:
        return run_slabs(args)

    import torch
    import torch.distributed as dist
    from paper_1912_04232_b200 import binding as B
    from paper_1912_04232_b200 import replicas as R
    from paper_1912_04232_b200 import workloads as W

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    if local >= torch.cuda.device_count():
        raise SystemExit(f"rank {rank}: local rank {local} but only {torch.cuda.device_count()} CUDA device(s) here")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    B.lib()

    # replicas: rank r simulates an independent sample of the same config
    w = W.config(args.config, replica=R.replica_index(rank))
    S = B.System(w, device=dev)
    if args.no_graph:
        B.md_set_option(S.sys, "use_graph", 0)
    stream = torch.cuda.Stream(device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # 2x the 126 MB L2
    md_steps = args.md_steps

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    with torch.cuda.stream(stream):
        S.build(stream)
        S.compute_force(True, stream)
        sampler = ClockSampler(local)
        sampler.start()
        for _ in range(args.warmup):
            S.step(md_steps, stream)
        barrier()
        t_region0 = time.time()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
              for _ in range(args.steps)]
        rebuilds = 0
        stats_acc = []
        for a, b in ev:
            flush.zero_()
            a.record(stream)
            S.step(md_steps, stream)
            b.record(stream)
            stats_acc.append(S.stats.clone())
        barrier()
        clocks = sampler.stop(t_region0, time.time())
        ms = sum(a.elapsed_time(b) for a, b in ev)
        rebuilds = int(sum(int(s[1]) for s in stats_acc))
        max_count = int(max(int(s[3]) for s in stats_acc))
        overflow = any(int(s[2]) >= 0 for s in stats_acc)

        # ---- roofline of the force kernel: the loop's variant (no energy, half-kick in the epilogue,
        # on a scratch copy of the velocities), cold L2, event pair per launch
        kbar = float(S.nbr_count.float().mean())
        reps = 30
        vel_scratch = S.vel.clone()

        def force_launch():
            B.md_force_half_kick(S.sys, S.pot, S.pos, S.nbr_idx, S.nbr_count, S.force, vel_scratch, w.dt, w.mass, stream)

        fev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        for a, b in fev:
            flush.zero_()
            a.record(stream)
            force_launch()
            b.record(stream)
        torch.cuda.synchronize(dev)
        force_ms_cold = statistics.median(a.elapsed_time(b) for a, b in fev)
        a0, b0 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a0.record(stream)
        for _ in range(reps):
            force_launch()
        b0.record(stream)
        torch.cuda.synchronize(dev)
        force_ms_warm = a0.elapsed_time(b0) / reps
        # ---- one rebuild (cell list + re-sort + neighbor list) through the API, cold L2
        bev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(10)]
        for a, b in bev:
            flush.zero_()
            a.record(stream)
            S.build(stream)
            b.record(stream)
        torch.cuda.synchronize(dev)
        build_ms = statistics.median(a.elapsed_time(b) for a, b in bev)
        S.compute_force(False, stream)

        # ---- initial state, 50 warm-up steps, the config's step count in one call, 5 repeats
        survey = None
        if not args.no_survey_timing:
            nst = CONFIG_STEPS[args.config]
            ts, rb = [], []
            for _ in range(5):
                S.reset()
                S.build(stream); S.compute_force(False, stream)
                S.step(50, stream)
                a1, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a1.record(stream)
                S.step(nst, stream)
                b1.record(stream)
                torch.cuda.synchronize(dev)
                ts.append(a1.elapsed_time(b1)); rb.append(int(S.stats[1]))
            t_med = statistics.median(ts)
            survey = {"md_steps": nst, "repeats": 5, "warmup_md_steps": 50, "state": "restored initial state per repeat",
                      "median_ms": t_med, "us_per_md_step": 1e3 * t_med / nst,
                      "particle_steps_per_s": w.n * nst / (t_med * 1e-3), "rebuilds": rb[len(rb) // 2]}

    ms_max = R.max_over_ranks(ms, dev)
    value = R.whole_job_rate(w.n * md_steps * args.steps, ms_max * 1e-3)

    # ---- e2e through the host-buffer entry point (pinned host memory)
    e2e = None
    if not args.no_e2e:
        pos_h = torch.from_numpy(w.pos.copy()).pin_memory()
        vel_h = torch.from_numpy(w.vel.copy()).pin_memory()
        force_h = torch.zeros_like(pos_h).pin_memory()
        stats_h = np.zeros(4, np.int32)
        B.md_nve_run_host(S.cfg, S.pot, pos_h, vel_h, force_h, w.dt, w.mass, md_steps, stats_h)  # warm
        e2e_steps = max(1, min(args.steps, 5))
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            B.md_nve_run_host(S.cfg, S.pot, pos_h, vel_h, force_h, w.dt, w.mass, md_steps, stats_h)
        barrier()
        dt_e2e = time.perf_counter() - t0
        e2e = {"value": R.whole_job_rate(w.n * md_steps * e2e_steps, R.max_over_ranks(dt_e2e, dev)), "unit": UNIT,
               "h2d_bytes_per_step": 2 * w.n * 16, "d2h_bytes_per_step": 3 * w.n * 16 + 8 + 16,
               "what": f"md_nve_run_host: pinned host pos/vel in, list build + {md_steps} MD steps, host pos/vel/force/energy/stats out"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peak, peak_src = peaks()
    traffic, traffic_src = measured_traffic(args.config)
    fused = (w.kind == W.KIND_LJ and w.dim == 3)      # the configs md_nve_step runs as fused graphs
    flagged = B.md_get_option(S.sys, "rebuild_flagged") != 0.0
    forked = B.md_get_option(S.sys, "step_fork") != 0.0
    algo_bytes = (4.0 * kbar + 68.0) * w.n          # list + count + pos + vel read, force + vel written
    achieved = algo_bytes / (force_ms_cold * 1e-3) / 1e9
    step_bytes = (4.0 * kbar + 164.0) * w.n
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": f"BASELINE.json configs[{args.config}]: {w.name}, rho=0.8442, r_cut=2.5, "
                               f"skin={w.skin}, capacity={w.capacity}, dt={w.dt}, re-sort at every rebuild",
                   "n": w.n, "md_steps_per_step": md_steps, "parallelism": f"replicas x{world}",
                   "l2": "flushed (256 MiB write) between bench steps; inside a bench step the loop "
                         "re-reads its own ~100 MB working set every MD step as in production",
                   "precision": "fp32 state; pair terms fp32 with fp64 re-evaluation where the error "
                                "estimate requires it (DESIGN.md §5)"},
        "us_per_md_step": 1e3 * ms_max / (args.steps * md_steps),
        "rebuilds": rebuilds, "md_steps_per_rebuild": (args.steps * md_steps) / max(1, rebuilds),
        "max_neighbors": max_count, "overflow": overflow,
        "step_hbm_frac": step_bytes / (1e3 * ms_max / (args.steps * md_steps) * 1e-6) / 1e9 / peak,
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": "force kernel of the step loop: no energy, second half-kick in the "
                                               "epilogue (md_force_half_kick)" if fused else "force kernel (md_force_half_kick)",
                     "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": traffic, "traffic_source": traffic_src,
                     "peak_source": peak_src, "algorithmic_bytes": algo_bytes, "kbar": kbar,
                     "launch_ms_cold_l2": force_ms_cold, "launch_ms_warm_l2": force_ms_warm},
        # per bench step: k_init_stats + one force kernel per MD step + one k_kick_drift per graph
        # launch (graphs of 9 fused steps, then single steps; unfused configs: one per MD step)
        # + the rebuild: two flagged launches (cooperative cell list, builder) in EVERY MD step, or
        # 6 kernels (4 cell list, copy back, neighbor list) per rebuild an IF node ran
        # (in the fused loop the flagged rebuild sits on a side branch that ends in a second launch of the force
        # kernel: of the step's two force launches the one whose turn it is not returns at once)
        "gpu_launches": args.steps * (1 + md_steps + (md_steps // 9 + md_steps % 9 if fused else md_steps))
                        + ((3 if fused and forked else 2) * args.steps * md_steps if flagged else 6 * rebuilds),
        "rebuild_in_graph": ("two launches per MD step that return at once while the step's flag is 0"
                             + (", on a branch beside the force kernel that ends in a second, conditional force launch"
                                if fused and forked else "")) if flagged
                            else "IF node around the rebuild's six kernels",
    }
    if build_ms is not None:
        out["build_ms_per_rebuild"] = build_ms
        # BASELINE.json config 4 asks for these three side by side (reported for every config)
        out["three_numbers"] = {"neighbor_build_us_per_rebuild": 1e3 * build_ms,
                                "pair_force_us_per_step": 1e3 * force_ms_cold,
                                "nve_particle_steps_per_s": value,
                                "what": "cell list + re-sort + neighbor list through the API (cold L2) / the loop's force kernel "
                                        "per launch (cold L2) / the whole loop incl. rebuilds"}
        # the rebuild (cell list with re-sort + neighbor list) on its own algorithmic bytes, (4K + 116) N
        rebuild_bytes = (4.0 * kbar + 116.0) * w.n
        rb_achieved = rebuild_bytes / (build_ms * 1e-3) / 1e9
        out["roofline_rebuild"] = {"bound": "alu (instruction issue; profiles/r2_profiles.md), reported against hbm",
                                   "kernels": "k_cell_assign, k_cell_scan, k_cell_scatter, k_cell_order_gather, k_copy_back, k_nbr_build2",
                                   "achieved": rb_achieved, "peak": peak, "unit": "GB/s", "frac": rb_achieved / peak,
                                   "algorithmic_bytes": rebuild_bytes, "ms_per_rebuild_cold_l2": build_ms}
    if survey is not None:
        out["survey_timing"] = survey
    if e2e is not None:
        out["e2e"] = e2e
    if not args.no_cpu_baseline:
        # about 5-10 s of wall time on 16 host cores (80-160 core-seconds) per config
        sample_steps = {0: 10000, 1: 5000, 2: 1500, 3: 150, 4: 30}[args.config]
        t, cores = oracle_sample(w, sample_steps)
        out["cpu_baseline"] = {"value": w.n * sample_steps / t, "unit": UNIT, "cores": cores,
                               "kind": "oracle",
                               "sample": f"{sample_steps} MD steps of the same workload (N={w.n}) incl. the "
                                         f"initial list build and half-skin rebuilds, {t:.1f} s"}
    print(json.dumps(out))
    S.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
