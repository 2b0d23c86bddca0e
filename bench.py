#!/usr/bin/env python
"""bench.py -- throughput of the MD hot path (BASELINE.json: particle-steps/sec for LJ at N=1M on one B200).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--scale s] [--impl ours|reference]

A "step" is one MD time step of md_step: half-kick + drift + displacement check, (when the check fires) cell binning +
neighbour-list rebuild, pair (+ bond) forces, half-kick -- i.e. one pass of every row of SURVEY.md 8(a); rebuilds fall
inside the timed region at their natural frequency.  N = 1 runs config 2 (LJ, N = 1,048,576, mixed precision).
Multi-GPU: "replicas only": every rank runs an independent replica, no collective on the data path; the
time is the max over ranks, the value the sum of all ranks' particle-steps.

Prints ONE JSON line (see the keys below).  `--impl reference` times the CPU oracle (a bounded sample per step).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "particle-steps/sec"
UNIT = "particle-steps/s"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def ncu_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel, from the committed
    `ncu --set full` captures (profiles/ncu_traffic.json: one entry per workload and kernel, stamped with the hash of
    the kernel source it was taken from).  None if there is no capture, or if the source has changed since (stale)."""
    import hashlib
    try:
        tab = json.load(open(os.path.join(ROOT, "profiles", "ncu_traffic.json")))
        src = open(os.path.join(ROOT, "paper_1412_3387_b200", "csrc", "tiles.cu"), "rb").read()
        sha = hashlib.sha256(src).hexdigest()[:16]
        for e in tab["entries"]:
            if e["workload"] == workload and e["kernel"] == kernel:
                return (float(e["dram_bytes_per_launch"]), None) if e["tiles_cu_sha16"] == sha else (
                    None, "capture %s is of tiles.cu %s, now %s" % (e.get("file", "?"), e["tiles_cu_sha16"], sha))
    except Exception as ex:  # noqa: BLE001
        return None, "profiles/ncu_traffic.json: %s" % ex
    return None, "no capture of this workload/kernel"


def measured_hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index=0):
        self.gpu = gpu_index
        self.rows = []
        self.first = 0
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
            t0 = time.time()
            while not self.rows and time.time() - t0 < 5.0:     # nvidia-smi takes ~0.1 s to print its first row
                time.sleep(0.005)
        except Exception:
            self.proc = None
        self.first = len(self.rows)                              # rows from here on fall inside the timed region

    def count(self):
        return len(self.rows) - self.first

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows[self.first:]:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def workload_for(args):
    from paper_1412_3387_b200 import inputs
    w = inputs.config(args.config, scale=args.scale)
    if getattr(args, "r_buff", None):
        # the paper tunes r_buff per benchmark; the configured value (0.4) stays
        # the default of every reported run, this override is for the tuning sweep only and is named in the workload
        import dataclasses
        w = dataclasses.replace(w, r_buff=float(args.r_buff), name=w.name + "-rbuff%g" % args.r_buff)
    return w


def algorithmic_ops(kind, nbar, rc, r_list):
    """SURVEY.md 8(d) "arithmetic work for context", per particle and force evaluation, as lane-instructions (an FMA
    counts once): n_bar distance tests of ~9 instructions (3 subtractions, 3 multiply-adds, compare, minimum image
    amortised) and n_c = n_bar (rc / r_list)^3 in-range pair terms -- LJ 7 instructions + 1 reciprocal; DPD 12 fp64
    instructions + rsqrt and ~70 integer instructions of Philox4x32-10."""
    n_c = nbar * (rc / r_list) ** 3
    if kind == "lj":
        return {"fp": 9.0 * nbar + 8.0 * n_c, "int": 0.0}
    return {"fp": 9.0 * nbar + 13.0 * n_c, "int": 70.0 * n_c}


def algorithmic_bytes(kind, nbar, k):
    """B_min per particle-step (strict, fully-fused ideal) and the staged minimum of the pair-force
    kernel (index stream + own position + force write [+ velocity and tag for DPD])."""
    dpd = kind in ("dpd", "polymer")
    b_min = 4.0 * nbar * (1.0 + 1.0 / k) + 120.0 + (4.0 if dpd else 0.0) + 130.0 / k
    force_kernel = 4.0 * nbar + (84.0 if dpd else 56.0)
    return b_min, force_kernel


# ----------------------------------------------------------------------------------------------------------------
def cpu_baseline(w, budget_s=15.0):
    """The oracle as it stands, one host core, on a bounded sample: force rows of M probe particles against all N
    (O(M N) brute force, oracle O9).  Value = probe rows per second = particle force evaluations per second, the
    dominant cost of a particle-step (integration is negligible next to the O(N) pair search per particle)."""
    import oracle
    from paper_1412_3387_b200 import inputs
    M = 8
    t_used, rows = 0.0, 0
    p = w.params
    while True:
        pr = inputs.probe_tags(w.N, M, seed=99 + M)
        t0 = time.perf_counter()
        if w.kind == "lj":
            oracle.probe_forces_lj(w.pos, w.box, w.rc, pr, p["epsilon"], p["sigma"], p["energy_shift"])
        else:
            oracle.probe_forces_dpd(w.pos, w.vel, w.box, w.rc, p["A"], p["gamma"], p["kT"], w.dt, 1, p["seed"], pr)
        dt = time.perf_counter() - t0
        t_used += dt; rows += len(pr)
        rate = len(pr) / dt
        if t_used > 0.6 * budget_s or len(pr) >= w.N:
            break
        M = int(min(w.N, max(2 * M, 0.5 * (budget_s - t_used) * rate)))
    return {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"pair-force rows of {len(pr)} seeded probe particles against all N={w.N} "
                      f"(O(M*N) brute force, oracle/md_oracle.c orc_probe_forces_*), {dt:.1f} s on 1 core; "
                      f"full step extrapolated = N/M x this"}


def run_reference(args):
    """--impl reference: the oracle, timed per 'step' on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    from paper_1412_3387_b200 import inputs
    w = workload_for(args)
    p = w.params
    # size the per-step sample so that the whole run stays within a few minutes
    probe = inputs.probe_tags(w.N, 4, seed=5)
    t0 = time.perf_counter()
    oracle.probe_forces_lj(w.pos, w.box, w.rc, probe) if w.kind == "lj" else oracle.probe_forces_dpd(
        w.pos, w.vel, w.box, w.rc, p["A"], p["gamma"], p["kT"], w.dt, 1, p["seed"], probe)
    per_row = (time.perf_counter() - t0) / len(probe)
    budget = 120.0 / max(1, args.steps + args.warmup)
    M = int(max(1, min(w.N, budget / per_row)))
    times = []
    for s in range(args.warmup + args.steps):
        pr = inputs.probe_tags(w.N, M, seed=1000 + s)
        t0 = time.perf_counter()
        if w.kind == "lj":
            oracle.probe_forces_lj(w.pos, w.box, w.rc, pr, p["epsilon"], p["sigma"], p["energy_shift"])
        else:
            oracle.probe_forces_dpd(w.pos, w.vel, w.box, w.rc, p["A"], p["gamma"], p["kT"], w.dt, s, p["seed"], pr)
        if s >= args.warmup:
            times.append(time.perf_counter() - t0)
    t = float(np.sum(times))
    value = M * len(times) / t
    sample = (f"each step = pair-force rows of {M} seeded probe particles against all N={w.N} (O(M*N) brute force); "
              f"value = rows/s = particle force evaluations/s")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / len(times),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "precision": w.precision},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------------------------------------------
def replica_max_times(times_ms, world, device):
    """Replicas only: no collective on the data path; the only exchange of a multi-rank run is this
    MAX over the ranks' timed regions (device-timed, max over ranks)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def aggregate_value(n_particles, steps, world, ms_max):
    """Whole-job particle-steps/s of `world` independent replicas of n_particles each, timed by the slowest rank."""
    return world * n_particles * steps / (ms_max * 1e-3)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1412_3387_b200 import binding as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = workload_for(args)
    precision = B.MD_MIXED if w.precision == "mixed" else B.MD_FP64
    stream = torch.cuda.Stream()
    order = {"lex": B.MD_ORDER_LEX, "morton": B.MD_ORDER_MORTON, "hilbert": B.MD_ORDER_HILBERT}[args.order]
    # device memory comes from torch (md_workspace_bytes -> torch.empty -> md_set_workspace); streams too
    md = B.MD(w.box, w.N, w.rc, w.r_buff, precision=precision, stream=stream.cuda_stream, order=order,
              sched={"sync": B.MD_SCHED_SYNC, "speculative": B.MD_SCHED_SPECULATIVE, "batch": B.MD_SCHED_BATCH}[args.sched],
              workspace=None if args.own_alloc else "torch")
    # measured issue rates of the pipes the pair-force kernel runs on (md_debug_peak), before the timed region
    peaks = {k: md.debug_peak(k) for k in ("fp32_fma", "fp64_fma", "int32_mad")} if rank == 0 else {}
    nvt = None
    if args.nvt or args.mtk:
        import dataclasses
        kT = float(w.params.get("kT", 1.2 if args.config == 2 else 1.0))
        nvt = dict(kT=kT, tau=0.5)
        if args.mtk:                     # the Martyna-Tobias-Klein update (R39) instead of the R30 scheme
            nvt["scheme"] = "mtk"
        w = dataclasses.replace(w, name=w.name + ("-nvt-mtk" if args.mtk else "-nvt"))
    angles = None
    if (args.angles or args.dihedrals) and w.kind == "polymer":
        # harmonic angles along the chains of the polymer melt (k = 5, theta0 = 2.0 rad); named in the
        # workload, not a BASELINE configuration
        import dataclasses
        L = 64
        nc = w.N // L
        idx = (np.arange(nc, dtype=np.uint32)[:, None] * L + np.arange(L - 2, dtype=np.uint32)[None, :]).reshape(-1)
        angles = np.stack([idx, idx + 1, idx + 2], axis=1).astype(np.uint32)
        # with dihedrals the angles are stiff (k = 50): the dihedral force grows as 1 / sin of the bond angles, and chains
        # that may straighten (k = 5) throw particles across the skin in one step (dangerous builds)
        ka = 50.0 if args.dihedrals else 5.0
        w = dataclasses.replace(w, name=w.name + ("-angles%g" % ka if args.dihedrals else "-angles"),
                                params=dict(w.params, angle_k=ka, angle_theta0=2.0))
    dihedrals = None
    if args.dihedrals and w.kind == "polymer":
        # periodic dihedrals along the chains, U = k/2 (1 + cos phi), k = 2 (R35); named in the workload
        import dataclasses
        L = 64
        nc = w.N // L
        idx = (np.arange(nc, dtype=np.uint32)[:, None] * L + np.arange(L - 3, dtype=np.uint32)[None, :]).reshape(-1)
        dihedrals = np.stack([idx, idx + 1, idx + 2, idx + 3], axis=1).astype(np.uint32)
        w = dataclasses.replace(w, name=w.name + "-dihedrals",
                                params=dict(w.params, dihedral_k=2.0, dihedral_sign=1, dihedral_n=1))
    desc = B.step_desc(w.kind, w.dt, w.params, nvt=nvt)

    # inputs resident in HBM before the timed region
    d_pos = torch.from_numpy(w.pos).to("cuda")
    d_vel = torch.from_numpy(w.vel).to("cuda")
    torch.cuda.synchronize()
    md.set_state(d_pos, d_vel)
    if w.bonds is not None:
        md.set_bonds(w.bonds)
    if angles is not None:
        md.set_angles(angles)
    if dihedrals is not None:
        md.set_dihedrals(dihedrals)
    if args.brick:
        md.set_option(B.MD_OPT_TILE_BRICK, args.brick)
        md.set_state(d_pos, d_vel)
        if w.bonds is not None:
            md.set_bonds(w.bonds)
    for spec in args.launch:                       # e.g. --launch lj=256,4 nlist=768,32 (fixes a kernel's block, w)
        name, val = spec.split("=")
        blk, ww = (int(x) for x in val.split(","))
        md.set_launch({v: k for k, v in B.KERNEL_NAMES.items()}[name], blk, ww)
    if not args.no_tune:
        md.tune(desc, False)
    if args.auto_rbuff:
        # the library picks the skin with the most steps per second (md_tune_rbuff); named in the
        # workload -- the reported BASELINE configuration keeps r_buff = 0.4
        import dataclasses
        # the bursts must see the state the run will be in: first past the start-up transient (a melt built as random walks
        # relaxes for ~100 steps with faster particles, which favours a larger skin than the steady state does)
        md.step(desc, max(200, args.warmup))
        rb = md.tune_rbuff(desc, None, 300)
        w = dataclasses.replace(w, r_buff=rb, name=w.name + "-autorbuff%g" % rb)
        if not args.no_tune:
            md.tune(desc, False)

    # ---- device-resident timing ---------------------------------------------------------------------------
    md.step(desc, max(3, args.warmup))
    # the end-to-end leg below starts from this same state (pinned host copy), so both legs time the same K steps
    h_pos = torch.empty((w.N, 3), dtype=torch.float64).pin_memory()
    h_vel = torch.empty((w.N, 3), dtype=torch.float64).pin_memory()
    md.get_state(h_pos, h_vel, None)
    torch.cuda.synchronize()
    # ... of every `ev_stride`-th launch: two events per launch cost a 30 us step (config 1) a third of its time
    ev_stride = 16 if args.steps >= 64 else 1
    md.set_option(B.MD_OPT_PROFILE_STRIDE, ev_stride)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    # three repetitions of exactly `steps` steps each (the trajectory continues); the median one is reported
    reps = []
    for rep in range(1 if args.reps < 2 else args.reps):
        ra = md.stats()
        md.set_profiling(2)        # CUDA events around the pair-force stage only (the roofline kernel) ...
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        barrier()
        with torch.cuda.stream(stream):
            e0.record(stream)
            md.step(desc, args.steps)
            e1.record(stream)
        barrier()
        reps.append((e0.elapsed_time(e1), ra, md.stats()))
    # a timed region shorter than a few sample periods (config 1: 30 us per step) is followed by an untimed continuation
    # of the same steps until the sampler has seen the GPU under this load at least 3 times
    extra_steps = 0
    if rank == 0 and sampler.proc:
        while sampler.count() < 3 and extra_steps < 200 * args.steps:
            md.step(desc, args.steps)
            extra_steps += args.steps
    clocks = sampler.stop() if rank == 0 else None
    if clocks is not None and extra_steps:
        clocks["note"] = "timed region shorter than 3 sample periods: sampling continued over %d more steps of the same run" % extra_steps
    rep_ms = [r[0] for r in reps]
    # stage shares: a short untimed continuation with every stage bracketed by events (about 8 events per step)
    md.set_option(B.MD_OPT_PROFILE_STRIDE, 1)
    md.set_profiling(1)
    n_share = max(20, min(200, args.steps // 4))
    with torch.cuda.stream(stream):
        s0 = torch.cuda.Event(enable_timing=True); s1 = torch.cuda.Event(enable_timing=True)
        s0.record(stream)
        md.step(desc, n_share)
        s1.record(stream)
    torch.cuda.synchronize()
    ms_share = s0.elapsed_time(s1)
    st_share = md.stats()
    md.set_profiling(0)

    # ---- end to end through the C-ABI with HOST buffers: upload state, K steps, download state ----------------
    o_pos = torch.empty_like(h_pos).pin_memory()
    o_vel = torch.empty_like(h_vel).pin_memory()
    md.set_state(h_pos, h_vel)
    md.step(desc, 3)                                   # warm (first list build of the new state)
    barrier()
    t0 = time.perf_counter()
    md.set_state(h_pos, h_vel)
    md.step(desc, args.steps)
    md.get_state(o_pos, o_vel, None)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    barrier()

    (e2e_ms,) = replica_max_times([e2e_s * 1e3], world, "cuda")
    rep_ms = replica_max_times(rep_ms, world, "cuda")                      # per repetition: the slowest rank
    mi = sorted(range(len(rep_ms)), key=lambda i: rep_ms[i])[len(rep_ms) // 2]
    ms_max, (_, st0, st1) = rep_ms[mi], reps[mi]

    if rank == 0:
        steps = st1["steps"] - st0["steps"]
        rebuilds = st1["rebuilds"] - st0["rebuilds"]
        k = steps / max(1, rebuilds)
        nbar = st1["mean_neighbors"]
        b_min, b_force = algorithmic_bytes(w.kind, nbar, k)
        peak, peak_src = measured_hbm_peak()
        value = aggregate_value(w.N, args.steps, world, ms_max)
        fk = "lj" if w.kind == "lj" else "dpd"
        if args.order != "morton":
            kernel = "k_forces_" + fk
        elif fk == "dpd":
            kernel = "k_tile_dpd2"
        elif precision == B.MD_MIXED:
            kernel = "k_tile_lj3"
        else:
            kernel = "k_tile_lj3d"
        f_ms = st1["stage_ms"][fk] / max(1, st1["stage_launches"][fk])
        achieved = w.N * b_force / (f_ms * 1e-3) / 1e9 if f_ms > 0 else 0.0
        stage_share = {n: round(v / ms_share, 4) for n, v in st_share["stage_ms"].items() if v > 0}
        traffic, traffic_note = ncu_traffic(w.name, kernel)
        ops = algorithmic_ops(w.kind, nbar, w.rc, w.rc + w.r_buff)
        fp_pipe = "fp32_fma" if precision == B.MD_MIXED else "fp64_fma"
        t_min = ops["fp"] / peaks[fp_pipe] + ops["int"] / peaks["int32_mad"]          # ns per particle at the pipe peaks
        alu_ach = w.N * (ops["fp"] + ops["int"]) / (f_ms * 1e-3) / 1e9 if f_ms > 0 else 0.0
        alu_peak = (ops["fp"] + ops["int"]) / t_min
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": ms_max / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32" if precision == B.MD_MIXED else "f64",
            "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "precision": w.precision, "rc": w.rc, "r_buff": w.r_buff,
                       "dt": w.dt, "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2": "inputs larger than L2 (neighbour list %.0f MB of 16-bit entries + %.0f MB of state per step)"
                             % (2e-6 * st1["nlist_entries"], 216e-6 * w.N),
                       "tps": world * args.steps / (ms_max * 1e-3) / world, "rebuild_period_k": k,
                       "mean_neighbors": nbar, "rebuilds": rebuilds, "dangerous_builds": st1["dangerous_builds"],
                       "order": args.order, "sched": args.sched,
                       "speculative_forces": st1["speculative_forces"] - st0["speculative_forces"],
                       "wasted_forces": st1["wasted_forces"] - st0["wasted_forces"],
                       "launch": {n: [v["block"], v["w"]] for n, v in st1["launch"].items()},
                       "reps_ms_per_step": [r / args.steps for r in rep_ms], "reported": "median of %d repetitions" % len(rep_ms),
                       "best_ms_per_step": min(rep_ms) / args.steps,
                       "device_memory": "own cudaMalloc" if args.own_alloc else "torch tensor (md_workspace_bytes, md_set_workspace)",
                       "stage_share_of_step": stage_share,
                       "stage_share_from": "%d further steps with every stage bracketed by CUDA events" % n_share,
                       "step_bmin_bytes_per_particle": b_min,
                       "step_roofline_frac": (w.N * b_min * args.steps / (ms_max * 1e-3)) / (peak * 1e9)},
            "e2e": {"value": world * w.N * args.steps / (e2e_ms * 1e-3), "unit": UNIT,
                    "h2d_bytes_per_step": int(2 * w.pos.nbytes / args.steps),
                    "d2h_bytes_per_step": int(2 * w.pos.nbytes / args.steps)},
            "gpu_launches": int(st1["launches"] - st0["launches"]),
            "clocks": clocks,
            "roofline": {"bound": "hbm", "kernel": kernel, "achieved": achieved, "peak": peak,
                         "peak_source": peak_src, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic, "traffic_note": traffic_note,
                         # achieved/frac use the ALGORITHMIC bytes of SURVEY 8(d) (4-byte indices: 4 n + 56, DPD 4 n + 84 per
                         # particle); the list is stored as 16-bit entries, so the measured DRAM traffic is lower:
                         "kernel_timing": "CUDA events on the library's stream around every %s pair-force launch of the timed region (%d launches)"
                                          % ("one" if ev_stride == 1 else "%dth" % ev_stride, st1["stage_launches"][fk]),
                         "bytes_model": "SURVEY 8(d) staged minimum of the pair-force kernel, 4-byte indices",
                         "traffic_gbs": (traffic / (f_ms * 1e-3) / 1e9) if (traffic and f_ms > 0) else None,
                         "traffic_frac": (traffic / (f_ms * 1e-3) / 1e9 / peak) if (traffic and f_ms > 0) else None,
                         "bytes_per_particle": b_force, "launch_ms": f_ms},
            # second roofline: the same kernel's ALGORITHMIC instruction rate against the measured issue
            # rate of the pipe(s) it runs on (md_debug_peak, giga lane-instructions per second, an FMA counts once)
            "roofline_alu": {"pipe": fp_pipe + ("+int32_mad" if ops["int"] else ""), "kernel": kernel,
                             "achieved": alu_ach, "peak": alu_peak, "unit": "G lane-instr/s",
                             "frac": alu_ach / alu_peak if alu_peak else None,
                             "instr_per_particle": ops, "measured_pipe_peaks": peaks},
        }
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(w)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=100)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--order", default="morton", choices=["lex", "morton", "hilbert"])
    ap.add_argument("--no-tune", action="store_true")
    ap.add_argument("--sched", default="batch", choices=["sync", "speculative", "batch"],
                    help="md_step scheduler (MD_SCHED_*): batch = kernels of several steps enqueued ahead, gated on the device")
    ap.add_argument("--launch", nargs="*", default=[], help="kernel=block,w (with --no-tune)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--r-buff", type=float, default=None, dest="r_buff",
                    help="override the configured skin r_buff = 0.4 (tuning sweep; not a reported configuration)")
    ap.add_argument("--dihedrals", action="store_true", help="config 4 with periodic dihedrals and stiff harmonic angles (k = 50) along the chains (SURVEY 8(f) row 3)")
    ap.add_argument("--angles", action="store_true", help="config 4 with harmonic angles along the chains (SURVEY 8(f) row 3)")
    ap.add_argument("--auto-rbuff", action="store_true", dest="auto_rbuff",
                    help="md_tune_rbuff: let the library choose the skin (tuning run; not a reported configuration)")
    ap.add_argument("--mtk", action="store_true", help="NVT with the Martyna-Tobias-Klein update (SURVEY 8(f) row 1, R39)")
    ap.add_argument("--nvt", action="store_true",
                    help="Nose-Hoover NVT (MD_F_NVT, kT = the workload's temperature, tau = 0.5) instead of NVE: "
                         "SURVEY 8(f) row 1; named in the workload, not a BASELINE configuration")
    ap.add_argument("--reps", type=int, default=3, help="timed repetitions of --steps steps; the median is reported")
    ap.add_argument("--own-alloc", action="store_true", help="let the library cudaMalloc instead of a torch workspace")
    ap.add_argument("--brick", type=int, default=0, help="MD_OPT_TILE_BRICK: 1, 2 or 4 cells per brick edge (0 = auto)")
    args = ap.parse_args()
    if args.impl == "reference":
        sys.exit(run_reference(args))
    sys.exit(run_ours(args))


if __name__ == "__main__":
    main()
