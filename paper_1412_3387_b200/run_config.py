"""Run one of the five BASELINE.json configurations for its configured number of steps and print the thermodynamics.

    python -m paper_1412_3387_b200.run_config --config 2 [--steps N] [--nvt]

A user-facing driver of the C ABI (through the ctypes binding): upload the seeded synthetic state, tune, md_step, and
md_thermo and md_pressure before and after.  Device memory comes from a torch tensor (md_set_workspace).  Needs a CUDA
device (no CPU fallback).
"""
import argparse
import time

import numpy as np

from . import binding as B
from . import inputs


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--steps", type=int, default=0, help="0 = the configuration's own length")
    ap.add_argument("--scale", type=float, default=1.0)
    ap.add_argument("--nvt", action="store_true", help="Nose-Hoover at the configuration's kT, tau = 0.5")
    a = ap.parse_args()
    w = inputs.config(a.config, scale=a.scale)
    n = a.steps or w.n_steps
    md = B.from_workload(w, workspace="torch")
    nvt = dict(kT=float(w.params.get("kT", 1.0)), tau=0.5) if a.nvt else None
    desc = B.step_desc(w.kind, w.dt, w.params, nvt=nvt)
    md.tune(desc)
    md.step(desc, 1)
    t0 = md.thermo()
    t = time.perf_counter()
    md.step(desc, n - 1)
    t1 = md.thermo()
    wall = time.perf_counter() - t
    p1 = md.pressure(desc)
    st = md.stats()
    e0 = (t0["kinetic"] + t0["potential"]) / w.N
    e1 = (t1["kinetic"] + t1["potential"]) / w.N
    print(f"{w.name}: N={w.N} steps={n} wall={wall:.2f}s ms/step={1e3 * wall / max(1, n - 1):.4f} "
          f"rebuilds={st['rebuilds']} dangerous={st['dangerous_builds']} T: {t0['temperature']:.4f} -> "
          f"{t1['temperature']:.4f}  (K+U)/N: {e0:.6f} -> {e1:.6f}  max|p|={np.abs(t1['momentum']).max():.2e}  "
          f"P={p1['pressure']:.4f}  r_buff={st['r_buff']}  sched=batch")


if __name__ == "__main__":
    main()
