"""Run one of the five BASELINE.json configurations for its configured number of steps and print the thermodynamics.

    python -m paper_1412_3387_b200.run_config --config 2 [--steps N] [--nvt | --mtk | --langevin GAMMA] [--angles] [--dihedrals]

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
    ap.add_argument("--mtk", action="store_true", help="NVT with the Martyna-Tobias-Klein update (R39), tau = 0.5")
    ap.add_argument("--langevin", type=float, default=0.0, metavar="GAMMA", help="Langevin thermostat (R36) at the configuration's kT")
    ap.add_argument("--angles", action="store_true", help="polymer melt: harmonic angles along the chains (k = 5, theta0 = 2.0)")
    ap.add_argument("--dihedrals", action="store_true", help="polymer melt: periodic dihedrals (k = 2, n = 1) and stiff angles (k = 50) along the chains")
    a = ap.parse_args()
    w = inputs.config(a.config, scale=a.scale)
    n = a.steps or w.n_steps
    md = B.from_workload(w, workspace="torch")
    kT = float(w.params.get("kT", 1.0))
    nvt = dict(kT=kT, tau=0.5) if (a.nvt or a.mtk) else None
    if a.mtk:
        nvt["scheme"] = "mtk"
    params = dict(w.params)
    if a.langevin > 0.0:
        params["langevin"] = dict(gamma=a.langevin, kT=kT, seed=2025)
    if w.kind == "polymer" and (a.angles or a.dihedrals):
        L = 64                                           # chain length of configuration 4
        first = (np.arange(w.N // L, dtype=np.uint32)[:, None] * L)
        if a.angles or a.dihedrals:
            # stiff angles with dihedrals: the dihedral force grows as 1 / sin of the bond angles, so chains that may
            # straighten throw particles across the skin in one step (dangerous builds)
            i = (first + np.arange(L - 2, dtype=np.uint32)[None, :]).reshape(-1)
            md.set_angles(np.stack([i, i + 1, i + 2], axis=1))
            params.update(angle_k=50.0 if a.dihedrals else 5.0, angle_theta0=2.0)
        if a.dihedrals:
            i = (first + np.arange(L - 3, dtype=np.uint32)[None, :]).reshape(-1)
            md.set_dihedrals(np.stack([i, i + 1, i + 2, i + 3], axis=1))
            params.update(dihedral_k=2.0, dihedral_sign=1, dihedral_n=1)
    desc = B.step_desc(w.kind, w.dt, params, nvt=nvt)
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
          f"P={p1['pressure']:.4f}  r_buff={st['r_buff']}  sched=batch"
          + (f"  thermostat xi, eta = {md.get_thermostat()[0]:.4f}, {md.get_thermostat()[1]:.4f}" if nvt else ""))


if __name__ == "__main__":
    main()
