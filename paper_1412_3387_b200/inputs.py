"""Seeded synthetic workloads.

This module serves BOTH the CPU oracle tests and the CUDA path.  It holds none of the method's
arithmetic (no forces, no cells, no neighbour search, no hash): only numpy random numbers, lattices
and random walks.  Everything is tag-ordered float64, box = [-L/2, L/2)^3.

The five configurations are those of BASELINE.json:configs.  They stand in for the paper's LJ-liquid
(PAPER.md:210, :276, :300), DPD and polymer benchmarks, whose
scripts and equilibrated start configurations are in a supplement that is not available
(PAPER.md:385).  Every config takes a `scale` so that parity tests can run a small box with the same
recipe (same density, same lattice / walk construction).
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

_FCC_BASIS = np.array([[0.0, 0.0, 0.0], [0.5, 0.5, 0.0], [0.5, 0.0, 0.5], [0.0, 0.5, 0.5]])


@dataclass
class Workload:
    """One synthetic MD state plus the parameters the run uses."""
    name: str
    kind: str                 # "lj" | "dpd" | "polymer"
    N: int
    box: np.ndarray           # (3,) float64 edge lengths
    pos: np.ndarray           # (N,3) float64, wrapped into [-L/2, L/2)
    vel: np.ndarray           # (N,3) float64
    rc: float
    r_buff: float
    dt: float
    n_steps: int
    precision: str            # "fp64" | "mixed"
    params: dict = field(default_factory=dict)
    bonds: np.ndarray | None = None   # (n_bonds,2) uint32 tag pairs

    @property
    def r_list(self) -> float:
        return self.rc + self.r_buff


def wrap(pos: np.ndarray, box: np.ndarray) -> np.ndarray:
    """Fold coordinates into [-L/2, L/2) (plain periodic folding of generator output)."""
    half = 0.5 * box
    out = pos - box * np.floor((pos + half) / box)
    # guard the upper edge against rounding (x == +L/2 -> -L/2)
    out = np.where(out >= half, out - box, out)
    out = np.where(out < -half, out + box, out)
    return np.ascontiguousarray(out)


def fcc_positions(n_cells: int, L: float, chunk: int = 64) -> np.ndarray:
    """FCC lattice of n_cells^3 unit cells in a cube of edge L, origin shifted by +a/4."""
    a = L / n_cells
    N = 4 * n_cells ** 3
    pos = np.empty((N, 3), dtype=np.float64)
    jk = np.stack(np.meshgrid(np.arange(n_cells), np.arange(n_cells), indexing="ij"), -1).reshape(-1, 2)
    per_i = jk.shape[0] * 4
    for i in range(n_cells):
        cell = np.empty((jk.shape[0], 3))
        cell[:, 0] = i
        cell[:, 1:] = jk
        blk = (cell[:, None, :] + _FCC_BASIS[None, :, :]).reshape(-1, 3)
        pos[i * per_i:(i + 1) * per_i] = blk * a + (0.25 * a - 0.5 * L)
    return pos


def thermal_velocities(N: int, kT: float, seed: int, mass: float = 1.0) -> np.ndarray:
    """Gaussian velocities, zero net momentum, rescaled so sum m v^2 = (3N-3) kT exactly."""
    rng = np.random.default_rng(seed)
    v = rng.standard_normal((N, 3)) * np.sqrt(kT / mass)
    v -= v.mean(axis=0, keepdims=True)
    if N > 1:
        ke2 = mass * float(np.einsum("ij,ij->", v, v))
        v *= np.sqrt((3 * N - 3) * kT / ke2)
    return np.ascontiguousarray(v)


def lj_fcc(n_cells: int, rho: float = 0.8442, rc: float = 2.5, r_buff: float = 0.4, kT: float = 1.0,
           dt: float = 0.005, n_steps: int = 100, jitter: float = 0.0, pos_seed: int = 2, vel_seed: int = 1,
           precision: str = "fp64", name: str = "lj") -> Workload:
    N = 4 * n_cells ** 3
    L = (N / rho) ** (1.0 / 3.0)
    box = np.array([L, L, L])
    pos = fcc_positions(n_cells, L)
    if jitter > 0.0:
        rng = np.random.default_rng(pos_seed)
        pos += rng.uniform(-jitter, jitter, size=pos.shape)
    pos = wrap(pos, box)
    vel = thermal_velocities(N, kT, vel_seed)
    return Workload(name=name, kind="lj", N=N, box=box, pos=pos, vel=vel, rc=rc, r_buff=r_buff, dt=dt,
                    n_steps=n_steps, precision=precision,
                    params=dict(epsilon=1.0, sigma=1.0, energy_shift=1, kT=kT, rho=rho))


def dpd_fluid(N: int, rho: float = 3.0, rc: float = 1.0, r_buff: float = 0.4, kT: float = 1.0, dt: float = 0.02,
              n_steps: int = 5000, pos_seed: int = 4, vel_seed: int = 5, name: str = "dpd") -> Workload:
    L = (N / rho) ** (1.0 / 3.0)
    box = np.array([L, L, L])
    rng = np.random.default_rng(pos_seed)
    pos = wrap(rng.uniform(-0.5 * L, 0.5 * L, size=(N, 3)), box)
    vel = thermal_velocities(N, kT, vel_seed)
    return Workload(name=name, kind="dpd", N=N, box=box, pos=pos, vel=vel, rc=rc, r_buff=r_buff, dt=dt,
                    n_steps=n_steps, precision="fp64",
                    params=dict(A=25.0, gamma=4.5, kT=kT, seed=42, rho=rho))


def polymer_melt(n_chains: int, chain_len: int = 64, rho: float = 3.0, rc: float = 1.0, r_buff: float = 0.4,
                 kT: float = 1.0, dt: float = 0.01, n_steps: int = 5000, bond_step: float = 0.97,
                 start_seed: int = 6, walk_seed: int = 7, vel_seed: int = 8, name: str = "polymer") -> Workload:
    N = n_chains * chain_len
    L = (N / rho) ** (1.0 / 3.0)
    box = np.array([L, L, L])
    rng0 = np.random.default_rng(start_seed)
    start = rng0.uniform(-0.5 * L, 0.5 * L, size=(n_chains, 3))
    rng1 = np.random.default_rng(walk_seed)
    # uniformly random directions: normalised Gaussians
    d = rng1.standard_normal((n_chains, chain_len - 1, 3))
    d /= np.linalg.norm(d, axis=2, keepdims=True)
    steps = np.concatenate([start[:, None, :], bond_step * d], axis=1)
    pos = wrap(np.cumsum(steps, axis=1).reshape(N, 3), box)
    vel = thermal_velocities(N, kT, vel_seed)
    first = (np.arange(n_chains, dtype=np.uint32)[:, None] * chain_len
             + np.arange(chain_len - 1, dtype=np.uint32)[None, :]).reshape(-1)
    bonds = np.ascontiguousarray(np.stack([first, first + 1], axis=1).astype(np.uint32))
    return Workload(name=name, kind="polymer", N=N, box=box, pos=pos, vel=vel, rc=rc, r_buff=r_buff, dt=dt,
                    n_steps=n_steps, precision="fp64",
                    params=dict(A=25.0, gamma=4.5, kT=kT, seed=42, bond_k=330.0, bond_r0=0.84, rho=rho),
                    bonds=bonds)


def config(idx: int, scale: float = 1.0) -> Workload:
    """BASELINE.json:configs[idx-1].  `scale` < 1 shrinks the particle count, keeping the recipe.

    1: LJ N=4,000 FCC 10^3, rc 2.5, fp64, 100 steps          (seeds: vel 1)
    2: LJ N=1,048,576 FCC 64^3 + jitter 0.05, rc 3.0, mixed   (seeds: jitter 2, vel 3)
    3: DPD N=1,000,000 uniform random, rho 3                  (seeds: pos 4, vel 5)
    4: polymer 20,000 x 64 random walks, rho 3                (seeds: start 6, walk 7, vel 8)
    5: LJ N=64,012,032 FCC 252^3, rc 2.5, fp64                (seeds: vel 9)
    """
    s = scale ** (1.0 / 3.0)
    if idx == 1:
        return lj_fcc(max(3, round(10 * s)), rc=2.5, kT=1.0, n_steps=100, vel_seed=1, name="cfg1-lj-4k-fp64")
    if idx == 2:
        return lj_fcc(max(4, round(64 * s)), rc=3.0, kT=1.2, n_steps=10000, jitter=0.05, pos_seed=2, vel_seed=3,
                      precision="mixed", name="cfg2-lj-1M-mixed")
    if idx == 3:
        return dpd_fluid(max(256, round(1_000_000 * scale)), name="cfg3-dpd-1M-fp64")
    if idx == 4:
        return polymer_melt(max(4, round(20_000 * scale)), name="cfg4-polymer-1.28M-fp64")
    if idx == 5:
        return lj_fcc(max(3, round(252 * s)), rc=2.5, kT=1.0, n_steps=1000, vel_seed=9, name="cfg5-lj-64M-fp64")
    raise ValueError(f"no such config {idx}")


def random_box(N: int, box, seed: int, min_sep: float = 0.0) -> np.ndarray:
    """Uniform random positions in an orthorhombic box (tiny-box parity cases)."""
    box = np.asarray(box, dtype=np.float64)
    rng = np.random.default_rng(seed)
    return wrap(rng.uniform(-0.5, 0.5, size=(N, 3)) * box, box)


def probe_tags(N: int, M: int, seed: int = 1234) -> np.ndarray:
    """M distinct seeded probe tags (sorted) for probe-row parity at scale."""
    rng = np.random.default_rng(seed)
    M = min(M, N)
    return np.sort(rng.choice(N, size=M, replace=False)).astype(np.uint32)
