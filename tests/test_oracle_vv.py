"""Pins for the oracle's velocity-Verlet (O7) and the driver loop."""
import numpy as np

import oracle
from paper_1412_3387_b200 import inputs


def test_free_flight_with_wraps_and_images():
    box = np.array([5.0, 6.0, 7.0])
    pos0 = inputs.random_box(20, box, 1)
    vel = np.random.default_rng(2).uniform(-30, 30, size=(20, 3))      # fast: many wraps
    sim = oracle.Sim(pos0, vel, box, 1.0, 0.4, {})                     # no forces
    dt, n = 0.01, 200
    sim.run(n, dt)
    unwrapped = sim.pos + sim.image * box
    assert np.abs(unwrapped - (pos0 + n * dt * vel)).max() < 1e-11
    assert np.all(sim.pos >= -0.5 * box) and np.all(sim.pos < 0.5 * box)
    assert np.array_equal(sim.vel, vel)
    assert np.abs(sim.image).max() >= 5


def test_harmonic_dimer_discrete_frequency():
    """Two unit masses on a harmonic bond: the relative coordinate s = r - r0 obeys s_n = s_0 cos(n th),
    cos th = 1 - (w dt)^2/2 with w^2 = 2k/m (exact solution of the velocity-Verlet recursion)."""
    k, r0, dt, s0 = 330.0, 0.84, 0.005, 0.1
    box = np.array([9.0, 9.0, 9.0])
    pos = np.array([[0.5 * (r0 + s0), 0, 0], [-0.5 * (r0 + s0), 0, 0]])
    sim = oracle.Sim(pos, np.zeros((2, 3)), box, 1.0, 0.4, {"bonds": dict(k=k, r0=r0)}, bonds=np.array([[0, 1]]))
    th = np.arccos(1 - 2 * k * dt * dt / 2)
    for n in range(1, 301):
        sim.run(1, dt)
        s = (sim.pos[0, 0] - sim.pos[1, 0]) - r0
        assert abs(s - s0 * np.cos(n * th)) < 1e-11
    assert np.abs(sim.pos[:, 1:]).max() == 0.0


def test_mass_enters_as_F_over_m():
    k, r0, dt = 100.0, 1.0, 0.002
    box = np.array([9.0, 9.0, 9.0])
    pos = np.array([[0.6, 0, 0], [-0.6, 0, 0]])
    sim = oracle.Sim(pos, np.zeros((2, 3)), box, 1.0, 0.4, {"bonds": dict(k=k, r0=r0)}, bonds=np.array([[0, 1]]),
                     mass=np.array([1.0, 3.0]))
    sim.run(50, dt)
    # centre of mass stays put; light particle moved 3x as far
    assert abs(1.0 * sim.pos[0, 0] + 3.0 * sim.pos[1, 0] - (0.6 - 1.8)) < 1e-12
    assert abs((sim.pos[0, 0] - 0.6) + 3.0 * (sim.pos[1, 0] + 0.6)) < 1e-12


def _lj_small(n=4, kT=1.0, scale=1.0):
    w = inputs.lj_fcc(n, rc=2.5, r_buff=0.4, kT=kT, vel_seed=5)
    return w


def test_time_reversal_lj():
    w = _lj_small(5)                                                    # N=500, L=8.4 (>= 2 rc)
    sim = oracle.Sim(w.pos, w.vel, w.box, 2.5, 0.4, {"lj": {}})
    p0 = sim.pos.copy()
    sim.run(60, 0.005)
    assert np.abs(sim.pos - p0).max() > 0.05
    sim.vel *= -1.0
    sim.run(60, 0.005)
    d = sim.pos - p0
    d -= w.box * np.rint(d / w.box)
    assert np.abs(d).max() < 1e-9


def test_energy_error_second_order_in_dt():
    """Smooth potential (harmonic bonds + conservative DPD, gamma = 0): the energy fluctuation of velocity-Verlet
    scales as dt^2.  The DPD potential energy is computed HERE from its closed form, not by the oracle."""
    w = inputs.polymer_melt(12, chain_len=16, rho=192 / 4.4 ** 3, start_seed=3, walk_seed=4, vel_seed=5)   # N=192, L=4.4
    box, pos = w.box, w.pos
    A, k, r0 = 25.0, 330.0, 0.84

    def soft_energy(p):
        U = 0.0
        for i in range(p.shape[0] - 1):
            d = p[i] - p[i + 1:]
            d -= box * np.rint(d / box)
            r = np.sqrt((d * d).sum(1))
            U += (0.5 * A * (1 - r[r < 1.0]) ** 2).sum()
        return U

    def max_dev(dt, T=0.2):
        sim = oracle.Sim(pos, w.vel, box, 1.0, 0.4,
                         {"dpd": dict(A=A, gamma=0.0, kT=1.0, seed=1), "bonds": dict(k=k, r0=r0)}, bonds=w.bonds)
        sim.compute_forces(dt, 0)
        e0 = sim.kinetic_energy() + sim.potential_energy() + soft_energy(sim.pos)
        dev = 0.0
        for _ in range(int(round(T / dt))):
            sim.run(1, dt)
            e = sim.kinetic_energy() + sim.potential_energy() + soft_energy(sim.pos)
            dev = max(dev, abs(e - e0))
        return dev

    d1, d2 = max_dev(0.004), max_dev(0.002)
    assert 3.0 < d1 / d2 < 5.5


def test_nve_energy_drift_bounded_1000_steps():
    """north_star: 'NVE energy drift bounded over 1000 steps' (R23: |E(t)-E(0)|/N <= 2e-3 eps)."""
    w = inputs.lj_fcc(6, rc=2.5, r_buff=0.4, kT=1.0, vel_seed=1)        # N=864, L=10.08: config 1's recipe, 6^3 cells
    sim = oracle.Sim(w.pos, w.vel, w.box, 2.5, 0.4, {"lj": dict(epsilon=1.0, sigma=1.0, energy_shift=1)})
    sim.compute_forces(0.005, 0)
    e0 = sim.kinetic_energy() + sim.potential_energy()
    worst = 0.0
    for _ in range(10):
        sim.run(100, 0.005)
        worst = max(worst, abs(sim.kinetic_energy() + sim.potential_energy() - e0) / w.N)
    assert worst < 2e-3
    # the lattice melts: kinetic temperature falls well below its start value 1.0 (equipartition with the potential)
    T = 2 * sim.kinetic_energy() / (3 * w.N - 3)
    assert 0.3 < T < 0.9
    assert 3 <= len(sim.rebuild_steps) <= 200                           # rebuilds happen, not every step


def test_rebuild_log_matches_trigger_definition():
    w = inputs.lj_fcc(4, rc=2.0, r_buff=0.4, kT=1.5, vel_seed=3)
    box = w.box * 1.1
    sim = oracle.Sim(w.pos * 1.1, w.vel, box, 2.0, 0.4, {"lj": {}})
    ref = sim.pos.copy()
    steps = []
    for s in range(1, 41):
        sim.run(1, 0.005)
        d = sim.pos - ref
        d -= box * np.rint(d / box)
        if ((d * d).sum(1) > 0.04).any():
            steps.append(s)
            ref = sim.pos.copy()
    assert steps == sim.rebuild_steps and len(steps) >= 1
