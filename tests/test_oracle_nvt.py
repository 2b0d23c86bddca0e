"""Pins of the oracle's Nose-Hoover NVT step (R30) -- no GPU.

The paper names the thermostat and prints no equation, so the pins are what the mathematics fixes:
the NVE limit, the closed two-variable ODE of a force-free gas (integrated independently with a high-order adaptive
method), second-order convergence, the conserved extended energy, and the temperature the thermostat settles at.
"""
import numpy as np
from scipy.integrate import solve_ivp

import oracle
from paper_1412_3387_b200 import inputs


def test_nvt_reduces_to_nve_when_the_thermostat_is_off():
    w = inputs.lj_fcc(4, rc=2.5, r_buff=0.4, kT=1.0, jitter=0.05, pos_seed=1, vel_seed=2)      # N = 256
    F, _ = oracle.forces_lj(w.pos, w.box, w.rc)
    pa, va, ia = w.pos.copy(), w.vel.copy(), np.zeros((w.N, 3), np.int32)
    pb, vb, ib = w.pos.copy(), w.vel.copy(), np.zeros((w.N, 3), np.int32)
    oracle.vv_half1(pa, va, ia, F, w.box, 0.005)
    oracle.nvt_half1(pb, vb, ib, F, w.box, 0.005, 0.0)
    assert np.abs(pa - pb).max() < 1e-15 and np.abs(va - vb).max() < 1e-15 and np.array_equal(ia, ib)
    oracle.vv_half2(va, F, 0.005)
    oracle.nvt_half2(vb, F, 0.005, 0.0)
    assert np.abs(va - vb).max() < 1e-15
    xi, eta, K = oracle.nvt_thermostat(vb, 0.005, 1.0, 1e150, 0.0, 0.0)
    assert abs(xi) < 1e-290 and abs(eta) < 1e-290 and abs(K - 0.5 * np.sum(vb * vb)) < 1e-12


def _free_gas(dt, n_steps, N=200, kT=1.0, tau=0.5, T_start=2.0):
    rng = np.random.default_rng(5)
    vel = rng.normal(size=(N, 3)) * np.sqrt(T_start)
    vel -= vel.mean(axis=0)
    pos = np.zeros((N, 3))
    img = np.zeros((N, 3), np.int32)
    F = np.zeros((N, 3))
    box = np.array([1e9, 1e9, 1e9])
    xi = eta = 0.0
    K0 = 0.5 * np.sum(vel * vel)
    for _ in range(n_steps):
        oracle.nvt_half1(pos, vel, img, F, box, dt, xi)
        xi, eta, _ = oracle.nvt_thermostat(vel, dt, kT, tau, xi, eta)
        oracle.nvt_half2(vel, F, dt, xi)
    return K0, 0.5 * np.sum(vel * vel), xi, eta


def test_free_gas_follows_the_nose_hoover_ode_at_second_order():
    """Without forces every velocity is scaled by the same factor, and (K, xi) obey dK/dt = -2 xi K,
    dxi/dt = (2K/(g kT) - 1)/tau^2: a closed ODE that an independent adaptive integrator solves to 1e-11."""
    N, kT, tau, t_end = 200, 1.0, 0.5, 1.0
    g = 3 * N - 3
    K0, K1, xi1, eta1 = _free_gas(0.01, 100, N, kT, tau)
    _, K2, xi2, eta2 = _free_gas(0.005, 200, N, kT, tau)
    ref = solve_ivp(lambda t, y: [-2.0 * y[1] * y[0], (2.0 * y[0] / (g * kT) - 1.0) / tau ** 2, y[1]], (0.0, t_end),
                    [K0, 0.0, 0.0], rtol=1e-12, atol=1e-12, method="DOP853")
    Kr, xir, etar = ref.y[:, -1]
    e1 = np.array([abs(K1 - Kr) / Kr, abs(xi1 - xir), abs(eta1 - etar)])
    e2 = np.array([abs(K2 - Kr) / Kr, abs(xi2 - xir), abs(eta2 - etar)])
    assert np.all(e1 < 2e-3)                       # the scheme follows the ODE ...
    assert np.all(e1 / e2 > 3.0) and np.all(e1 / e2 < 5.5)   # ... with an error that falls 4x when dt is halved
    assert abs(xir) > 0.3 and Kr < 0.9 * K0        # and the case is not trivial: the gas was cooled substantially


def _lj_nvt(dt, n_steps, kT0, T_start=0.6, tau=0.5):
    w = inputs.lj_fcc(4, rc=2.5, r_buff=0.4, kT=T_start, jitter=0.05, pos_seed=3, vel_seed=4)  # N = 256
    sim = oracle.Sim(w.pos, w.vel, w.box, w.rc, w.r_buff, {"lj": w.params}, nvt=dict(kT=kT0, tau=tau))
    sim.compute_forces(dt, 0)
    h, T = [sim.nvt_conserved()], []
    for _ in range(n_steps):
        sim.run(1, dt)
        h.append(sim.nvt_conserved())
        T.append(2.0 * sim.kinetic_energy() / (3 * sim.N - 3))
    return np.array(h), np.array(T), sim.N


def test_lj_extended_energy_is_conserved_and_temperature_settles():
    h1, T1, N = _lj_nvt(0.004, 2500, kT0=1.0)
    h2, _, _ = _lj_nvt(0.002, 1000, kT0=1.0)
    d1 = np.abs(h1[:501] - h1[0]).max() / N
    d2 = np.abs(h2 - h2[0]).max() / N
    # K + U + g kT (tau^2 xi^2/2 + eta) over the same 2 time units: bounded (the plain-shifted LJ force jumps at rc,
    # cf. R23) and second order in dt
    assert d1 < 1e-2
    assert 3.0 < d1 / d2 < 5.5
    assert np.abs(h1 - h1[0]).max() / N < 2e-2         # and no secular drift over 10 time units
    # started at T = 0.5 after equipartition with the lattice, thermostat at 1.0: Nose-Hoover oscillates around the
    # target (0.3 ... 2.3 here); the average over the last 6 time units is within 5 %
    assert T1[:20].mean() < 0.7
    assert abs(T1[1000:].mean() - 1.0) < 0.05
