"""Pins of the oracle's Martyna-Tobias-Klein NVT step (R39) -- no GPU.

The paper names the update and prints no equation, so the pins are what the mathematics fixes: the NVE
limit, exact time reversibility of the symmetric factorisation, the closed (K, xi, eta) ODE of a force-free gas solved
by an independent adaptive integrator (second order), the conserved extended energy (second order, no drift), the
temperature it settles at, and that it is NOT the R30 discretisation while converging to the same trajectory.
"""
import numpy as np
from scipy.integrate import solve_ivp

import oracle
from paper_1412_3387_b200 import inputs


def _sim(dt_unused=None, kT0=1.0, tau=0.5, T_start=0.6, scheme="mtk", n=4):
    w = inputs.lj_fcc(n, rc=2.5, r_buff=0.4, kT=T_start, jitter=0.05, pos_seed=3, vel_seed=4)   # N = 4 n^3
    nvt = dict(kT=kT0, tau=tau)
    if scheme:
        nvt["scheme"] = scheme
    return w, oracle.Sim(w.pos, w.vel, w.box, w.rc, w.r_buff, {"lj": w.params}, nvt=nvt)


def test_mtk_reduces_to_nve_when_the_thermostat_is_off():
    w, a = _sim(tau=1e150)
    b = oracle.Sim(w.pos, w.vel, w.box, w.rc, w.r_buff, {"lj": w.params})
    a.run(20, 0.005); b.run(20, 0.005)
    assert np.abs(a.pos - b.pos).max() < 1e-14 and np.abs(a.vel - b.vel).max() < 1e-14
    assert abs(a.xi) < 1e-290 and abs(a.eta) < 1e-290


def test_mtk_step_is_time_reversible():
    """Forward n steps, negate velocities and xi, forward n steps: back at the start (a symmetric composition of exact
    flows).  Rounding only: 1e-11 after 2 x 60 steps; the thermostat is strongly active (xi reaches 0.5)."""
    w, s = _sim(kT0=1.5, tau=0.3)
    x0, v0 = s.pos.copy(), s.vel.copy()
    s.run(60, 0.004)
    assert abs(s.xi) > 0.3 and np.abs(s.pos - x0).max() > 0.05
    eta_mid = s.eta
    s.vel *= -1.0
    s.xi = -s.xi
    s.run(60, 0.004)
    d = s.pos - x0
    d -= w.box * np.round(d / w.box)
    assert np.abs(d).max() < 1e-11
    assert np.abs(s.vel + v0).max() < 1e-11 and abs(s.xi) < 1e-12
    assert abs(eta_mid) > 1e-3 and abs(s.eta) < 1e-12                   # eta runs back to 0 as well


def _free_gas(dt, n_steps, N=200, kT=1.0, tau=0.5, T_start=2.0):
    rng = np.random.default_rng(5)
    vel = rng.normal(size=(N, 3)) * np.sqrt(T_start)
    vel -= vel.mean(axis=0)
    xi = eta = 0.0
    K0 = 0.5 * np.sum(vel * vel)
    for _ in range(n_steps):           # no forces: kick and drift leave the velocities alone
        xi, eta = oracle.mtk_thermostat_half(vel, dt, kT, tau, xi, eta)
        xi, eta = oracle.mtk_thermostat_half(vel, dt, kT, tau, xi, eta)
    return K0, 0.5 * np.sum(vel * vel), xi, eta


def test_mtk_free_gas_follows_the_nose_hoover_ode_at_second_order():
    N, kT, tau, t_end = 200, 1.0, 0.5, 1.0
    g = 3 * N - 3
    K0, K1, xi1, eta1 = _free_gas(0.01, 100, N, kT, tau)
    _, K2, xi2, eta2 = _free_gas(0.005, 200, N, kT, tau)
    ref = solve_ivp(lambda t, y: [-2.0 * y[1] * y[0], (2.0 * y[0] / (g * kT) - 1.0) / tau ** 2, y[1]], (0.0, t_end),
                    [K0, 0.0, 0.0], rtol=1e-12, atol=1e-12, method="DOP853")
    Kr, xir, etar = ref.y[:, -1]
    e1 = np.array([abs(K1 - Kr) / Kr, abs(xi1 - xir), abs(eta1 - etar)])
    e2 = np.array([abs(K2 - Kr) / Kr, abs(xi2 - xir), abs(eta2 - etar)])
    assert np.all(e1 < 2e-4)
    assert np.all(e1 / e2 > 3.5) and np.all(e1 / e2 < 4.5)
    assert abs(xir) > 0.3 and Kr < 0.9 * K0
    # every velocity is scaled by the same factor: directions untouched (checked through the momentum-free start)
    assert abs(K1 / K0 - K2 / K0) < 1e-3


def test_mtk_extended_energy_and_temperature():
    w, s1 = _sim()
    s1.compute_forces(0.004, 0)
    h1, T1 = [s1.nvt_conserved()], []
    for _ in range(2500):
        s1.run(1, 0.004)
        h1.append(s1.nvt_conserved())
        T1.append(2.0 * s1.kinetic_energy() / (3 * s1.N - 3))
    h1, T1 = np.array(h1), np.array(T1)
    w, s2 = _sim()
    s2.compute_forces(0.002, 0)
    h2 = [s2.nvt_conserved()]
    for _ in range(1000):
        s2.run(1, 0.002)
        h2.append(s2.nvt_conserved())
    h2 = np.array(h2)
    d1 = np.abs(h1[:501] - h1[0]).max() / s1.N
    d2 = np.abs(h2 - h2[0]).max() / s1.N
    assert d1 < 1e-2 and 3.0 < d1 / d2 < 5.5                   # second order over the same 2 time units
    assert np.abs(h1 - h1[0]).max() / s1.N < 2e-2              # no secular drift over 10 time units
    assert T1[:20].mean() < 0.7 and abs(T1[1000:].mean() - 1.0) < 0.05


def test_mtk_and_the_r30_scheme_differ_at_second_order_only():
    """Two discretisations of the same equations of motion: after 0.4 time units they agree to O(dt^2) (the difference
    falls 4x when dt is halved) and are not the same numbers."""
    diffs = []
    for dt, n in ((0.004, 100), (0.002, 200)):
        _, a = _sim(scheme="mtk")
        _, b = _sim(scheme=None)
        a.run(n, dt); b.run(n, dt)
        diffs.append(max(np.abs(a.vel - b.vel).max(), abs(a.xi - b.xi)))
    assert 1e-7 < diffs[1] < diffs[0] < 1e-3
    assert 3.0 < diffs[0] / diffs[1] < 5.5
