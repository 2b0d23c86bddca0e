"""Pins for the oracle's DPD pair force (O5) and harmonic bonds (O6)."""
import numpy as np

import oracle
from paper_1412_3387_b200 import inputs

BOX = np.array([9.0, 9.0, 9.0])


def _pair(r, direction=(1.0, 2.0, -0.5)):
    u = np.array(direction) / np.linalg.norm(direction)
    pos = np.zeros((2, 3))
    pos[0] = 0.5 * r * u
    pos[1] = -0.5 * r * u
    return pos, u


def test_conservative_term_is_gradient_of_soft_potential():
    # gamma = 0 -> sigma_R = 0: F = A (1 - r/rc) rhat = -d/dr [A rc (1-r/rc)^2 / 2]
    A, rc = 25.0, 1.0
    for r in (0.1, 0.5, 0.93):
        pos, u = _pair(r)
        F = oracle.forces_dpd(pos, np.zeros((2, 3)), BOX, rc, A, 0.0, 1.0, 0.02, 3, 42)
        assert np.abs(F[0] - A * (1 - r / rc) * u).max() < 1e-13
        assert np.abs(F[0] + F[1]).max() == 0.0
        U = lambda x: 0.5 * A * rc * (1 - x / rc) ** 2
        h = 1e-6
        assert abs(np.dot(F[0], u) + (U(r + h) - U(r - h)) / (2 * h)) < 1e-7
    pos, u = _pair(1.0)                      # r == rc: outside (strict <)
    assert np.abs(oracle.forces_dpd(pos, np.zeros((2, 3)), BOX, rc, A, 0.0, 1.0, 0.02, 3, 42)).max() == 0.0
    pos = np.zeros((2, 3))                   # r == 0: no direction -> no force
    assert np.abs(oracle.forces_dpd(pos, np.zeros((2, 3)), BOX, rc, A, 4.5, 1.0, 0.02, 3, 42)).max() == 0.0


def test_dissipative_term_closed_form_and_one_step_decay():
    # A = 0, kT = 0: F_a = -gamma w^2 (rhat . v_ab) rhat ; only the radial relative velocity is damped
    gamma, rc, r = 4.5, 1.0, 0.6
    pos, u = _pair(r)
    vel = np.array([[0.3, -0.2, 0.9], [-0.1, 0.4, 0.2]])
    F = oracle.forces_dpd(pos, vel, BOX, rc, 0.0, gamma, 0.0, 0.02, 1, 42)
    w = 1 - r / rc
    vr = np.dot(u, vel[0] - vel[1])
    assert np.abs(F[0] - (-gamma * w * w * vr) * u).max() < 1e-14
    assert np.abs(F[0] + F[1]).max() == 0.0
    # one explicit Euler step of length dt: radial relative velocity decays by the factor (1 - 2 gamma w^2 dt / m)
    dt = 1e-3
    v_new = vel + dt * F
    vr_new = np.dot(u, v_new[0] - v_new[1])
    assert abs(vr_new - vr * (1 - 2 * gamma * w * w * dt)) < 1e-15
    # tangential part untouched
    t_old = (vel[0] - vel[1]) - vr * u
    t_new = (v_new[0] - v_new[1]) - vr_new * u
    assert np.abs(t_old - t_new).max() < 1e-15


def test_random_term_amplitude_and_pair_keying():
    # A = 0, v = 0: F_a = sqrt(2 gamma kT) w theta_ab / sqrt(dt) rhat with theta from (min tag, max tag, step, seed)
    gamma, kT, dt, rc, r = 4.5, 1.3, 0.02, 1.0, 0.4
    pos, u = _pair(r)
    F = oracle.forces_dpd(pos, np.zeros((2, 3)), BOX, rc, 0.0, gamma, kT, dt, 9, 42)
    th = oracle.dpd_theta(0, 1, 9, 42)
    assert np.abs(F[0] - np.sqrt(2 * gamma * kT) * (1 - r / rc) * th / np.sqrt(dt) * u).max() < 1e-13
    assert np.abs(F[0] + F[1]).max() == 0.0
    F2 = oracle.forces_dpd(pos, np.zeros((2, 3)), BOX, rc, 0.0, gamma, kT, dt, 10, 42)
    assert np.abs(F2 - F).max() > 0      # new step, new number
    # the pair's number depends on the TAGS, not on the positions or on which of the two is "a":
    F3 = oracle.forces_dpd(pos[::-1].copy(), np.zeros((2, 3)), BOX, rc, 0.0, gamma, kT, dt, 9, 42)
    assert np.abs(F3[0] - F[1]).max() < 1e-15


def test_dpd_newton_third_law_and_probe_rows():
    w = inputs.dpd_fluid(600, pos_seed=1, vel_seed=2)       # L = 5.85 >= 3*1.4
    p = w.params
    F = oracle.forces_dpd(w.pos, w.vel, w.box, w.rc, p["A"], p["gamma"], p["kT"], w.dt, 17, p["seed"])
    assert np.abs(F.sum(axis=0)).max() < 1e-12 * np.abs(F).sum()
    pr = inputs.probe_tags(w.N, 50, seed=4)
    Fp = oracle.probe_forces_dpd(w.pos, w.vel, w.box, w.rc, p["A"], p["gamma"], p["kT"], w.dt, 17, p["seed"], pr)
    assert np.abs(Fp - F[pr]).max() < 1e-11 * np.abs(F).max()


def test_random_force_variance_fluctuation_dissipation():
    """<F_R^2> over many pairs at fixed w equals 2 gamma kT w^2 / dt (theta has unit variance)."""
    gamma, kT, dt, rc, r = 4.5, 1.0, 0.02, 1.0, 0.5
    pos, u = _pair(r)
    vals = []
    for step in range(4000):
        F = oracle.forces_dpd(pos, np.zeros((2, 3)), BOX, rc, 0.0, gamma, kT, dt, step, 42)
        vals.append(np.dot(F[0], u))
    vals = np.array(vals)
    expect = 2 * gamma * kT * (1 - r / rc) ** 2 / dt
    assert abs(vals.var() / expect - 1.0) < 0.06
    assert abs(vals.mean()) < 4 * np.sqrt(expect / len(vals))


def test_harmonic_bond_two_body_and_gradient():
    k, r0 = 330.0, 0.84
    for r in (0.5, 0.84, 1.3):
        pos, u = _pair(r)
        F, E = oracle.forces_bonds(pos, BOX, np.array([[0, 1]]), k, r0)
        assert np.abs(F[0] - (-k * (r - r0)) * u).max() < 1e-11
        assert np.abs(F[0] + F[1]).max() == 0.0
        assert abs(E.sum() - 0.5 * k * (r - r0) ** 2) < 1e-12 and E[0] == E[1]
    # through the periodic boundary, and accumulate semantics
    pos = np.array([[4.3, 0, 0], [-4.2, 0, 0]])              # distance 0.5 through the wrap, a is "left" of b
    F = np.ones((2, 3)); E = np.ones(2)
    oracle.forces_bonds(pos, BOX, np.array([[0, 1]]), k, r0, F, E)
    assert abs(F[0, 0] - 1.0 - (+k * (0.5 - r0))) < 1e-10    # compressed bond pushes 0 to -x (d = -0.5)
    assert abs(E.sum() - 2.0 - 0.5 * k * (0.5 - r0) ** 2) < 1e-12
    # coincident particles: zero force
    F, E = oracle.forces_bonds(np.zeros((2, 3)), BOX, np.array([[0, 1]]), k, r0)
    assert np.abs(F).max() == 0.0


def test_bonds_chain_gradient_and_newton():
    w = inputs.polymer_melt(6, chain_len=16, rho=96 / 512.0, start_seed=1, walk_seed=2)     # N=96, L=8
    box, pos = w.box, w.pos
    F, E = oracle.forces_bonds(pos, box, w.bonds, 330.0, 0.84)
    assert np.abs(F.sum(axis=0)).max() < 1e-10
    h = 1e-6
    for i, a in ((0, 0), (5, 1), (15, 2), (40, 0), (95, 1)):
        p = pos.copy(); p[i, a] += h
        m = pos.copy(); m[i, a] -= h
        Up = oracle.forces_bonds(p, box, w.bonds, 330.0, 0.84)[1].sum()
        Um = oracle.forces_bonds(m, box, w.bonds, 330.0, 0.84)[1].sum()
        assert abs(-(Up - Um) / (2 * h) - F[i, a]) < 1e-5 * max(1.0, abs(F[i, a]))
    # every bond of the recipe has length 0.97 (random-walk step) -> energy per bond k/2 (0.97-0.84)^2
    assert abs(E.sum() / len(w.bonds) - 0.5 * 330.0 * 0.13 ** 2) < 1e-9
