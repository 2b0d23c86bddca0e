"""Pins of oracle/md_oracle_ext.c: virial / pressure, Yukawa / Gaussian / Morse pairs, FENE
bonds, harmonic angles -- against closed forms, numerical gradients, invariants and the routines of md_oracle.c they
must reduce to.  No GPU."""
import math

import numpy as np
import pytest

import oracle
from paper_1412_3387_b200 import inputs

BOX = np.array([12.0, 13.0, 14.0])


def _two(r, axis=(1.0, 0.0, 0.0), at=(5.5, -6.0, 6.5)):
    """Two particles a distance r apart along `axis`, straddling the periodic boundary."""
    a = np.array(at)
    b = a - r * np.array(axis) / np.linalg.norm(axis)
    return oracle.wrap(np.stack([a, b]), BOX)


# ------------------------------------------------------------------------------------------------- pair potentials
CLOSED = [  # kind, params, r, U(r), F(r) = -dU/dr  (written out by hand from the textbook forms, R31)
    ("yukawa", (2.0, 1.5), 1.2, 2.0 * math.exp(-1.8) / 1.2, 2.0 * math.exp(-1.8) * (1.5 * 1.2 + 1.0) / 1.2 ** 2),
    ("gaussian", (3.0, 0.8), 1.1, 3.0 * math.exp(-1.21 / 1.28), 3.0 * math.exp(-1.21 / 1.28) * 1.1 / 0.64),
    ("morse", (1.7, 2.0, 1.0), 1.3, 1.7 * (math.exp(-1.2) - 2.0 * math.exp(-0.6)),
     2.0 * 2.0 * 1.7 * (math.exp(-1.2) - math.exp(-0.6))),
    ("morse", (1.7, 2.0, 1.0), 1.0, -1.7, 0.0),                      # the minimum: depth D0, zero force
]


@pytest.mark.parametrize("kind,p,r,U,F", CLOSED)
def test_pair_closed_forms(kind, p, r, U, F):
    pos = _two(r, axis=(1.0, 2.0, -0.5))
    Fo, Eo = oracle.pair_forces(pos, BOX, 3.0, kind, p, energy_shift=0)
    assert abs(Eo.sum() - U) < 1e-14 * max(1.0, abs(U))
    d = pos[0] - pos[1]
    d -= BOX * np.rint(d / BOX)
    assert np.abs(Fo[0] - F * d / r).max() < 1e-13 * max(1.0, abs(F))   # along the separation, repulsive if F > 0
    assert np.abs(Fo[0] + Fo[1]).max() == 0.0                             # Newton's third law, exactly


@pytest.mark.parametrize("kind,p", [("yukawa", (2.0, 1.5)), ("gaussian", (3.0, 0.8)), ("morse", (1.7, 2.0, 1.0)),
                                     ("lj", (0.9, 1.05))])
def test_pair_force_is_minus_gradient_and_cutoff_is_strict(kind, p):
    for r in (0.95, 1.4, 2.2):
        h = 1e-6
        U = [oracle.pair_forces(_two(x), BOX, 3.0, kind, p, 0)[1].sum() for x in (r - h, r + h)]
        F = oracle.pair_forces(_two(r), BOX, 3.0, kind, p, 0)[0][0, 0]
        assert abs(F + (U[1] - U[0]) / (2 * h)) < 1e-7 * max(1.0, abs(F))
    rc = 2.0
    inside, outside = np.nextafter(rc, 0.0), rc
    assert np.abs(oracle.pair_forces(_two(inside, at=(0.5, 0.0, 0.0)), BOX, rc, kind, p, 0)[0]).max() > 0.0
    assert np.abs(oracle.pair_forces(_two(outside, at=(0.5, 0.0, 0.0)), BOX, rc, kind, p, 0)[0]).max() == 0.0
    # the shift removes U(rc): a pair just inside the cut-off has (almost) no energy left
    assert abs(oracle.pair_forces(_two(inside, at=(0.5, 0.0, 0.0)), BOX, rc, kind, p, 1)[1].sum()) < 1e-12


def test_pair_kind0_is_the_lj_routine_and_many_body_sums():
    w = inputs.lj_fcc(4, rc=2.5, r_buff=0.4, kT=1.0, jitter=0.08, pos_seed=3, vel_seed=4)
    F0, E0 = oracle.pair_forces(w.pos, w.box, 2.5, "lj", (0.9, 1.05), 1)
    F1, E1 = oracle.forces_lj(w.pos, w.box, 2.5, 0.9, 1.05, 1)
    assert np.array_equal(F0, F1) and np.array_equal(E0, E1)
    for kind, p in (("yukawa", (2.0, 1.5)), ("gaussian", (3.0, 0.8)), ("morse", (1.7, 2.0, 1.0))):
        F, E = oracle.pair_forces(w.pos, w.box, 2.5, kind, p, 1)
        assert np.abs(F.sum(axis=0)).max() < 1e-11 * np.abs(F).sum()


# ------------------------------------------------------------------------------------------------- virial, pressure
def test_virial_two_body_and_symmetry():
    pos = _two(1.2, axis=(1.0, 2.0, -0.5))
    d = pos[0] - pos[1]
    d -= BOX * np.rint(d / BOX)
    F = oracle.pair_forces(pos, BOX, 3.0, "yukawa", (2.0, 1.5), 0)[0][0]
    W = oracle.virial_pair(pos, BOX, 3.0, "yukawa", (2.0, 1.5))
    assert np.allclose(W[:3], d * F, rtol=0, atol=1e-15) and np.allclose(W[3:], [d[0] * F[1], d[0] * F[2], d[1] * F[2]], atol=1e-15)
    assert abs(W[:3].sum() - 1.2 * CLOSED[0][4]) < 1e-13                      # tr W = r F(r)
    assert abs(d[0] * F[1] - d[1] * F[0]) < 1e-15                             # central force: the tensor is symmetric


def test_ideal_gas_pressure_and_virial_theorem_by_box_rescale():
    w = inputs.lj_fcc(4, rc=2.5, r_buff=0.4, kT=1.3, jitter=0.08, pos_seed=3, vel_seed=4)     # N = 256
    V = float(np.prod(w.box))
    assert abs(oracle.pressure(w.vel, w.box, np.zeros(6)) - (w.N - 1) * 1.3 / V) < 1e-12      # P = rho kT ((3N-3) dof, R18)
    for kind, p in (("lj", (1.0, 1.0)), ("yukawa", (2.0, 1.5)), ("morse", (1.7, 2.0, 1.0))):
        # tr W = -3 V dU/dV for the UNSHIFTED, smoothly truncated energy: scale box and positions by (1 +- h); pairs
        # must not cross the cut-off during the rescale, so the cut-off scales along (rc is a length of the system here)
        W = oracle.virial_pair(w.pos, w.box, 2.5, kind, p)
        h = 1e-6
        U = [oracle.pair_forces(w.pos * s, w.box * s, 2.5 * s, kind, p, 0)[1].sum() for s in (1 - h, 1 + h)]
        dU_dlnV = (U[1] - U[0]) / (2 * h) / 3.0
        if kind == "lj":                                                       # (sigma does not scale: U really changes)
            assert abs(W[:3].sum() + 3.0 * dU_dlnV) < 2e-6 * abs(W[:3].sum())
        else:
            assert abs(W[:3].sum() + 3.0 * dU_dlnV) < 2e-6 * max(1.0, abs(W[:3].sum()))
    # perfect FCC: the virial tensor is isotropic and its off-diagonal part vanishes by symmetry
    f = inputs.lj_fcc(4, rc=2.5, r_buff=0.4)
    W = oracle.virial_pair(f.pos, f.box, 2.5, "lj", (1.0, 1.0))
    assert np.abs(W[3:]).max() < 1e-9 * abs(W[0]) and abs(W[0] - W[1]) < 1e-9 * abs(W[0]) and abs(W[1] - W[2]) < 1e-9 * abs(W[0])


def test_dpd_virial_reduces_to_the_conservative_pair_form_and_equation_of_state():
    w = inputs.dpd_fluid(3000, pos_seed=4, vel_seed=5)
    p = w.params
    # gamma = 0 switches drag and noise off: F = A (1 - r/rc) rhat, whose virial is sum A (1 - r) r over pairs
    W = oracle.virial_dpd(w.pos, w.vel, w.box, 1.0, p["A"], 0.0, p["kT"], w.dt, 3, p["seed"])
    pairs = oracle.neighbor_pairs(w.pos, w.box, 1.0)
    d = w.pos[pairs[:, 0]] - w.pos[pairs[:, 1]]
    d -= w.box * np.rint(d / w.box)
    r = np.sqrt((d * d).sum(1))
    assert abs(W[:3].sum() - (p["A"] * (1.0 - r) * r).sum()) < 1e-10 * W[:3].sum()
    # tr W of the full force = sum over pairs of d . F_pair, F from the force routine on a two-particle system
    Wf = oracle.virial_dpd(w.pos[:2] * 0 + np.array([[0.0, 0, 0], [0.6, 0.1, -0.2]]), w.vel[:2], w.box, 1.0, p["A"], p["gamma"],
                           p["kT"], w.dt, 7, p["seed"])
    F2 = oracle.forces_dpd(np.array([[0.0, 0, 0], [0.6, 0.1, -0.2]]), w.vel[:2], w.box, 1.0, p["A"], p["gamma"], p["kT"],
                           w.dt, 7, p["seed"])
    assert abs(Wf[:3].sum() - np.dot(np.array([-0.6, -0.1, 0.2]), F2[0])) < 1e-13
    # Groot-Warren equation of state p = rho kT + 0.101 A rho^2 at rho = 3, A = 25 (= 25.7): weak, statistical pin on the
    # UNEQUILIBRATED uniform random start (ideal-gas structure: the mean-field value A rho^2 pi/30 = 23.6 + 3)
    P = oracle.pressure(w.vel, w.box, W)
    assert abs(P - (3.0 + math.pi / 30.0 * 25.0 * 9.0)) < 0.05 * P


# ------------------------------------------------------------------------------------------------- bonds
def test_fene_closed_form_gradient_and_harmonic_equivalence():
    k, r0 = 30.0, 1.5
    for r in (0.4, 0.97, 1.45):
        pos = _two(r, axis=(0.3, -1.0, 2.0))
        F, E, W = oracle.forces_bonds_kind(pos, BOX, [[0, 1]], "fene", k, r0)
        assert abs(E.sum() + 0.5 * k * r0 * r0 * math.log(1.0 - (r / r0) ** 2)) < 1e-12 * max(1.0, abs(E.sum()))
        Fr = -k * r / (1.0 - (r / r0) ** 2)                                    # attractive: pulls a towards b
        d = pos[0] - pos[1]
        d -= BOX * np.rint(d / BOX)
        assert np.abs(F[0] - Fr * d / r).max() < 1e-12 * abs(Fr) and np.abs(F[0] + F[1]).max() == 0.0
        assert abs(W[:3].sum() - r * Fr) < 1e-12 * abs(r * Fr)
        h = 1e-6
        U = [oracle.forces_bonds_kind(_two(x, axis=(0.3, -1.0, 2.0)), BOX, [[0, 1]], "fene", k, r0)[1].sum() for x in (r - h, r + h)]
        assert abs(Fr + (U[1] - U[0]) / (2 * h)) < 1e-6 * abs(Fr)
    assert abs(oracle.forces_bonds_kind(_two(1.4999999), BOX, [[0, 1]], "fene", k, r0)[0][0, 0]) > 1e7   # diverges at r0
    assert np.isnan(oracle.forces_bonds_kind(_two(1.6), BOX, [[0, 1]], "fene", k, r0)[0]).any()           # broken bond
    w = inputs.polymer_melt(8, chain_len=16)
    q = w.params
    Fh, Eh, Wh = oracle.forces_bonds_kind(w.pos, w.box, w.bonds, "harmonic", q["bond_k"], q["bond_r0"])
    F1, E1 = oracle.forces_bonds(w.pos, w.box, w.bonds, q["bond_k"], q["bond_r0"])
    assert np.array_equal(Fh, F1) and np.array_equal(Eh, E1)
    # bond virial by the box rescale (bond lengths scale with the box)
    h = 1e-6
    U = [oracle.forces_bonds(w.pos * s, w.box * s, w.bonds, q["bond_k"], q["bond_r0"])[1].sum() for s in (1 - h, 1 + h)]
    assert abs(Wh[:3].sum() + (U[1] - U[0]) / (2 * h)) < 1e-6 * abs(Wh[:3].sum())


# ------------------------------------------------------------------------------------------------- angles
def _tri(theta, l1=1.1, l2=0.8):
    b = np.array([5.8, 6.2, -6.9])                      # vertex next to the periodic boundary
    a = b + l1 * np.array([1.0, 0.0, 0.0])
    c = b + l2 * np.array([math.cos(theta), math.sin(theta), 0.0])
    return oracle.wrap(np.stack([a, b, c]), BOX)


def test_angle_zero_at_theta0_right_angle_closed_form_and_energy():
    k = 12.0
    F, E, W = oracle.forces_angles(_tri(2.0), BOX, [[0, 1, 2]], k, 2.0)
    assert np.abs(F).max() < 1e-13 and abs(E.sum()) < 1e-26
    th, th0 = math.pi / 2, 2.0
    F, E, W = oracle.forces_angles(_tri(th), BOX, [[0, 1, 2]], k, th0)
    assert abs(E.sum() - 0.5 * k * (th - th0) ** 2) < 1e-14 and abs(E[0] - E[1]) < 1e-16
    # at a right angle: |F_a| = k |theta - theta0| / l1, perpendicular to r1, opening the angle (theta < theta0)
    assert np.abs(F[0] - np.array([0.0, -k * (th0 - th) / 1.1, 0.0])).max() < 1e-13
    assert np.abs(F[2] - np.array([-k * (th0 - th) / 0.8, 0.0, 0.0])).max() < 1e-13
    assert np.abs(F.sum(axis=0)).max() < 1e-14


def test_angle_gradient_net_force_and_torque():
    rng = np.random.default_rng(5)
    w = inputs.polymer_melt(6, chain_len=12)
    ang = np.array([[12 * c + i, 12 * c + i + 1, 12 * c + i + 2] for c in range(6) for i in range(10)], dtype=np.uint32)
    k, th0 = 7.0, 1.9
    F, E, W = oracle.forces_angles(w.pos, w.box, ang, k, th0)
    assert np.abs(F.sum(axis=0)).max() < 1e-11 * np.abs(F).sum()
    # torque about the chain's own frame: unwrap each chain, sum r x F per chain = 0
    for c in range(6):
        x = w.pos[12 * c:12 * c + 12].copy()
        for i in range(1, 12):
            d = x[i] - x[i - 1]
            x[i] = x[i - 1] + d - w.box * np.rint(d / w.box)
        assert np.abs(np.cross(x, F[12 * c:12 * c + 12]).sum(axis=0)).max() < 1e-10 * np.abs(F).sum()
    for _ in range(6):                                   # F = -grad U by central differences on random coordinates
        i, a = int(rng.integers(0, w.N)), int(rng.integers(0, 3))
        h = 1e-6
        U = []
        for s in (-h, h):
            p = w.pos.copy(); p[i, a] += s
            U.append(oracle.forces_angles(p, w.box, ang, k, th0)[1].sum())
        assert abs(F[i, a] + (U[1] - U[0]) / (2 * h)) < 1e-6 * max(1.0, abs(F[i, a]))
    h = 1e-6                                             # angles do not change under a uniform rescale: zero virial trace
    assert abs(W[:3].sum()) < 1e-10 * np.abs(F).sum()


# ------------------------------------------------------------------------------------------------- dihedrals (R35)
def _quad(phi, l=(1.1, 0.9, 1.2), th=(1.9, 2.1)):
    """a-b-c-d with bond lengths l, bond angles th and dihedral angle phi, built by hand next to the periodic boundary."""
    b = np.array([5.7, -6.3, 6.6])
    c = b + l[1] * np.array([1.0, 0.0, 0.0])
    a = b + l[0] * np.array([math.cos(th[0]), math.sin(th[0]), 0.0])        # angle a-b-c = th[0], a in the xy plane (+y)
    d = c + l[2] * np.array([-math.cos(th[1]), math.sin(th[1]) * math.cos(phi), math.sin(th[1]) * math.sin(phi)])
    return oracle.wrap(np.stack([a, b, c, d]), BOX)


def test_dihedral_angle_special_values_and_invariance():
    for phi in (0.0, 0.4, math.pi / 2, 2.5, math.pi, -1.3):
        x = _quad(phi)
        got = oracle.dihedral_angle(x[0], x[1], x[2], x[3], BOX)
        assert abs(math.cos(got) - math.cos(phi)) < 1e-13 and abs(math.sin(got) - math.sin(phi)) < 1e-13
    # the sign convention is fixed by one hand-made case: d out of the abc plane towards +z of a right-handed frame
    assert abs(oracle.dihedral_angle([1, 1, 0], [0, 0, 0], [1, 0, 0], [1, 0, 1], [20, 20, 20]) - math.pi / 2) < 1e-15
    assert abs(oracle.dihedral_angle([1, 1, 0], [0, 0, 0], [1, 0, 0], [1, 0, -1], [20, 20, 20]) + math.pi / 2) < 1e-15
    # reversal of the chain (d, c, b, a) keeps phi; a rigid rotation keeps it too
    x = _quad(0.9)
    p0 = oracle.dihedral_angle(x[0], x[1], x[2], x[3], BOX)
    assert abs(oracle.dihedral_angle(x[3], x[2], x[1], x[0], BOX) - p0) < 1e-13
    rng = np.random.default_rng(2)
    Q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] *= -1
    y = (x - x[1]) - BOX * np.rint((x - x[1]) / BOX)
    y = y @ Q.T
    assert abs(oracle.dihedral_angle(y[0], y[1], y[2], y[3], [50, 50, 50]) - p0) < 1e-13


@pytest.mark.parametrize("s,n", [(1, 1), (-1, 1), (1, 2), (-1, 3)])
def test_dihedral_energy_gradient_net_force_torque_virial(s, n):
    k = 6.0
    for phi in (0.3, 1.1, 2.6, -0.8):
        x = _quad(phi)
        F, E, W = oracle.forces_dihedrals(x, BOX, [[0, 1, 2, 3]], k, s, n)
        p = oracle.dihedral_angle(x[0], x[1], x[2], x[3], BOX)
        assert abs(E.sum() - 0.5 * k * (1.0 + s * math.cos(n * p))) < 1e-14 and abs(E[0] - E[3]) < 1e-16
        assert np.abs(F.sum(axis=0)).max() < 1e-13
        y = (x - x[1]) - BOX * np.rint((x - x[1]) / BOX)
        assert np.abs(np.cross(y, F).sum(axis=0)).max() < 1e-12                      # no net torque
        assert abs(W[:3].sum()) < 1e-12                                               # angles do not feel a uniform rescale
        for i in range(4):
            for a in range(3):
                h = 1e-6
                U = []
                for sg in (-h, h):
                    z = x.copy(); z[i, a] += sg
                    U.append(oracle.forces_dihedrals(z, BOX, [[0, 1, 2, 3]], k, s, n)[1].sum())
                assert abs(F[i, a] + (U[1] - U[0]) / (2 * h)) < 2e-8 * max(1.0, np.abs(F).max())
    # extrema of the potential: no force at phi = 0 and pi
    for phi in (0.0, math.pi):
        assert np.abs(oracle.forces_dihedrals(_quad(phi), BOX, [[0, 1, 2, 3]], k, s, n)[0]).max() < 1e-12
    # many terms along chains: Newton's third law over the whole system
    w = inputs.polymer_melt(5, chain_len=12)
    dih = np.array([[12 * c + i, 12 * c + i + 1, 12 * c + i + 2, 12 * c + i + 3] for c in range(5) for i in range(9)], dtype=np.uint32)
    F, E, W = oracle.forces_dihedrals(w.pos, w.box, dih, k, s, n)
    assert np.abs(F.sum(axis=0)).max() < 1e-11 * max(1.0, np.abs(F).sum())


# ---- R36 Langevin thermostat ------------------------------------------------------------------------------------------
def test_langevin_uniforms_stream_and_moments():
    """u_k = 2 (X_k + 0.5) 2^-32 - 1 from the KAT-pinned Philox with counter (tag, 0xffffffff, step lo, step hi); range,
    mean 0, variance 1/3, the three components and successive steps / tags uncorrelated; stream apart from DPD's."""
    for tag, step, seed in [(0, 0, 0), (5, 7, 0x1234), (123456, (1 << 33) + 5, (0xdeadbeef << 32) | 77)]:
        X = oracle.philox4x32_10([tag, 0xFFFFFFFF, step & 0xFFFFFFFF, step >> 32], [seed & 0xFFFFFFFF, seed >> 32])
        u = oracle.langevin_u(tag, step, seed)
        want = [(int(x) * 2 + 1) / 2.0 ** 32 - 1.0 for x in X[:3]]      # = 2 (X + 0.5) 2^-32 - 1, exact in fp64
        assert u.tolist() == want
    n = 40000
    U = np.array([oracle.langevin_u(t, 11, 99) for t in range(n)])
    assert U.min() > -1.0 and U.max() < 1.0
    assert np.abs(U.mean(axis=0)).max() < 4.0 / math.sqrt(3 * n)
    assert np.abs(U.var(axis=0) - 1.0 / 3.0).max() < 4.0 * math.sqrt(4.0 / 45.0 / n)      # Var(u^2) = 1/5 - 1/9
    c = np.corrcoef(U.T)
    assert np.abs(c - np.eye(3)).max() < 4.0 / math.sqrt(n)
    U2 = np.array([oracle.langevin_u(t, 12, 99) for t in range(n)])
    assert abs(np.corrcoef(U[:, 0], U2[:, 0])[0, 1]) < 4.0 / math.sqrt(n)          # next step
    assert abs(np.corrcoef(U[:-1, 0], U[1:, 0])[0, 1]) < 4.0 / math.sqrt(n)        # next tag
    # not the DPD stream: theta of the pair (tag, anything) never reuses these words' counter (second word 0xffffffff)
    th = oracle.dpd_theta(3, 4, 11, 99) / math.sqrt(3.0)
    assert all(abs(th - x) > 1e-12 for x in oracle.langevin_u(3, 11, 99))


def test_langevin_force_limits_and_accumulation():
    rng = np.random.default_rng(5)
    v = rng.normal(size=(50, 3))
    F0 = rng.normal(size=(50, 3))
    # kT = 0: pure drag, added to what is there
    F = oracle.forces_langevin(v, 2.5, 0.0, 0.01, 3, 8, force=F0.copy())
    assert np.abs(F - (F0 - 2.5 * v)).max() < 1e-15
    # v = 0: pure noise of amplitude sqrt(6 gamma kT / dt) u
    F = oracle.forces_langevin(np.zeros((50, 3)), 2.5, 1.7, 0.01, 3, 8)
    U = np.array([oracle.langevin_u(t, 3, 8) for t in range(50)])
    assert np.abs(F - math.sqrt(6 * 2.5 * 1.7 / 0.01) * U).max() < 1e-12
    # gamma = 0 switches the thermostat off
    assert np.abs(oracle.forces_langevin(v, 0.0, 1.7, 0.01, 3, 8)).max() == 0.0
    # variance of a component 2 gamma kT / dt
    n = 30000
    F = oracle.forces_langevin(np.zeros((n, 3)), 0.8, 1.3, 0.02, 21, 4)
    assert abs(F.var() / (2 * 0.8 * 1.3 / 0.02) - 1.0) < 4.0 * math.sqrt(0.8 / (3 * n))  # kurtosis of a uniform: Var(u^2)/Var(u)^2 = 0.8


def test_langevin_free_particles_decay_and_equilibrium():
    """Free particles (no other force) through Sim's velocity-Verlet: the half-step velocity obeys
    v_h' = (1 - gamma dt / m) v_h + (dt / m) R, so (a) at kT = 0 it decays by exactly (1 - gamma dt / m) per step and
    (b) its stationary variance is (kT / m) / (1 - gamma dt / (2 m)) -- both closed forms of the discrete scheme."""
    box, N, dt, g = 50.0, 4000, 0.01, 3.0
    rng = np.random.default_rng(2)
    pos = rng.uniform(0, box, size=(N, 3))
    v0 = rng.normal(size=(N, 3))
    s = oracle.Sim(pos, v0, box, 1.0, 0.4, {"langevin": dict(gamma=g, kT=0.0, seed=1)})
    s.run(1, dt)
    # after step 1: v = v_h1 (1 - a/2) with v_h1 = v0 (1 - a/2) (F(t0) = -gamma v0), a = gamma dt
    a = g * dt
    assert np.abs(s.vel - v0 * (1 - a / 2) ** 2).max() < 1e-14
    s.run(9, dt)
    # v after n steps = v_h,n (1 - a/2), v_h,n = v_h,1 (1 - a)^(n-1)
    assert np.abs(s.vel - v0 * (1 - a / 2) ** 2 * (1 - a) ** 9).max() < 1e-13
    # (b) equilibrium: long run from cold, many particles; full-step velocity v = v_h (1 - a/2) + (dt/2m) R'
    kT, g, dt = 1.5, 5.0, 0.02
    a = g * dt
    s = oracle.Sim(pos, np.zeros((N, 3)), box, 1.0, 0.4, {"langevin": dict(gamma=g, kT=kT, seed=7)})
    s.run(300, dt)                                  # 300 dt = 30 relaxation times 1/gamma
    var_h = kT / (1 - a / 2)                        # stationary variance of the half-step velocity
    var_full = var_h * (1 - a / 2) ** 2 + (dt / 2) ** 2 * (2 * g * kT / dt)
    got = (s.vel ** 2).mean()
    assert abs(got / var_full - 1.0) < 4.0 * math.sqrt(2.0 / (3 * N))


# ---- R37 tabulated pair potential -------------------------------------------------------------------------------------
def _two_at(r, box=20.0, direction=(0.36, -0.48, 0.8)):
    d = np.array(direction) / np.linalg.norm(direction)
    return np.array([[1.0, 2.0, 3.0], np.array([1.0, 2.0, 3.0]) - r * d]), box, d      # d = unit vector from b to a


def test_pair_table_nodes_linear_tables_and_range():
    r_min, r_max, M = 0.5, 2.5, 41                       # h = 0.05
    rk = np.linspace(r_min, r_max, M)
    rng = np.random.default_rng(3)
    U, F = rng.normal(size=M), rng.normal(size=M)
    # at a node the table values come back; between two nodes the straight line between them
    for k, t in [(0, 0.0), (7, 0.0), (7, 0.25), (39, 0.5), (39, 0.999)]:
        r = rk[k] + t * (rk[1] - rk[0])
        pos, box, d = _two_at(r)
        Fo, E, W = oracle.pair_table(pos, box, r_min, r_max, U, F)
        f = F[k] + t * (F[k + 1] - F[k])
        u = U[k] + t * (U[k + 1] - U[k])
        assert np.abs(Fo[0] - f * d).max() < 1e-12 and np.abs(Fo[0] + Fo[1]).max() == 0.0
        assert abs(E[0] - 0.5 * u) < 1e-12 and abs(E[1] - 0.5 * u) < 1e-12
        assert abs(W[0] + W[1] + W[2] - r * f) < 1e-12                     # tr W = r F(r) for one pair
    # a table that is linear in r is reproduced at any r
    a0, a1, b0, b1 = 1.5, -0.7, 0.3, 2.0
    for r in (0.5, 0.777, 1.93, 2.4999):
        pos, box, d = _two_at(r)
        Fo, E, _ = oracle.pair_table(pos, box, r_min, r_max, a0 + a1 * rk, b0 + b1 * rk)
        assert np.abs(Fo[0] - (b0 + b1 * r) * d).max() < 1e-12 and abs(2 * E[0] - (a0 + a1 * r)) < 1e-12
    # outside [r_min, r_max): nothing; strict at r_max
    for r in (0.49, 0.4999999, 2.5, 2.6):
        pos, box, d = _two_at(r)
        Fo, E, W = oracle.pair_table(pos, box, r_min, r_max, U, F)
        assert np.abs(Fo).max() == 0.0 and np.abs(E).max() == 0.0 and np.abs(W).max() == 0.0
    # through the periodic wrap
    pos, box, d = _two_at(1.2, box=6.0)
    pos2 = pos.copy(); pos2[1] += [6.0, -6.0, 0.0]
    A, B_ = oracle.pair_table(pos, box, r_min, r_max, U, F), oracle.pair_table(oracle.wrap(pos2, box), box, r_min, r_max, U, F)
    assert np.abs(A[0] - B_[0]).max() < 1e-12


def test_pair_table_of_lj_converges_to_lj_at_second_order():
    """A table filled from the LJ closed forms reproduces orc_forces_lj on a liquid-like configuration with the error of
    linear interpolation, h^2/8 max|f''|: quartering h gives 1/16 of the error."""
    rng = np.random.default_rng(8)
    n = 5
    g = (np.stack(np.meshgrid(*[np.arange(n)] * 3, indexing="ij"), -1).reshape(-1, 3) + 0.5) * 1.2
    pos = g + rng.uniform(-0.08, 0.08, size=g.shape)
    box, rc, r_min = n * 1.2, 2.5, 0.8
    Fr, Er = oracle.forces_lj(pos, box, rc, 1.0, 1.0, 0)
    errs = []
    for M in (1701, 6801):
        rk = np.linspace(r_min, rc, M)
        U = 4 * (rk ** -12 - rk ** -6)
        F = 24 * (2 * rk ** -13 - rk ** -7)
        Fo, E, W = oracle.pair_table(pos, box, r_min, rc, U, F)
        errs.append(np.abs(Fo - Fr).max())
        assert np.abs(E - Er).max() < 30 * (rk[1] - rk[0]) ** 2
        Wr = oracle.virial_pair(pos, box, rc, "lj", (1.0, 1.0))
        assert np.abs(W - Wr).max() < 1e-3 * np.abs(Wr).max()
    assert errs[0] < 2e-3 and 12.0 < errs[0] / errs[1] < 20.0
    assert np.abs(Fo.sum(axis=0)).max() < 1e-11                      # Newton's third law


# ---- R38 tabulated bonds ----------------------------------------------------------------------------------------------
def test_bond_table_nodes_lines_range_and_accumulation():
    r_min, r_max, M = 0.4, 1.6, 25                       # h = 0.05
    rk = np.linspace(r_min, r_max, M)
    rng = np.random.default_rng(31)
    U, F = rng.normal(size=M), rng.normal(size=M)
    bond = np.array([[0, 1]], dtype=np.uint32)
    for k, t in [(0, 0.0), (5, 0.0), (5, 0.4), (23, 0.5), (23, 0.999)]:
        r = rk[k] + t * (rk[1] - rk[0])
        pos, box, d = _two_at(r)
        Fo, E, W = oracle.bond_table(pos, box, bond, r_min, r_max, U, F)
        f = F[k] + t * (F[k + 1] - F[k])
        u = U[k] + t * (U[k + 1] - U[k])
        assert np.abs(Fo[0] - f * d).max() < 1e-12 and np.abs(Fo[0] + Fo[1]).max() == 0.0
        assert abs(E[0] - 0.5 * u) < 1e-12 and abs(E[1] - 0.5 * u) < 1e-12
        assert abs(W[0] + W[1] + W[2] - r * f) < 1e-12
    # a bond that has left its table is broken: NaN on both ends (like FENE beyond r0)
    for r in (0.39, 1.6, 1.7):
        pos, box, d = _two_at(r)
        Fo, E, _ = oracle.bond_table(pos, box, bond, r_min, r_max, U, F)
        assert np.isnan(Fo).all() and np.isnan(E).all()
    # accumulates onto what is there; the reversed bond gives the same forces; through the wrap
    pos, box, d = _two_at(1.1, box=5.0)
    F0 = rng.normal(size=(2, 3)); E0 = rng.normal(size=2); W0 = rng.normal(size=6)
    A = oracle.bond_table(pos, box, bond, r_min, r_max, U, F)
    Bc = oracle.bond_table(pos, box, bond, r_min, r_max, U, F, force=F0.copy(), energy=E0.copy(), virial=W0.copy())
    assert np.abs(Bc[0] - (F0 + A[0])).max() < 1e-15 and np.abs(Bc[1] - (E0 + A[1])).max() < 1e-15
    assert np.abs(Bc[2] - (W0 + A[2])).max() < 1e-15
    R = oracle.bond_table(pos, box, bond[:, ::-1], r_min, r_max, U, F)
    assert np.abs(R[0] - A[0]).max() < 1e-15 and np.abs(R[2] - A[2]).max() < 1e-15
    pos2 = pos.copy(); pos2[1] += [-5.0, 5.0, 5.0]
    assert np.abs(oracle.bond_table(oracle.wrap(pos2, box), box, bond, r_min, r_max, U, F)[0] - A[0]).max() < 1e-12


def test_bond_table_of_the_harmonic_bond_is_the_harmonic_bond():
    """F of a harmonic bond is linear in r, so its table reproduces orc_forces_bonds exactly (to rounding) on a chain;
    U is quadratic: the interpolation error is at most k h^2 / 8 per bond."""
    rng = np.random.default_rng(32)
    n = 40
    steps = rng.normal(size=(n - 1, 3)); steps *= (rng.uniform(0.7, 1.3, size=n - 1) / np.linalg.norm(steps, axis=1))[:, None]
    pos = oracle.wrap(np.vstack([[3.0, 3.0, 3.0], 3.0 + np.cumsum(steps, axis=0)]), 9.0)
    bonds = np.stack([np.arange(n - 1), np.arange(1, n)], axis=1).astype(np.uint32)
    k, r0, r_min, r_max, M = 30.0, 0.9, 0.5, 1.5, 201
    rk = np.linspace(r_min, r_max, M)
    Ft, Et, Wt = oracle.bond_table(pos, 9.0, bonds, r_min, r_max, 0.5 * k * (rk - r0) ** 2, -k * (rk - r0))
    Fh, Eh, Wh = oracle.forces_bonds_kind(pos, 9.0, bonds, "harmonic", k, r0)
    assert np.abs(Ft - Fh).max() < 1e-11 and np.abs(Wt - Wh).max() < 1e-11
    h = rk[1] - rk[0]
    assert 0.0 <= (Et - Eh).min() and (Et - Eh).max() <= 2 * 0.5 * k * h * h / 8 + 1e-12   # chord above a convex U; 2 bonds per bead


# ---- degenerate bonded terms (R34, R35): collinear particles -----------------------------------------------------------
def test_collinear_angle_and_dihedral_terms_are_skipped():
    """theta = 0 or pi has no defined gradient direction (sin theta = 0), and a dihedral with three collinear particles no
    defined angle: both terms are skipped (no force, no energy, no NaN), while the same particles moved off the line by
    1e-6 give finite values that follow the closed forms."""
    box = 20.0
    line = np.array([[0.0, 0.0, 0.0], [1.0, 0.0, 0.0], [2.1, 0.0, 0.0], [3.0, 0.5, 0.0]])
    F, E, W = oracle.forces_angles(line, box, np.array([[0, 1, 2]], dtype=np.uint32), 7.0, 2.0)
    assert np.abs(F).max() == 0.0 and np.abs(E).max() == 0.0 and np.abs(W).max() == 0.0
    fold = line.copy(); fold[2] = [0.4, 0.0, 0.0]                       # theta = 0: c folded back onto the a side
    F, E, _ = oracle.forces_angles(fold, box, np.array([[0, 1, 2]], dtype=np.uint32), 7.0, 2.0)
    assert np.abs(F).max() == 0.0 and np.abs(E).max() == 0.0
    bent = line.copy(); bent[2, 1] = 1e-6
    F, E, _ = oracle.forces_angles(bent, box, np.array([[0, 1, 2]], dtype=np.uint32), 7.0, 2.0)
    th = math.pi - math.atan2(1e-6, 1.1)
    assert np.isfinite(F).all() and abs(E.sum() - 0.5 * 7.0 * (th - 2.0) ** 2) < 1e-9
    # dihedral: a, b, c collinear (A = F x G = 0), then b, c, d collinear (B = 0)
    q = np.array([[0, 1, 2, 3]], dtype=np.uint32)
    for pts in (line, line[::-1].copy()):
        F, E, W = oracle.forces_dihedrals(pts, box, q, 3.0, 1, 2)
        assert np.abs(F).max() == 0.0 and np.abs(E).max() == 0.0 and np.abs(W).max() == 0.0
    off = line.copy(); off[0] = [0.0, 0.0, 1e-3]                        # a lifted out of the line: phi = +-pi/2 exactly
    F, E, _ = oracle.forces_dihedrals(off, box, q, 3.0, 1, 2)
    assert np.isfinite(F).all() and abs(abs(oracle.dihedral_angle(*off, box)) - 0.5 * math.pi) < 1e-12
    assert abs(E.sum() - 0.5 * 3.0 * (1.0 + math.cos(math.pi))) < 1e-9  # U = k/2 (1 + cos(2 phi)) = 0 at phi = pi/2
    assert abs(F.sum(axis=0)).max() < 1e-6 * np.abs(F).max()


def test_probe_pair_forces_are_the_rows_of_the_full_routines():
    rng = np.random.default_rng(41)
    n = 5
    g = (np.stack(np.meshgrid(*[np.arange(n)] * 3, indexing="ij"), -1).reshape(-1, 3) + 0.5) * 1.25
    pos = g + rng.uniform(-0.1, 0.1, size=g.shape)
    box, rc = n * 1.25, 2.5
    probes = np.array([0, 7, 63, 124], dtype=np.uint32)
    for kind, p in (("yukawa", (2.0, 1.5)), ("gaussian", (3.0, 0.8)), ("morse", (1.7, 2.0, 1.0)), ("lj", (0.9, 1.05))):
        for shift in (0, 1):
            F, E = oracle.pair_forces(pos, box, rc, kind, p, shift)
            Fp, Ep = oracle.probe_pair_forces(pos, box, rc, kind, p, probes, shift)
            assert np.abs(Fp - F[probes]).max() < 1e-12 * np.abs(F).max() and np.abs(Ep - E[probes]).max() < 1e-12 * np.abs(E).max()
    U, Ft = rng.normal(size=65), rng.normal(size=65)
    F, E, _ = oracle.pair_table(pos, box, 0.6, 2.2, U, Ft)
    Fp, Ep = oracle.probe_pair_forces(pos, box, rc, "table", (), probes, table=(0.6, 2.2, U, Ft))
    assert np.abs(Fp - F[probes]).max() < 1e-12 * np.abs(F).max() and np.abs(Ep - E[probes]).max() < 1e-12 * np.abs(E).max()
