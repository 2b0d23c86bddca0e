"""Pins for the oracle's Lennard-Jones force/energy (O4) -- closed forms, FCC shell sums, invariants."""
import itertools
import math
import os
from collections import Counter

import numpy as np

import oracle
from paper_1412_3387_b200 import inputs

GOLD = {}
for _l in open(os.path.join(os.path.dirname(__file__), "golden", "lj_closed_forms.txt")):
    if _l.strip() and not _l.startswith("#"):
        k, v = _l.split()
        GOLD[k] = float(v)

BOX = np.array([20.0, 20.0, 20.0])


def _two(r, axis=0, shift=0):
    pos = np.zeros((2, 3))
    pos[0, axis] = 0.5 * r
    pos[1, axis] = -0.5 * r
    return oracle.forces_lj(pos, BOX, 3.5, 1.0, 1.0, shift)


def test_force_vanishes_at_minimum_and_energy_is_minus_eps():
    F, E = _two(GOLD["r_min"])
    assert np.abs(F).max() < 1e-13
    assert abs(E.sum() - GOLD["U_at_r_min"]) < 1e-14


def test_closed_form_energy_and_force_at_cutoffs():
    for r, name in ((2.5, "2.5"), (3.0, "3.0")):
        F, E = _two(r)
        assert abs(E.sum() - GOLD["U_at_" + name]) < 1e-13            # unshifted U(rc)
        # force on particle 0 (at +r/2) along +x is F(r) = -dU/dr: attractive -> negative
        assert abs(F[0, 0] - GOLD["F_at_" + name]) < 1e-13
        assert abs(F[1, 0] + GOLD["F_at_" + name]) < 1e-13
        assert np.abs(F[:, 1:]).max() == 0.0


def test_energy_shift_is_U_of_rc_and_truncation_is_strict():
    pos = np.zeros((2, 3))
    pos[0, 0] = 1.7
    F0, E0 = oracle.forces_lj(pos, BOX, 2.5, 1.0, 1.0, 0)
    F1, E1 = oracle.forces_lj(pos, BOX, 2.5, 1.0, 1.0, 1)
    assert np.array_equal(F0, F1)                                     # shift never changes forces
    assert abs((E0.sum() - E1.sum()) - GOLD["U_at_2.5"]) < 1e-15
    pos[0, 0] = 2.5                                                   # r == rc exactly: excluded (strict <)
    F, E = oracle.forces_lj(pos, BOX, 2.5, 1.0, 1.0, 0)
    assert np.abs(F).max() == 0.0 and E.sum() == 0.0
    pos[0, 0] = np.nextafter(2.5, 0.0)
    F, E = oracle.forces_lj(pos, BOX, 2.5, 1.0, 1.0, 0)
    assert abs(F[0, 0] - GOLD["F_at_2.5"]) < 1e-12


def test_force_is_minus_gradient_of_energy():
    rng = np.random.default_rng(5)
    w = inputs.lj_fcc(3, rc=2.5, jitter=0.08, pos_seed=11)            # N=108, L=5.04... too small for rc: use bigger box
    pos = w.pos * 1.25
    box = w.box * 1.25                                                # L = 6.3 > 2 rc
    F, E = oracle.forces_lj(pos, box, 2.5, 1.0, 1.0, 1)
    h = 1e-5
    for i, a in ((0, 0), (17, 1), (55, 2), (101, 0)):
        p = pos.copy(); p[i, a] += h
        m = pos.copy(); m[i, a] -= h
        Up = oracle.forces_lj(p, box, 2.5)[1].sum()
        Um = oracle.forces_lj(m, box, 2.5)[1].sum()
        # pairs crossing rc within +-h would break this; the shifted potential is continuous, the error is O(h)*F(rc)
        assert abs(-(Up - Um) / (2 * h) - F[i, a]) < 5e-6 * max(1.0, abs(F[i, a]))


def test_epsilon_sigma_scaling():
    # U(r; eps, sigma) = eps * U(r/sigma; 1, 1);  F = eps/sigma * F(r/sigma)
    pos = np.zeros((2, 3)); pos[0, 1] = 1.3 * 1.7
    F, E = oracle.forces_lj(pos, BOX, 2.5 * 1.7, 0.6, 1.7, 0)
    pos1 = np.zeros((2, 3)); pos1[0, 1] = 1.3
    F1, E1 = oracle.forces_lj(pos1, BOX, 2.5, 1.0, 1.0, 0)
    assert abs(E.sum() - 0.6 * E1.sum()) < 1e-14
    assert abs(F[0, 1] - 0.6 / 1.7 * F1[0, 1]) < 1e-14


def test_newton_third_law_and_translation_invariance():
    w = inputs.lj_fcc(4, rc=2.5, jitter=0.1, pos_seed=3)              # N=256, L=6.72
    F, E = oracle.forces_lj(w.pos, w.box, 2.5)
    assert np.abs(F.sum(axis=0)).max() < 1e-11 * np.abs(F).sum()
    # rigid shift through the periodic boundary leaves forces unchanged (exercises the minimum image)
    shifted = inputs.wrap(w.pos + np.array([3.1, -2.2, 0.7]), w.box)
    F2, E2 = oracle.forces_lj(shifted, w.box, 2.5)
    assert np.abs(F2 - F).max() < 1e-9 * np.abs(F).max()
    assert abs(E2.sum() - E.sum()) < 1e-10 * abs(E.sum())


def _fcc_shells(R=4):
    """Shell table of the FCC lattice from integer lattice vectors (independent of any pair search):
    {n: count} for squared distance n/2 in units of a^2."""
    basis = [(0, 0, 0), (.5, .5, 0), (.5, 0, .5), (0, .5, .5)]
    sh = Counter()
    for i, j, k in itertools.product(range(-R, R + 1), repeat=3):
        for b in basis:
            d2 = (i + b[0]) ** 2 + (j + b[1]) ** 2 + (k + b[2]) ** 2
            if d2 > 0:
                sh[round(2 * d2)] += 1
    return sh


def test_perfect_fcc_shell_sums():
    """Configs 1 and 5 at t=0: neighbour counts, energy per particle and zero forces follow from the
    lattice shells (SURVEY 8(c) pin: 78 list neighbours / 54 within rc=2.5, U/N = -6.332811992581)."""
    sh = _fcc_shells()
    w = inputs.config(1)
    a = w.box[0] / 10
    u = lambda r: 4 * (r ** -12 - r ** -6)
    n_list = sum(c for n, c in sh.items() if a * math.sqrt(n / 2) < w.r_list)
    n_rc = sum(c for n, c in sh.items() if a * math.sqrt(n / 2) < w.rc)
    U = sum(0.5 * c * (u(a * math.sqrt(n / 2)) - u(w.rc)) for n, c in sh.items() if a * math.sqrt(n / 2) < w.rc)
    assert (n_list, n_rc) == (78, 54)
    assert abs(U - (-6.332811992581)) < 1e-11
    F, E = oracle.forces_lj(w.pos, w.box, w.rc, 1.0, 1.0, 1)
    assert np.abs(E - U).max() < 1e-12                               # every particle has the same energy
    assert np.abs(F).max() < 1e-12                                   # and zero force by symmetry
    pairs = oracle.neighbor_pairs(w.pos, w.box, w.r_list)
    assert pairs.shape[0] == 39 * w.N                                # 78/2 per particle
    deg = np.bincount(pairs.reshape(-1), minlength=w.N)
    assert deg.min() == 78 and deg.max() == 78


def test_perfect_fcc_rc3():
    """Unjittered config-2 lattice (small replica): 140 list neighbours (r_list 3.4), 86 within rc=3.0,
    U/N = -6.700547102519."""
    sh = _fcc_shells()
    w = inputs.lj_fcc(7, rc=3.0, r_buff=0.4)                          # L = 11.76 >= 3*3.4
    a = w.box[0] / 7
    u = lambda r: 4 * (r ** -12 - r ** -6)
    in_rc = [(n, c) for n, c in sh.items() if a * math.sqrt(n / 2) < 3.0]
    assert sum(c for n, c in sh.items() if a * math.sqrt(n / 2) < 3.4) == 140
    assert sum(c for _, c in in_rc) == 86
    U = sum(0.5 * c * (u(a * math.sqrt(n / 2)) - u(3.0)) for n, c in in_rc)
    assert abs(U - (-6.700547102519)) < 1e-11
    F, E = oracle.forces_lj(w.pos, w.box, 3.0, 1.0, 1.0, 1)
    assert np.abs(E - U).max() < 1e-12 and np.abs(F).max() < 1e-12
    deg = np.bincount(oracle.neighbor_pairs(w.pos, w.box, 3.4).reshape(-1), minlength=w.N)
    assert deg.min() == 140 and deg.max() == 140


def test_probe_rows_equal_full_rows():
    w = inputs.lj_fcc(4, rc=2.5, jitter=0.1, pos_seed=8)
    F, E = oracle.forces_lj(w.pos, w.box, 2.5)
    pr = inputs.probe_tags(w.N, 40, seed=1)
    Fp, Ep = oracle.probe_forces_lj(w.pos, w.box, 2.5, pr)
    assert np.abs(Fp - F[pr]).max() < 1e-11 * np.abs(F).max()
    assert np.abs(Ep - E[pr]).max() < 1e-12 * np.abs(E).max()
