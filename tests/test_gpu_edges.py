"""-m gpu edge cases of the hot path: one and two particles, boxes that are almost empty (most cells and whole tiles hold
no particle), a box at the smallest legal size with overlapping particles; every kernel variant (fp64, mixed, DPD) against the O(N^2) oracle.  Neighbour lists bit-exact, forces within the bars of test_gpu_parity.py."""
import numpy as np
import pytest

import oracle
from paper_1412_3387_b200 import binding as B
from gpu_util import sort_pairs, force_rel_err

pytestmark = pytest.mark.gpu

CASES = [(1, 9.0), (2, 9.0), (7, 30.0), (50, 40.0), (333, 9.1)]


@pytest.mark.parametrize("prec", [B.MD_FP64, B.MD_MIXED])
@pytest.mark.parametrize("N,L", CASES)
def test_lj_sparse_and_tiny_systems(prec, N, L):
    rng = np.random.default_rng(100 * N + int(L))
    box = np.array([L, L * 1.1, L * 1.3])
    pos = (rng.random((N, 3)) - 0.5) * box
    if N == 2:
        pos[1] = pos[0] + [1.1, 0.2, -0.3]                      # one interacting pair
    vel = rng.normal(size=(N, 3)) * 0.5
    wpos = oracle.wrap(pos, box)
    ref = oracle.neighbor_pairs(wpos, box, 2.9)
    Fr, _ = oracle.forces_lj(wpos, box, 2.5)
    tol = 1e-10 if prec == B.MD_FP64 else 1e-4
    for _ in (0,):
        md = B.MD(box, N, 2.5, 0.4, precision=prec)
        md.set_state(pos, vel)
        md.build_nlist()
        assert np.array_equal(sort_pairs(md.get_nlist()), ref)
        md.forces_lj()
        F, _ = md.get_forces()
        assert force_rel_err(F, Fr) <= tol or np.abs(F - Fr).max() <= 1e-13       # R11 (all-zero forces: absolute)
        md.step(B.step_desc("lj", 0.002, dict(epsilon=1.0, sigma=1.0, energy_shift=1)), 5)
        if N <= 50:   # (the dense random box has overlapping particles: they fly apart faster than any skin)
            assert md.stats()["dangerous_builds"] == 0
        t = md.thermo()
        assert np.isfinite(t["kinetic"]) and np.isfinite(t["potential"])


@pytest.mark.parametrize("N,L", [(1, 5.0), (3, 12.0), (40, 4.3)])
def test_dpd_sparse_and_tiny_systems(N, L):
    rng = np.random.default_rng(7 * N)
    box = np.array([L, L, L * 1.2])
    pos = (rng.random((N, 3)) - 0.5) * box
    vel = rng.normal(size=(N, 3))
    wpos = oracle.wrap(pos, box)
    md = B.MD(box, N, 1.0, 0.4)
    md.set_state(pos, vel)
    md.build_nlist()
    assert np.array_equal(sort_pairs(md.get_nlist()), oracle.neighbor_pairs(wpos, box, 1.4))
    md.forces_dpd(25.0, 4.5, 1.0, 0.02, 9, 42)
    F, _ = md.get_forces()
    Fr = oracle.forces_dpd(wpos, vel, box, 1.0, 25.0, 4.5, 1.0, 0.02, 9, 42)
    assert force_rel_err(F, Fr) <= 1e-10 or np.abs(F - Fr).max() <= 1e-13


@pytest.mark.parametrize("prec", [B.MD_FP64, B.MD_MIXED])
def test_inhomogeneous_slab_grows_the_row_stride(prec):
    """All particles in a slab a quarter of the box wide: local density 4x the mean, so the rows are ~4x longer than the
    density-based stride estimate -> the build reports the overflow, the stride grows and the list is built again."""
    rng = np.random.default_rng(1)
    box = np.array([14.0, 14.0, 14.0])
    N = 1500
    pos = (rng.random((N, 3)) - 0.5) * box
    pos[:, 0] = (rng.random(N) - 0.5) * 3.5
    wpos = oracle.wrap(pos, box)
    ref = oracle.neighbor_pairs(wpos, box, 2.9)
    assert 2 * len(ref) / N > 2.5 * (N / box.prod()) * 4.18879 * 2.9 ** 3        # rows far beyond the mean-density estimate
    md = B.MD(box, N, 2.5, 0.4, precision=prec)
    md.set_state(pos, np.zeros((N, 3)))
    md.build_nlist()
    assert np.array_equal(sort_pairs(md.get_nlist()), ref)
    assert abs(md.stats()["mean_neighbors"] - 2 * len(ref) / N) < 0.01 * 2 * len(ref) / N
    md.forces_lj()
    F, _ = md.get_forces()
    Fr, _ = oracle.forces_lj(wpos, box, 2.5)
    assert force_rel_err(F, Fr) <= (1e-10 if prec == B.MD_FP64 else 1e-4)
