"""Pins for the oracle's cell assignment (O1), neighbour set (O2), rebuild trigger (O3), probe rows (O9)."""
import numpy as np
import pytest
from scipy.spatial import cKDTree

import oracle
from paper_1412_3387_b200 import inputs


def _numpy_pairs(pos, box, r):
    """Independent vectorised brute force with a different minimum-image formula (d - L rint(d/L))."""
    out = []
    for i in range(pos.shape[0] - 1):
        d = pos[i] - pos[i + 1:]
        d -= box * np.rint(d / box)
        j = np.nonzero((d * d).sum(1) < r * r)[0] + i + 1
        out.append(np.stack([np.full(j.shape, i), j], 1))
    return np.concatenate(out).astype(np.uint32)


@pytest.mark.parametrize("N,box,r,seed", [
    (300, (9.0, 9.0, 9.0), 2.9, 1),         # L just >= 3 r_list: every pair of cells is adjacent through the wrap
    (500, (4.3, 5.1, 6.7), 1.4, 2),         # orthorhombic
    (2000, (13.0, 13.0, 13.0), 3.4, 3),
])
def test_neighbor_pairs_equal_kdtree_and_numpy(N, box, r, seed):
    box = np.array(box)
    pos = inputs.random_box(N, box, seed)
    got = oracle.neighbor_pairs(pos, box, r)
    # sorted, a<b, unique
    assert np.all(got[:, 0] < got[:, 1])
    key = got[:, 0].astype(np.uint64) << np.uint64(32) | got[:, 1].astype(np.uint64)
    assert np.all(np.diff(key.astype(np.int64)) > 0)
    # library routine: periodic k-d tree (positions shifted to [0, L))
    kd = cKDTree(pos + 0.5 * box, boxsize=box)
    ref = np.array(sorted(kd.query_pairs(r)), dtype=np.uint32).reshape(-1, 2)
    # pairs within 1e-9 of the radius may differ by rounding; none are expected for random input
    assert np.array_equal(got, ref)
    assert np.array_equal(got, _numpy_pairs(pos, box, r))


def test_neighbor_radius_is_strict():
    box = np.array([12.0, 12.0, 12.0])
    pos = np.array([[0.0, 0.0, 0.0], [2.0, 0.0, 0.0], [0.0, np.nextafter(2.0, 0.0), 0.0], [-5.5, 0, 0], [5.5, 0, 0]])
    got = oracle.neighbor_pairs(pos, box, 2.0)
    # |x0-x1| == r exactly -> NOT a neighbour; x2 just inside -> neighbour; 3-4 are 1.0 apart through the wrap
    assert [tuple(p) for p in got] == [(0, 2), (3, 4)]


def test_probe_rows_equal_full_list():
    box = np.array([10.0, 9.0, 11.0])
    pos = inputs.random_box(800, box, 7)
    pairs = oracle.neighbor_pairs(pos, box, 2.9)
    probes = inputs.probe_tags(800, 64, seed=2)
    counts, nbrs = oracle.probe_nlist(pos, box, 2.9, probes, row_stride=256)
    for p, c, row in zip(probes, counts, nbrs):
        ref = np.sort(np.concatenate([pairs[pairs[:, 0] == p, 1], pairs[pairs[:, 1] == p, 0]]))
        assert c == len(ref)
        assert np.array_equal(row[:c], ref)


def test_cell_dims_and_containment():
    box = np.array([16.795962, 13.1, 9.0])
    r_list = 2.9
    dims = oracle.cell_dims(box, r_list)
    assert list(dims) == [5, 4, 3]
    pos = inputs.random_box(5000, box, 11)
    cell, dims2 = oracle.cell_assign(pos, box, r_list)
    assert np.array_equal(dims, dims2)
    assert np.bincount(cell, minlength=int(dims.prod())).sum() == 5000
    cx = cell % dims[0]
    cy = (cell // dims[0]) % dims[1]
    cz = cell // (dims[0] * dims[1])
    for a, c in enumerate((cx, cy, cz)):
        w = box[a] / dims[a]
        lo = -0.5 * box[a] + c * w
        assert w >= r_list
        assert np.all(pos[:, a] >= lo - 1e-12) and np.all(pos[:, a] < lo + w + 1e-12)


def test_cell_edges_and_faces():
    box = np.array([12.0, 12.0, 12.0])       # r_list 3 -> 4 cells of width 3: faces at -6,-3,0,3
    x = np.array([-6.0, np.nextafter(-3.0, -10), -3.0, 0.0, -1e-15, 3.0, np.nextafter(6.0, 0.0)])
    pos = np.zeros((len(x), 3)); pos[:, 0] = x; pos[:, 1] = -6.0; pos[:, 2] = np.nextafter(6.0, 0.0)
    cell, dims = oracle.cell_assign(pos, box, 3.0)
    assert list(dims) == [4, 4, 4]
    assert list(cell % 4) == [0, 0, 1, 2, 1, 3, 3]         # a face belongs to the upper cell; top edge clamps
    # (x = -1e-15 is the closest double below the face whose offset x - lo is still < 6: the IEEE expression decides)
    assert np.all((cell // 4) % 4 == 0) and np.all(cell // 16 == 3)


def test_cell_grid_never_finer_than_r_list():
    for L, rl in ((16.795962, 2.9), (107.494156, 3.4), (69.336127, 1.4), (75.282882, 1.4), (423.25824, 2.9)):
        d = oracle.cell_dims(np.array([L, L, L]), rl)
        assert L / d[0] >= rl and L / (d[0] + 1) < rl
    # the derived sizes of SURVEY.md 8: 5, 31, 49, 53, 145 cells per dimension
    assert [int(oracle.cell_dims(np.array([L] * 3), rl)[0]) for L, rl in
            ((16.795962, 2.9), (107.494156, 3.4), (69.336127, 1.4), (75.282882, 1.4), (423.25824, 2.9))] == [5, 31, 49, 53, 145]


def test_rebuild_trigger_free_flight_closed_form():
    """One particle moving with speed v along x crosses r_buff/2 after ceil-like n* steps: |n dt v| > r_buff/2."""
    box = np.array([10.0, 10.0, 10.0])
    ref = inputs.random_box(50, box, 3)
    r_buff, dt, v = 0.4, 0.005, 1.7
    first = None
    for n in range(1, 60):
        pos = ref.copy()
        pos[7, 0] += n * dt * v
        pos = inputs.wrap(pos, box)
        if oracle.needs_rebuild(pos, ref, box, r_buff):
            first = n
            break
    assert first == int(np.floor(0.5 * r_buff / (dt * v))) + 1 == 24
    # exactly at the threshold: not "more than half" -> no rebuild (strict >)
    pos = ref.copy(); pos[:, :] = 0.0; ref0 = pos.copy(); pos[3, 2] = 0.2
    assert (0.2 * 0.2) == (0.5 * 0.4) ** 2
    assert not oracle.needs_rebuild(pos, ref0, box, 0.4)
    pos[3, 2] = np.nextafter(0.2, 1.0)
    assert oracle.needs_rebuild(pos, ref0, box, 0.4)
    # displacement is minimum-imaged: a wrap through the face is not a jump of L
    ref1 = np.zeros((1, 3)); ref1[0, 0] = 4.95
    pos1 = np.zeros((1, 3)); pos1[0, 0] = -4.95
    assert not oracle.needs_rebuild(pos1, ref1, box, 0.4)


def test_list_superset_property_between_rebuilds():
    """rebuilding when a particle moved > r_buff/2 'guarantees correct force computations':
    every pair within rc at any step since the last build is in that build's list."""
    w = inputs.lj_fcc(4, rc=2.0, r_buff=0.4, kT=2.0, vel_seed=4, jitter=0.05, pos_seed=9)   # N=256, L=6.72 > 3*2.4? no
    box = w.box * 1.1                                                                       # L = 7.39 >= 7.2
    sim = oracle.Sim(w.pos * 1.1, w.vel, box, 2.0, 0.4, {"lj": {}})
    listed = set(map(tuple, oracle.neighbor_pairs(sim.pos, box, 2.4)))
    n_rebuild = 0
    for _ in range(60):
        before = len(sim.rebuild_steps)
        sim.run(1, 0.005)
        if len(sim.rebuild_steps) > before:
            listed = set(map(tuple, oracle.neighbor_pairs(sim.pos, box, 2.4)))
            n_rebuild += 1
        within = set(map(tuple, oracle.neighbor_pairs(sim.pos, box, 2.0)))
        assert within <= listed
    assert n_rebuild >= 2
