"""GPU-vs-oracle parity through the C-ABI (python -m pytest tests -m gpu).

Bars (BASELINE.json:north_star): cell ids and neighbour lists (as sorted tag pairs) bit-exact; per-particle forces
max relative error 1e-10 (fp64) / 1e-4 (mixed), norm of DESIGN.md R11; single-step positions 1e-12 (fp64).
"""
import numpy as np
import pytest

import oracle
from paper_1412_3387_b200 import binding as B
from paper_1412_3387_b200 import inputs
from gpu_util import sort_pairs, force_rel_err, min_image_diff

pytestmark = pytest.mark.gpu

ORDERS = [B.MD_ORDER_LEX, B.MD_ORDER_MORTON, B.MD_ORDER_HILBERT]


def _thermalised_lj(n_cells, rc=2.5, jitter=0.08, seed=3, kT=1.0):
    return inputs.lj_fcc(n_cells, rc=rc, r_buff=0.4, kT=kT, jitter=jitter, pos_seed=seed, vel_seed=seed + 1)


# ---------------------------------------------------------------------------------------------------- hash
def test_device_philox_equals_oracle_and_kat():
    md = B.MD([9, 9, 9], 10, 1.0, 0.4)
    rng = np.random.default_rng(0)
    ctr = rng.integers(0, 2 ** 32, size=(4096, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, size=(4096, 2), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0; key[0] = 0
    ctr[1] = 0xFFFFFFFF; key[1] = 0xFFFFFFFF
    ctr[2] = [0x243F6A88, 0x85A308D3, 0x13198A2E, 0x03707344]; key[2] = [0xA4093822, 0x299F31D0]
    out = md.debug_philox(ctr, key)
    assert [hex(x) for x in out[0]] == ["0x6627e8d5", "0xe169c58d", "0xbc57ac4c", "0x9b00dbd8"]
    assert [hex(x) for x in out[2]] == ["0xd16cfe09", "0x94fdcceb", "0x5001e420", "0x24126ea1"]
    ref = np.stack([oracle.philox4x32_10(c, k) for c, k in zip(ctr[:512], key[:512])])
    assert np.array_equal(out[:512], ref)


# ---------------------------------------------------------------------------------------------------- state
def test_state_roundtrip_wrap_and_errors():
    box = np.array([9.0, 10.0, 11.0])
    pos = inputs.random_box(1000, box, 1) + np.array([9.0, -20.0, 0.0])   # outside the box: wrapped on input
    vel = np.random.default_rng(2).standard_normal((1000, 3))
    md = B.MD(box, 1000, 2.5, 0.4)
    with pytest.raises(B.MDError):
        md.build_cells()                                                  # MD_ESTATE before set_state
    md.set_state(pos, vel)
    for order_dependent in (False, True):
        if order_dependent:
            md.build_cells()                                              # internal reorder must be invisible
        p, v, im = md.get_state()
        assert np.array_equal(p, oracle.wrap(pos, box))
        assert np.array_equal(v, vel) and not im.any()
    with pytest.raises(B.MDError):
        md.get_forces()
    with pytest.raises(B.MDError):
        B.MD([5.0, 5.0, 5.0], 10, 2.5, 0.4)                               # floor(5/2.9) = 1 < 3 cells


def test_device_and_host_pointers_agree():
    import torch
    w = _thermalised_lj(6)
    md = B.MD(w.box, w.N, w.rc, w.r_buff)
    md.set_state(torch.from_numpy(w.pos).cuda(), torch.from_numpy(w.vel).cuda())
    md.build_nlist(); md.forces_lj()
    F_dev = torch.empty((w.N, 3), dtype=torch.float64, device="cuda")
    md.get_forces(F_dev, None)
    md2 = B.from_workload(w)
    md2.build_nlist(); md2.forces_lj()
    F_host, _ = md2.get_forces()
    assert np.array_equal(F_dev.cpu().numpy(), F_host)


# ---------------------------------------------------------------------------------------------------- S1 cells
@pytest.mark.parametrize("order", ORDERS)
@pytest.mark.parametrize("N,box,r_list", [(3000, (9.0, 9.0, 9.0), 2.9), (5000, (16.795962, 13.1, 9.0), 2.9),
                                          (20000, (30.0, 7.0, 11.0), 1.4)])
def test_cells_bit_exact(order, N, box, r_list):
    box = np.array(box)
    pos = inputs.random_box(N, box, 5)
    md = B.MD(box, N, r_list - 0.4, 0.4, order=order)
    md.set_state(pos, np.zeros_like(pos))
    md.build_cells()
    cell, dims = md.get_cells()
    ref, rdims = oracle.cell_assign(pos, box, r_list)
    assert np.array_equal(dims, rdims)
    assert np.array_equal(cell, ref)


def test_cells_exact_faces():
    box = np.array([12.0, 12.0, 12.0])
    faces = np.array([-6.0, -3.0, 0.0, 3.0])
    x = np.concatenate([faces, np.nextafter(faces, -10), np.nextafter(faces, 10), [np.nextafter(6.0, 0)], faces - 1e-15])
    g = np.stack(np.meshgrid(x, x[:5], x[-5:], indexing="ij"), -1).reshape(-1, 3)
    g = oracle.wrap(g, box)
    md = B.MD(box, len(g), 2.6, 0.4)
    md.set_state(g, np.zeros_like(g)); md.build_cells()
    cell, _ = md.get_cells()
    assert np.array_equal(cell, oracle.cell_assign(g, box, 3.0)[0])


def test_cells_config1():
    w = inputs.config(1)
    md = B.from_workload(w); md.build_cells()
    cell, dims = md.get_cells()
    ref, rd = oracle.cell_assign(w.pos, w.box, w.r_list)
    assert list(dims) == [5, 5, 5] and np.array_equal(cell, ref)


# ---------------------------------------------------------------------------------------------------- S2 nlist
@pytest.mark.parametrize("order", ORDERS)
@pytest.mark.parametrize("N,box,r_list,seed", [
    (300, (9.0, 9.0, 9.0), 2.9, 1),          # 3x3x3 cells: every stencil wraps
    (777, (4.3, 5.7, 6.7), 1.4, 2),          # orthorhombic 3x4x4, ragged N
    (2000, (13.0, 13.0, 13.0), 3.4, 3),
])
def test_nlist_bit_exact_tiny_boxes(order, N, box, r_list, seed):
    box = np.array(box)
    pos = inputs.random_box(N, box, seed)
    md = B.MD(box, N, r_list - 0.4, 0.4, order=order)
    md.set_state(pos, np.zeros_like(pos))
    md.build_nlist()
    got = sort_pairs(md.get_nlist())
    ref = oracle.neighbor_pairs(pos, box, r_list)
    assert got.shape == ref.shape and np.array_equal(got, ref)
    st = md.stats()
    assert st["rebuilds"] == 1 and st["nlist_entries"] >= 2 * len(ref)


@pytest.mark.parametrize("w,block", [(1, 32), (2, 64), (4, 96), (8, 128), (16, 256), (32, 1024), (32, 32)])
def test_nlist_every_w_and_block(w, block):
    wl = _thermalised_lj(6)                                         # N=864
    md = B.from_workload(wl)
    md.set_launch(B.MD_K_NLIST, block, w)
    md.build_nlist()
    assert np.array_equal(sort_pairs(md.get_nlist()), oracle.neighbor_pairs(wl.pos, wl.box, wl.r_list))


def test_nlist_config1_fcc_shells_and_rows():
    w = inputs.config(1)
    md = B.from_workload(w); md.build_nlist()
    got = sort_pairs(md.get_nlist())
    assert got.shape[0] == 39 * w.N                                 # 78 neighbours each (FCC shells within 2.9)
    assert np.array_equal(got, oracle.neighbor_pairs(w.pos, w.box, w.r_list))
    pr = inputs.probe_tags(w.N, 97, seed=3)
    counts, nbrs = md.get_nlist_rows(pr, row_stride=128)
    rc, rn = oracle.probe_nlist(w.pos, w.box, w.r_list, pr, row_stride=128)
    assert np.array_equal(counts, rc) and (counts == 78).all()
    assert np.array_equal(np.sort(nbrs, axis=1), np.sort(rn, axis=1))


def test_nlist_invariants_and_dense_cell():
    # a clump of 200 particles inside one cell (cell population > 32 exercises the large-cell sort path)
    box = np.array([9.0, 9.0, 9.0])
    rng = np.random.default_rng(4)
    pos = np.concatenate([inputs.random_box(500, box, 9), rng.uniform(-0.3, 0.3, size=(200, 3))])
    md = B.MD(box, len(pos), 2.5, 0.4)
    md.set_state(pos, np.zeros_like(pos)); md.build_nlist()
    got = sort_pairs(md.get_nlist())
    assert np.array_equal(got, oracle.neighbor_pairs(pos, box, 2.9))
    assert md.stats()["max_cell_count"] >= 200
    counts, nbrs = md.get_nlist_rows(np.arange(len(pos), dtype=np.uint32), row_stride=700)
    deg = np.bincount(got.reshape(-1), minlength=len(pos))
    assert np.array_equal(counts, deg)                              # double-sided: row length = degree
    for i in (0, 13, 650):
        row = nbrs[i, :counts[i]]
        assert i not in row and len(np.unique(row)) == len(row)    # no self, no duplicates


# ---------------------------------------------------------------------------------------------------- S4a LJ
@pytest.mark.parametrize("w,block", [(1, 64), (2, 128), (4, 128), (8, 128), (32, 256)])
def test_lj_forces_fp64(w, block):
    wl = _thermalised_lj(6)                                         # N=864
    md = B.from_workload(wl)
    md.set_launch(B.MD_K_LJ, block, w)
    md.build_nlist(); md.forces_lj(1.0, 1.0, 1)
    # the row layout follows w (rotation 0/2/4/6 for w = 2): the exported list is the same list
    assert np.array_equal(sort_pairs(md.get_nlist()), oracle.neighbor_pairs(wl.pos, wl.box, wl.r_list))
    F, E = md.get_forces()
    Fr, Er = oracle.forces_lj(wl.pos, wl.box, wl.rc, 1.0, 1.0, 1)
    assert force_rel_err(F, Fr) < 1e-10
    assert np.abs(E - Er).max() < 1e-11 * np.abs(Er).max()
    assert np.abs(F.sum(axis=0)).max() < 1e-10 * np.abs(F).sum()   # Newton's third law


def test_lj_forces_params_and_unshifted():
    wl = _thermalised_lj(5, rc=2.0)
    box = wl.box * 1.2
    md = B.MD(box, wl.N, 2.0 * 1.1, 0.4)
    md.set_state(wl.pos * 1.2, wl.vel); md.build_nlist(); md.forces_lj(0.7, 1.1, 0)
    F, E = md.get_forces()
    Fr, Er = oracle.forces_lj(oracle.wrap(wl.pos * 1.2, box), box, 2.2, 0.7, 1.1, 0)
    assert force_rel_err(F, Fr) < 1e-10 and np.abs(E - Er).max() < 1e-11 * np.abs(Er).max()


def test_lj_forces_mixed_1e4():
    wl = inputs.lj_fcc(7, rc=3.0, r_buff=0.4, kT=1.2, jitter=0.05, pos_seed=2, vel_seed=3)   # config-2 recipe, N=1372
    md = B.from_workload(wl, precision=B.MD_MIXED)
    md.build_nlist(); md.forces_lj()
    F, E = md.get_forces()
    Fr, Er = oracle.forces_lj(wl.pos, wl.box, 3.0)
    err = force_rel_err(F, Fr)
    assert err < 1e-4
    assert err > 1e-9                                               # it really is the fp32 path
    assert np.abs(E - Er).max() < 1e-4 * np.abs(Er).max()


def test_lj_perfect_fcc_energy():
    w = inputs.config(1)
    md = B.from_workload(w); md.build_nlist(); md.forces_lj()
    F, E = md.get_forces()
    assert np.abs(E - (-6.332811992581)).max() < 1e-10 and np.abs(F).max() < 1e-10


# ---------------------------------------------------------------------------------------------------- S4b DPD
@pytest.mark.parametrize("w", [1, 2, 4, 32])
def test_dpd_forces(w):
    wl = inputs.dpd_fluid(3000, pos_seed=4, vel_seed=5)             # L=10: 7^3 cells of width 1.43
    p = wl.params
    md = B.from_workload(wl)
    md.set_launch(B.MD_K_DPD, 128, w)
    md.build_nlist()
    for step in (0, 7, 2 ** 33 + 5):
        md.forces_dpd(p["A"], p["gamma"], p["kT"], wl.dt, step, p["seed"])
        F, _ = md.get_forces()
        Fr = oracle.forces_dpd(wl.pos, wl.vel, wl.box, wl.rc, p["A"], p["gamma"], p["kT"], wl.dt, step, p["seed"])
        assert force_rel_err(F, Fr) < 1e-10
    assert np.abs(F.sum(axis=0)).max() < 1e-10 * np.abs(F).sum()


# ---------------------------------------------------------------------------------------------------- S5 bonds
def test_bond_forces_accumulate():
    wl = inputs.polymer_melt(40, chain_len=32, start_seed=6, walk_seed=7, vel_seed=8)   # N=1280, L=7.5
    p = wl.params
    md = B.from_workload(wl)
    md.build_nlist()
    md.forces_dpd(p["A"], p["gamma"], p["kT"], wl.dt, 3, p["seed"])
    md.forces_bonds(p["bond_k"], p["bond_r0"])
    F, E = md.get_forces()
    Fr = oracle.forces_dpd(wl.pos, wl.vel, wl.box, wl.rc, p["A"], p["gamma"], p["kT"], wl.dt, 3, p["seed"])
    Fb, Eb = oracle.forces_bonds(wl.pos, wl.box, wl.bonds, p["bond_k"], p["bond_r0"])
    assert force_rel_err(F, Fr + Fb) < 1e-10
    # bonds alone (no pair term): branched topology, several bonds per particle
    rng = np.random.default_rng(1)
    extra = np.stack([rng.integers(0, wl.N, 500), rng.integers(0, wl.N, 500)], 1)
    extra = extra[extra[:, 0] != extra[:, 1]].astype(np.uint32)
    bonds = np.concatenate([wl.bonds, extra])
    md.set_bonds(bonds)
    md.set_state(wl.pos, wl.vel); md.build_cells()
    md.forces_bonds(100.0, 1.0)
    F2, E2 = md.get_forces()
    Fb2, Eb2 = oracle.forces_bonds(wl.pos, wl.box, bonds, 100.0, 1.0)
    assert force_rel_err(F2, Fb2) < 1e-10 and np.abs(E2 - Eb2).max() < 1e-10 * np.abs(Eb2).max()


# ---------------------------------------------------------------------------------------------------- S6/S3/S7
def test_single_step_positions_1e12_and_trajectory():
    wl = _thermalised_lj(6, kT=1.5)
    desc = B.step_desc("lj", wl.dt, wl.params)
    md = B.from_workload(wl)
    sim = oracle.Sim(wl.pos, wl.vel, wl.box, wl.rc, wl.r_buff, {"lj": wl.params})
    md.step(desc, 1); sim.run(1, wl.dt)
    p, v, im = md.get_state()
    assert np.abs(min_image_diff(p, sim.pos, wl.box)).max() < 1e-12
    assert np.abs(v - sim.vel).max() < 1e-12
    md.step(desc, 59); sim.run(59, wl.dt)
    p, v, im = md.get_state()
    assert np.abs(min_image_diff(p, sim.pos, wl.box)).max() < 1e-9       # chaotic growth of rounding differences
    assert np.array_equal(im, sim.image)
    st = md.stats()
    assert st["steps"] == 60 and st["dangerous_builds"] == 0
    assert st["rebuilds"] == 1 + len(sim.rebuild_steps) and len(sim.rebuild_steps) >= 2


def test_manual_sequence_equals_md_step_and_rebuild_flag():
    wl = _thermalised_lj(6, kT=2.0)
    desc = B.step_desc("lj", wl.dt, wl.params)
    a = B.from_workload(wl); b = B.from_workload(wl)
    a.step(desc, 25)
    b.build_nlist(); b.forces_lj()
    sim = oracle.Sim(wl.pos, wl.vel, wl.box, wl.rc, wl.r_buff, {"lj": wl.params})
    flagged = []
    for s in range(25):
        b.integrate_nve(wl.dt, 1)
        if b.needs_rebuild():
            flagged.append(s + 1)
            b.build_cells(); b.build_nlist()
        b.forces_lj()
        b.integrate_nve(wl.dt, 2)
    sim.run(25, wl.dt)
    pa, va, _ = a.get_state(); pb, vb, _ = b.get_state()
    assert np.array_equal(pa, pb) and np.array_equal(va, vb)             # same kernels, same order: bit-identical
    assert flagged == sim.rebuild_steps


@pytest.mark.parametrize("kind", ["lj", "dpd"])
def test_speculative_scheduler_equals_synchronous(kind):
    """MD_SCHED_SPECULATIVE (forces enqueued before the rebuild flag is known, discarded if a rebuild is due,
    half 2 + half 1 fused) gives bit-identical trajectories and the same rebuild steps as MD_SCHED_SYNC, also
    when md_step is called in pieces."""
    wl = _thermalised_lj(6, kT=2.0) if kind == "lj" else inputs.dpd_fluid(3000, pos_seed=4, vel_seed=5)
    desc = B.step_desc(kind, wl.dt, wl.params)
    a = B.from_workload(wl, sched=B.MD_SCHED_SYNC)
    b = B.from_workload(wl, sched=B.MD_SCHED_SPECULATIVE)
    c = B.from_workload(wl, sched=B.MD_SCHED_SPECULATIVE)
    a.step(desc, 40); b.step(desc, 40)
    for n in (1, 7, 2, 30):
        c.step(desc, n)
    pa, va, ia = a.get_state(); pb, vb, ib = b.get_state(); pc, vc, ic = c.get_state()
    assert np.array_equal(pa, pb) and np.array_equal(va, vb) and np.array_equal(ia, ib)
    assert np.array_equal(pa, pc) and np.array_equal(va, vc)
    sa, sb = a.stats(), b.stats()
    assert sa["rebuilds"] == sb["rebuilds"] >= 3 and sa["speculative_forces"] == 0
    assert sb["speculative_forces"] > 0 and sb["wasted_forces"] <= sb["rebuilds"]
    fa, _ = a.get_forces(); fb, _ = b.get_forces()
    assert np.array_equal(fa, fb)
    # MD_SCHED_BATCH: kernels of whole batches enqueued ahead, gated on the device-side flag; no host round trip per step
    d = B.from_workload(wl, sched=B.MD_SCHED_BATCH)
    e = B.from_workload(wl, sched=B.MD_SCHED_BATCH)
    d.step(desc, 40)
    for n in (1, 7, 2, 30):
        e.step(desc, n)
    for md in (d, e):
        p, v, i = md.get_state()
        assert np.array_equal(pa, p) and np.array_equal(va, v) and np.array_equal(ia, i)
        assert np.array_equal(md.get_forces()[0], fa)
        st = md.stats()
        assert st["rebuilds"] == sa["rebuilds"] and st["steps"] == 40 and st["dangerous_builds"] == 0


def test_free_flight_images_and_rebuild_step():
    box = np.array([9.0, 9.0, 9.0])
    pos = inputs.random_box(400, box, 1)
    vel = np.zeros_like(pos); vel[7] = [40.0, -35.0, 0.0]; vel[9] = [0.0, 0.0, 1.7]
    md = B.MD(box, 400, 2.5, 0.4)
    md.set_state(pos, vel)
    desc = B.step_desc("none", 0.005, {})
    md.step(desc, 200)
    p, v, im = md.get_state()
    assert np.abs((p + im * box) - (pos + 200 * 0.005 * vel)).max() < 1e-11
    assert im[7, 0] >= 4 and im[7, 1] <= -3


def test_dpd_and_polymer_trajectories():
    for wl in (inputs.dpd_fluid(2000, pos_seed=4, vel_seed=5), inputs.polymer_melt(40, chain_len=32)):
        kind = wl.kind
        desc = B.step_desc(kind, wl.dt, wl.params)
        md = B.from_workload(wl)
        what = {"dpd": dict(A=wl.params["A"], gamma=wl.params["gamma"], kT=wl.params["kT"], seed=wl.params["seed"])}
        if kind == "polymer":
            what["bonds"] = dict(k=wl.params["bond_k"], r0=wl.params["bond_r0"])
        sim = oracle.Sim(wl.pos, wl.vel, wl.box, wl.rc, wl.r_buff, what, bonds=wl.bonds)
        md.step(desc, 1); sim.run(1, wl.dt)
        p, v, _ = md.get_state()
        assert np.abs(min_image_diff(p, sim.pos, wl.box)).max() < 1e-12
        assert np.abs(v - sim.vel).max() < 1e-11
        md.step(desc, 19); sim.run(19, wl.dt)
        p, v, _ = md.get_state()
        assert np.abs(min_image_diff(p, sim.pos, wl.box)).max() < 1e-8
        assert md.stats()["rebuilds"] == 1 + len(sim.rebuild_steps)


def test_step0_enters_the_hash():
    wl = inputs.dpd_fluid(1500, pos_seed=4, vel_seed=5)
    desc = B.step_desc("dpd", wl.dt, wl.params)
    out = []
    for step0 in (0, 1000):
        md = B.MD(wl.box, wl.N, wl.rc, wl.r_buff)
        md.set_state(wl.pos, wl.vel, None, step0)
        md.step(desc, 3)
        out.append(md.get_state()[0])
    assert np.abs(out[0] - out[1]).max() > 1e-6
    p = wl.params
    sim = oracle.Sim(wl.pos, wl.vel, wl.box, wl.rc, wl.r_buff,
                     {"dpd": dict(A=p["A"], gamma=p["gamma"], kT=p["kT"], seed=p["seed"])}, step0=1000)
    sim.run(3, wl.dt)
    assert np.abs(min_image_diff(out[1], sim.pos, wl.box)).max() < 1e-11


def test_nve_energy_drift_gpu_config1():
    """Config 1 (N=4000, 100 steps fp64) + drift bound over 1000 steps (R23)."""
    w = inputs.config(1)
    desc = B.step_desc("lj", w.dt, w.params)
    md = B.from_workload(w)
    md.build_nlist(); md.forces_lj()
    def energy():
        _, v, _ = md.get_state(); _, E = md.get_forces()
        return 0.5 * (v * v).sum() + E.sum()
    e0 = energy()
    worst = 0.0
    for _ in range(10):
        md.step(desc, 100)
        worst = max(worst, abs(energy() - e0) / w.N)
    assert worst < 2e-3
    st = md.stats()
    assert st["dangerous_builds"] == 0 and 1000 / 25 <= st["rebuilds"] <= 1000 / 4


def test_thermo_reductions():
    """md_thermo (device reductions): kinetic and potential energy, momentum, temperature against
    plain sums over the read-back state and the oracle's per-particle energies; bit-reproducible."""
    wl = _thermalised_lj(6, kT=1.3)
    md = B.from_workload(wl)
    md.step(B.step_desc("lj", wl.dt, wl.params), 12)                # forces left by md_step: energies on demand
    t1 = md.thermo(); t2 = md.thermo()
    assert t1["kinetic"] == t2["kinetic"] and t1["potential"] == t2["potential"]
    pos, vel, _ = md.get_state()
    ke = 0.5 * np.sum(vel * vel)
    _, Er = oracle.forces_lj(pos, wl.box, wl.rc)
    assert abs(t1["kinetic"] - ke) < 1e-12 * ke
    assert abs(t1["potential"] - Er.sum()) < 1e-10 * abs(Er.sum())
    assert np.abs(t1["momentum"] - vel.sum(axis=0)).max() < 1e-11 * np.abs(vel).sum()
    assert abs(t1["temperature"] - 2.0 * ke / (3 * wl.N - 3)) < 1e-12
    # NVE: the total energy of the thermalised state stays put over the 12 steps (R23 bound, per particle)
    e0 = 0.5 * np.sum(wl.vel * wl.vel) + oracle.forces_lj(wl.pos, wl.box, wl.rc)[1].sum()
    assert abs(t1["kinetic"] + t1["potential"] - e0) / wl.N < 2e-3
    # polymer: DPD conservative energy + bond energy lanes are summed as well
    wp = inputs.polymer_melt(20, chain_len=32)
    mp = B.from_workload(wp)
    q = wp.params
    mp.build_nlist()
    mp.forces_dpd(q["A"], q["gamma"], q["kT"], wp.dt, 3, q["seed"])
    mp.forces_bonds(q["bond_k"], q["bond_r0"])
    _, E = mp.get_forces()
    tp = mp.thermo()
    assert abs(tp["potential"] - E.sum()) < 1e-12 * abs(E.sum())
    assert abs(tp["kinetic"] - 0.5 * np.sum(wp.vel * wp.vel)) < 1e-12 * tp["kinetic"]


def test_nvt_single_steps_and_trajectory():
    """Nose-Hoover NVT (R30): md_integrate_nvt half by half and md_step(MD_F_NVT) against the oracle."""
    wl = _thermalised_lj(6, kT=0.7)                                   # N = 864
    kT0, tau, dt = 1.2, 0.4, wl.dt
    # --- one step, half by half: positions 1e-12, thermostat variables to rounding
    md = B.from_workload(wl)
    md.build_nlist(); md.forces_lj()
    md.set_thermostat(0.05, -0.01)
    sim = oracle.Sim(wl.pos, wl.vel, wl.box, wl.rc, wl.r_buff, {"lj": wl.params}, nvt=dict(kT=kT0, tau=tau))
    sim.xi, sim.eta = 0.05, -0.01
    sim.compute_forces(dt, 0)
    md.integrate_nvt(dt, 1, kT0, tau)
    oracle.nvt_half1(sim.pos, sim.vel, sim.image, sim.force, sim.box, dt, sim.xi)
    xi1, eta1, _ = oracle.nvt_thermostat(sim.vel, dt, kT0, tau, sim.xi, sim.eta)
    pos, vel, img = md.get_state()
    assert np.abs(min_image_diff(pos, sim.pos, wl.box)).max() < 1e-12
    assert np.abs(vel - sim.vel).max() < 1e-12 and np.array_equal(img, sim.image)
    gxi, geta = md.get_thermostat()
    assert abs(gxi - xi1) < 1e-13 and abs(geta - eta1) < 1e-14
    if md.needs_rebuild():
        md.build_cells(); md.build_nlist()
    md.forces_lj()
    sim.xi, sim.eta = xi1, eta1
    sim.compute_forces(dt, 1)
    md.integrate_nvt(dt, 2, kT0, tau)
    oracle.nvt_half2(sim.vel, sim.force, dt, sim.xi)
    _, vel, _ = md.get_state()
    assert np.abs(vel - sim.vel).max() < 1e-11
    # --- md_step with the thermostat (fused half 2 + half 1, device-side K reduction), 40 steps with rebuilds
    md2 = B.from_workload(wl)
    md2.step(B.step_desc("lj", dt, wl.params, nvt=dict(kT=kT0, tau=tau)), 40)
    sim2 = oracle.Sim(wl.pos, wl.vel, wl.box, wl.rc, wl.r_buff, {"lj": wl.params}, nvt=dict(kT=kT0, tau=tau)).run(40, dt)
    pos, vel, _ = md2.get_state()
    assert np.abs(min_image_diff(pos, sim2.pos, wl.box)).max() < 1e-9     # Lyapunov growth from 1e-16 over 40 steps
    gxi, geta = md2.get_thermostat()
    assert abs(gxi - sim2.xi) < 1e-10 and abs(geta - sim2.eta) < 1e-10
    assert md2.stats()["rebuilds"] >= 2 and md2.stats()["dangerous_builds"] == 0
    # the thermostat heats the T = 0.35 liquid (0.7 equipartitioned with the lattice) towards 1.2: xi went negative
    assert sim2.xi < 0.0
    # --- the batch scheduler with the thermostat: bit-identical to the speculative one
    md3 = B.from_workload(wl, sched=B.MD_SCHED_BATCH)
    md3.step(B.step_desc("lj", dt, wl.params, nvt=dict(kT=kT0, tau=tau)), 40)
    p3, v3, _ = md3.get_state()
    assert np.array_equal(p3, pos) and np.array_equal(v3, vel) and md3.get_thermostat() == (gxi, geta)
    # --- thermostat off (xi = 0, tau huge) is NVE, bit for bit in the positions
    a = B.from_workload(wl); b = B.from_workload(wl)
    a.step(B.step_desc("lj", dt, wl.params), 10)
    b.step(B.step_desc("lj", dt, wl.params, nvt=dict(kT=kT0, tau=1e150)), 10)
    pa, va, _ = a.get_state(); pb, vb, _ = b.get_state()
    assert np.abs(min_image_diff(pa, pb, wl.box)).max() < 1e-13 and np.abs(va - vb).max() < 1e-13


def test_tuner_runs_and_keeps_results():
    wl = _thermalised_lj(8)                                             # N=2048
    desc = B.step_desc("lj", wl.dt, wl.params)
    md = B.from_workload(wl)
    md.tune(desc, False)
    st = md.stats()
    assert st["tuner_runs"] == 1 and st["launch"]["lj"]["us"] > 0 and st["launch"]["nlist"]["us"] > 0
    assert st["launch"]["lj"]["w"] in (1, 2, 4, 8, 16, 32) and st["launch"]["lj"]["block"] % 32 == 0
    md.build_nlist(); md.forces_lj()
    F, _ = md.get_forces()
    assert force_rel_err(F, oracle.forces_lj(wl.pos, wl.box, wl.rc)[0]) < 1e-10


# ---------------------------------------------------------------------------------------------------- tile path
@pytest.mark.parametrize("brick", [1, 2, 4])
def test_tile_bricks_lists_and_forces(brick):
    """MD_ORDER_MORTON tile kernels (staged stencil, 16-bit entries) for every brick size, odd and small grids."""
    # LJ, 5x5x5 cells (odd: partial bricks), fp64 and mixed
    wl = inputs.lj_fcc(9, rc=2.5, r_buff=0.4, kT=1.0, jitter=0.08, pos_seed=5, vel_seed=6)     # N=2916, L=15.1
    ref_pairs = oracle.neighbor_pairs(wl.pos, wl.box, wl.r_list)
    Fr, Er = oracle.forces_lj(wl.pos, wl.box, wl.rc)
    for prec, tol in ((B.MD_FP64, 1e-10), (B.MD_MIXED, 1e-4)):
        md = B.from_workload(wl, precision=prec)
        md.set_option(B.MD_OPT_TILE_BRICK, brick)
        md.set_state(wl.pos, wl.vel)
        md.build_nlist()
        assert np.array_equal(sort_pairs(md.get_nlist()), ref_pairs)
        md.forces_lj()
        F, E = md.get_forces()
        assert force_rel_err(F, Fr) < tol
        assert np.abs(E - Er).max() < tol * 10 * np.abs(Er).max()
    # DPD, 7x7x7 cells
    wd = inputs.dpd_fluid(3000, pos_seed=4, vel_seed=5)
    p = wd.params
    md = B.from_workload(wd)
    md.set_option(B.MD_OPT_TILE_BRICK, brick)
    md.set_state(wd.pos, wd.vel)
    md.build_nlist()
    assert np.array_equal(sort_pairs(md.get_nlist()), oracle.neighbor_pairs(wd.pos, wd.box, wd.r_list))
    md.forces_dpd(p["A"], p["gamma"], p["kT"], wd.dt, 11, p["seed"])
    F, _ = md.get_forces()
    Fd = oracle.forces_dpd(wd.pos, wd.vel, wd.box, wd.rc, p["A"], p["gamma"], p["kT"], wd.dt, 11, p["seed"])
    assert force_rel_err(F, Fd) < 1e-10


def test_tile_3x3x3_grid_every_image():
    """Smallest legal grid: the (B+2)^3 stencil of a brick wraps onto itself, every staged cell is an image."""
    box = np.array([9.0, 9.3, 10.0])
    pos = inputs.random_box(900, box, 12)
    for brick in (1, 2):
        for prec in (B.MD_FP64, B.MD_MIXED):
            md = B.MD(box, 900, 2.5, 0.4, precision=prec)
            md.set_option(B.MD_OPT_TILE_BRICK, brick)
            md.set_state(pos, np.zeros_like(pos)); md.build_nlist()
            assert np.array_equal(sort_pairs(md.get_nlist()), oracle.neighbor_pairs(pos, box, 2.9))
            md.forces_lj()
            F, _ = md.get_forces()
            assert force_rel_err(F, oracle.forces_lj(pos, box, 2.5)[0]) < (1e-10 if prec == B.MD_FP64 else 1e-4)


def test_mixed_accumulation_blocks_agree():
    wl = inputs.lj_fcc(7, rc=3.0, r_buff=0.4, kT=1.2, jitter=0.05, pos_seed=2, vel_seed=3)
    Fr, _ = oracle.forces_lj(wl.pos, wl.box, 3.0)
    errs = []
    for blk in (1, 8):
        md = B.from_workload(wl, precision=B.MD_MIXED)
        md.set_option(B.MD_OPT_ACC_BLOCK, blk)
        md.build_nlist(); md.forces_lj()
        errs.append(force_rel_err(md.get_forces()[0], Fr))
    assert max(errs) < 1e-4


def test_tile_guard_band_pairs_at_the_cutoff():
    """Pairs placed within 1e-7 of r_list and of rc (inside the fp32 guard band) take the exact fp64 decision.  The
    base configuration is a jittered lattice (a liquid-like force distribution), so the R11 norm applies as it stands:
    1e-10 in fp64, 1e-4 in mixed precision, for md_forces_lj and for the kernels md_step launches."""
    wl = inputs.lj_fcc(8, rc=2.5, r_buff=0.4, kT=1.0, jitter=0.05, pos_seed=11, vel_seed=12)     # N=2048, L=13.4
    pos, box = wl.pos.copy(), wl.box
    rng = np.random.default_rng(3)
    used = np.zeros(wl.N, dtype=bool)
    n_made = 0
    for i in rng.permutation(wl.N):
        if used[i]:
            continue
        d = pos - pos[i]
        d -= box * np.rint(d / box)
        r = np.sqrt((d * d).sum(1))
        target = 2.5 if n_made % 2 else 2.9
        cand = np.nonzero((np.abs(r - target) < 0.2) & ~used)[0]             # FCC shells at 2.375, 2.656, 2.909
        if len(cand) == 0:
            continue
        j = cand[0]
        # neighbours of i and j must stay put, or earlier pairs would move
        used[np.nonzero(r < 3.2)[0]] = True
        dj = pos - pos[j]; dj -= box * np.rint(dj / box)
        used[np.nonzero(np.sqrt((dj * dj).sum(1)) < 3.2)[0]] = True
        pos[j] = pos[i] + d[j] / r[j] * (target + rng.uniform(-1e-7, 1e-7))
        n_made += 1
    assert n_made >= 20
    pos = oracle.wrap(pos, box)
    ref_pairs = oracle.neighbor_pairs(pos, box, 2.9)
    Fr = oracle.forces_lj(pos, box, 2.5)[0]
    desc = B.step_desc("lj", 1e-300, wl.params)          # a step that moves nothing: the forces are those of `pos`
    for prec, bar in ((B.MD_FP64, 1e-10), (B.MD_MIXED, 1e-4)):
        md = B.MD(box, len(pos), 2.5, 0.4, precision=prec)
        md.set_state(pos, np.zeros_like(pos)); md.build_nlist()
        assert np.array_equal(sort_pairs(md.get_nlist()), ref_pairs)
        md.forces_lj()
        F, _ = md.get_forces()
        # a wrongly included / excluded pair at rc changes a force by |F(rc)| = 0.039: far above either bar
        assert force_rel_err(F, Fr) < bar
        # the kernels md_step launches (k_tile_lj3 / k_tile_lj3d, no energies): forces read back WITHOUT an energy buffer
        ms = B.MD(box, len(pos), 2.5, 0.4, precision=prec)
        ms.set_state(pos, np.zeros_like(pos))
        ms.step(desc, 1)
        Fs = np.empty_like(F); ms.get_forces(Fs, None)
        assert force_rel_err(Fs, Fr) < bar


def _step_forces(md, desc, n=1):
    """Forces left by md_step, read back without an energy buffer (so nothing is re-evaluated), and the state."""
    md.step(desc, n)
    F = np.empty((md.N, 3)); md.get_forces(F, None)
    pos, vel, _ = md.get_state()
    return F, pos, vel


def test_step_kernels_forces_against_oracle():
    """The kernels bench.py times (md_step: k_tile_lj3 with its near section and guard band, k_tile_lj3d) compared DIRECTLY with the oracle at the positions md_step left: no energy
    buffer is passed, so md_get_forces returns what the step's own kernel wrote."""
    wl = inputs.lj_fcc(9, rc=3.0, r_buff=0.4, kT=1.2, jitter=0.05, pos_seed=2, vel_seed=3)       # config-2 recipe, N=2916
    desc = B.step_desc("lj", wl.dt, wl.params)
    for prec, bar in ((B.MD_MIXED, 1e-4), (B.MD_FP64, 1e-10)):
        for w in (1, 2, 4, 8):
            md = B.from_workload(wl, precision=prec)
            md.set_state(wl.pos, wl.vel)
            md.set_launch(B.MD_K_LJ, 256, w)
            F, pos, _ = _step_forces(md, desc, 25)          # 25 steps: at least one displacement-triggered rebuild
            assert md.stats()["rebuilds"] >= 2
            Fr, _ = oracle.forces_lj(pos, wl.box, wl.rc)
            assert force_rel_err(F, Fr) < bar, (prec, w)
            # reading energies afterwards must not change the forces the next half-kick uses
            F2, E2 = md.get_forces()
            assert np.array_equal(F2, F)
            assert np.abs(E2 - oracle.forces_lj(pos, wl.box, wl.rc)[1]).max() < 10 * bar * np.abs(E2).max()


def test_mixed_precision_other_sigma_and_near_section():
    """sigma != 1: the near section of the rows is sized for the sigma md_step is called with (list rebuilt if it was
    built for a smaller one); md_forces_lj with yet another sigma goes through the generic kernel; both within 1e-4."""
    wl = inputs.lj_fcc(8, rc=2.5, r_buff=0.4, kT=1.0, jitter=0.05, pos_seed=5, vel_seed=6)
    box, pos = wl.box * 1.15, oracle.wrap(wl.pos * 1.15, wl.box * 1.15)
    for sigma in (1.15, 0.9):
        md = B.MD(box, wl.N, 2.5 * 1.15, 0.4, precision=B.MD_MIXED)
        md.set_state(pos, np.zeros_like(pos))
        md.build_nlist()                                    # built before any sigma is known (hint = 1)
        desc = B.step_desc("lj", 1e-300, dict(epsilon=0.8, sigma=sigma, energy_shift=1))
        F, p2, _ = _step_forces(md, desc)
        Fr, _ = oracle.forces_lj(p2, box, 2.5 * 1.15, 0.8, sigma, 1)
        assert force_rel_err(F, Fr) < 1e-4
        md.forces_lj(0.8, 1.3 * sigma, 1)
        Fg, _ = md.get_forces()
        assert force_rel_err(Fg, oracle.forces_lj(p2, box, 2.5 * 1.15, 0.8, 1.3 * sigma, 1)[0]) < 1e-4


def test_build_nlist_after_integration_rebins():
    """md_build_nlist alone after md_integrate_nve: the stale binning is redone, list bit-exact."""
    for prec in (B.MD_FP64, B.MD_MIXED):
        wl = _thermalised_lj(6, kT=3.0)
        md = B.from_workload(wl, precision=prec)
        md.build_nlist(); md.forces_lj()
        for _ in range(40):
            md.integrate_nve(wl.dt, 1)
            if md.needs_rebuild():
                break
            md.forces_lj()
            md.integrate_nve(wl.dt, 2)
        assert md.needs_rebuild()
        md.build_nlist()                                    # no md_build_cells before it
        pos, _, _ = md.get_state()
        assert np.array_equal(sort_pairs(md.get_nlist()), oracle.neighbor_pairs(pos, wl.box, wl.r_list))
        assert np.array_equal(md.get_cells()[0], oracle.cell_assign(pos, wl.box, wl.r_list)[0])
        assert not md.needs_rebuild()
        md.forces_lj()
        assert force_rel_err(md.get_forces()[0], oracle.forces_lj(pos, wl.box, wl.rc)[0]) < (1e-10 if prec == B.MD_FP64 else 1e-4)


def test_tuner_reports_launched_sizes_and_retunes():
    """md_tune sweeps every kernel family over launchable block sizes only; md_get_stats reports the launched (block, w);
    MD_OPT_RETUNE_PERIOD makes md_step re-scan after that many rebuilds; results unchanged."""
    wl = inputs.lj_fcc(10, rc=3.0, r_buff=0.4, kT=1.5, jitter=0.05, pos_seed=2, vel_seed=3)      # N=4000
    desc = B.step_desc("lj", wl.dt, wl.params)
    md = B.from_workload(wl, precision=B.MD_MIXED)
    md.tune(desc, False)
    st = md.stats()
    assert st["launch"]["lj"]["block"] <= 256 and st["launch"]["nlist"]["block"] <= 512      # compiled limits
    assert st["launch"]["integrate"]["block"] <= 256 and st["launch"]["lj"]["w"] <= 8
    for k in ("cells", "nlist", "lj", "integrate"):
        assert st["launch"][k]["us"] > 0, k
    assert st["rebuilds"] == 1                              # the tuner's replays are not rebuilds of the run
    md.set_launch(B.MD_K_LJ, 1024, 2)                       # a hand-set size above the limit is reported as launched
    assert md.stats()["launch"]["lj"]["block"] == 256
    md.set_option(B.MD_OPT_RETUNE_PERIOD, 2)
    ref = B.from_workload(wl, precision=B.MD_MIXED)
    ref.set_launch(B.MD_K_LJ, 256, 2)
    md.step(desc, 60); ref.step(desc, 60)
    assert md.stats()["tuner_runs"] >= 2 and md.stats()["rebuilds"] == ref.stats()["rebuilds"] >= 4
    pa, _, _ = md.get_state(); pb, _, _ = ref.get_state()
    assert np.abs(min_image_diff(pa, pb, wl.box)).max() < 1e-6   # same trajectory up to the summation order of other W


def test_caller_workspace_bit_identical_and_enomem():
    """md_workspace_bytes + md_set_workspace: every internal buffer carved from a torch tensor; results
    bit-identical to the cudaMalloc path for LJ mixed (tile list, exports) and the polymer melt; a workspace that is too
    small fails with MD_ENOMEM and names the missing bytes."""
    import torch
    for wl, prec in ((inputs.lj_fcc(9, rc=3.0, r_buff=0.4, kT=1.2, jitter=0.05, pos_seed=2, vel_seed=3), B.MD_MIXED),
                     (inputs.polymer_melt(40, chain_len=32), B.MD_FP64)):
        desc = B.step_desc(wl.kind, wl.dt, wl.params)
        a = B.from_workload(wl, precision=prec)
        need = B.workspace_bytes(wl.box, wl.N, wl.rc, wl.r_buff, prec)
        ws = torch.empty(need, dtype=torch.uint8, device="cuda")
        b = B.from_workload(wl, precision=prec, workspace=ws)
        c = B.from_workload(wl, precision=prec, workspace="torch")
        for md in (a, b, c):
            md.step(desc, 30)
        pa, va, _ = a.get_state()
        for md in (b, c):
            p, v, _ = md.get_state()
            assert np.array_equal(p, pa) and np.array_equal(v, va)
            assert np.array_equal(sort_pairs(md.get_nlist()), sort_pairs(a.get_nlist()))
            assert np.array_equal(md.get_forces()[0], a.get_forces()[0])
        st = b.stats()
        assert 0 < st["device_bytes"] <= need
        b.close(); c.close()
    small = torch.empty(1 << 16, dtype=torch.uint8, device="cuda")
    with pytest.raises(B.MDError, match="workspace too small"):
        B.from_workload(wl, workspace=small)
    md = B.MD(wl.box, wl.N, wl.rc, wl.r_buff)               # after md_configure the workspace can no longer be set
    assert md.L.md_set_workspace(md.h, small.data_ptr(), small.numel()) == -2


def test_tune_rbuff_keeps_the_state_and_the_trajectory():
    """md_tune_rbuff: bursts over candidate skins start from the same saved state; afterwards state,
    step counter and statistics are untouched, the chosen skin is one of the candidates and is reported, skins the box
    cannot hold are skipped, and the run that follows matches the oracle (forces never depend on the skin)."""
    wl = inputs.dpd_fluid(3000, pos_seed=4, vel_seed=5)                  # L = 10: at most r_list = 3.33
    desc = B.step_desc("dpd", wl.dt, wl.params)
    md = B.from_workload(wl)
    md.step(desc, 5)
    p0, v0, i0 = md.get_state()
    st0 = md.stats()
    cands = [0.2, 0.4, 0.6, 0.8, 5.0]                                    # 5.0: floor(10 / 6) = 1 cell -> skipped
    rb = md.tune_rbuff(desc, cands, 40)
    assert rb in cands[:4]
    p1, v1, i1 = md.get_state()
    assert np.array_equal(p0, p1) and np.array_equal(v0, v1) and np.array_equal(i0, i1)
    st1 = md.stats()
    assert st1["steps"] == st0["steps"] == 5 and st1["rebuilds"] == st0["rebuilds"] and st1["r_buff"] == rb
    assert st1["rbuff_tuned_tps"] > 0
    md.step(desc, 10)
    q = wl.params
    sim = oracle.Sim(wl.pos, wl.vel, wl.box, wl.rc, wl.r_buff,
                     {"dpd": dict(A=q["A"], gamma=q["gamma"], kT=q["kT"], seed=q["seed"])}).run(15, wl.dt)
    p2, _, _ = md.get_state()
    assert np.abs(min_image_diff(p2, sim.pos, wl.box)).max() < 1e-9
    # the list is the one of the chosen skin
    md.build_nlist()
    assert np.array_equal(sort_pairs(md.get_nlist()), oracle.neighbor_pairs(p2, wl.box, wl.rc + rb))
    # LJ mixed with the tile path and a torch workspace
    wj = inputs.lj_fcc(9, rc=3.0, r_buff=0.4, kT=1.2, jitter=0.05, pos_seed=2, vel_seed=3)
    mj = B.from_workload(wj, precision=B.MD_MIXED, workspace="torch")
    dj = B.step_desc("lj", wj.dt, wj.params)
    mj.step(dj, 3)
    a = mj.get_state()[0]
    rj = mj.tune_rbuff(dj, None, 30)
    assert 0.2 <= rj <= 0.8 and np.array_equal(a, mj.get_state()[0])
    F, pos, _ = _step_forces(mj, dj, 10)
    assert force_rel_err(F, oracle.forces_lj(pos, wj.box, wj.rc)[0]) < 1e-4
