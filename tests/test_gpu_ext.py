"""-m gpu parity of SURVEY 8(f) rows 1 and 3 against oracle/md_oracle_ext.c: Yukawa / Gaussian / Morse pair forces,
FENE bonds, harmonic angles, periodic dihedrals (forces and energies within 1e-10, R11 norm), virial tensor and pressure of every term
(1e-10 of the tensor's scale), through the single calls and through md_step."""
import math

import numpy as np
import pytest

import oracle
from paper_1412_3387_b200 import binding as B
from paper_1412_3387_b200 import inputs
from gpu_util import force_rel_err, min_image_diff

pytestmark = pytest.mark.gpu

PAIRS = [("yukawa", (2.0, 1.5)), ("gaussian", (3.0, 0.8)), ("morse", (1.7, 2.0, 1.0)), ("lj", (0.9, 1.05))]


def _chain_angles(n_chains, length):
    return np.array([[length * c + i, length * c + i + 1, length * c + i + 2]
                     for c in range(n_chains) for i in range(length - 2)], dtype=np.uint32)


def _chain_dihedrals(n_chains, length):
    return np.array([[length * c + i, length * c + i + 1, length * c + i + 2, length * c + i + 3]
                     for c in range(n_chains) for i in range(length - 3)], dtype=np.uint32)


@pytest.mark.parametrize("order", [B.MD_ORDER_MORTON, B.MD_ORDER_LEX])
@pytest.mark.parametrize("kind,p", PAIRS)
def test_pair_potentials_forces_energies_virial(kind, p, order):
    wl = inputs.lj_fcc(7, rc=2.5, r_buff=0.4, kT=1.0, jitter=0.08, pos_seed=3, vel_seed=4)       # N = 1372
    for w in (1, 4, 8):
        md = B.from_workload(wl, order=order)
        md.set_launch(B.MD_K_LJ, 128, w)
        md.build_nlist()
        md.forces_pair(kind, p, 1)
        F, E = md.get_forces()
        Fr, Er = oracle.pair_forces(wl.pos, wl.box, wl.rc, kind, p, 1)
        assert force_rel_err(F, Fr) < 1e-10 and np.abs(E - Er).max() < 1e-11 * np.abs(Er).max()
    desc = B.step_desc("pair", wl.dt, dict(pair_kind=kind, pair_p=p))
    pr = md.pressure(desc)
    W = oracle.virial_pair(wl.pos, wl.box, wl.rc, kind, p)
    assert np.abs(pr["virial"] - W).max() < 1e-10 * np.abs(W).max()
    assert abs(pr["pressure"] - oracle.pressure(wl.vel, wl.box, W)) < 1e-11 * abs(pr["pressure"])
    assert pr["virial"].tolist() == md.pressure(desc)["virial"].tolist()          # fixed summation order
    # md_step with the pair potential: single step 1e-12, then a short trajectory
    if kind != "lj":
        ms = B.from_workload(wl, order=order)
        ms.step(desc, 1)
        pos, vel, _ = ms.get_state()
        F1 = oracle.pair_forces(wl.pos, wl.box, wl.rc, kind, p, 1)[0]
        v = wl.vel + 0.5 * wl.dt * F1
        x = oracle.wrap(wl.pos + wl.dt * v, wl.box)
        assert np.abs(min_image_diff(pos, x, wl.box)).max() < 1e-12
        v2 = v + 0.5 * wl.dt * oracle.pair_forces(x, wl.box, wl.rc, kind, p, 1)[0]
        assert np.abs(vel - v2).max() < 1e-11


def test_fene_bonds_and_angles_forces_energy_virial_and_step():
    wl = inputs.polymer_melt(40, chain_len=32, start_seed=6, walk_seed=7, vel_seed=8)             # N = 1280, bond step 0.97
    ang = _chain_angles(40, 32)
    k_f, r0_f, k_a, th0 = 30.0, 1.5, 8.0, 2.0
    md = B.from_workload(wl)
    md.set_angles(ang)
    md.build_cells()
    # FENE + angles alone (accumulate onto zero)
    md.forces_fene(k_f, r0_f)
    md.forces_angles(k_a, th0)
    F, E = md.get_forces()
    Fr, Er, Wb = oracle.forces_bonds_kind(wl.pos, wl.box, wl.bonds, "fene", k_f, r0_f)
    Wa = np.zeros(6)
    oracle.forces_angles(wl.pos, wl.box, ang, k_a, th0, force=Fr, energy=Er, virial=Wa)
    assert force_rel_err(F, Fr) < 1e-10 and np.abs(E - Er).max() < 1e-11 * np.abs(Er).max()
    # virial of DPD + FENE + angles together
    q = wl.params
    prm = dict(q, bond_kind="fene", bond_k=k_f, bond_r0=r0_f, angle_k=k_a, angle_theta0=th0)
    desc = B.step_desc("polymer", wl.dt, prm)
    assert desc.flags == B.MD_F_DPD | B.MD_F_BONDS | B.MD_F_ANGLES and desc.bond_kind == 1
    pr = md.pressure(desc)
    Wd = oracle.virial_dpd(wl.pos, wl.vel, wl.box, wl.rc, q["A"], q["gamma"], q["kT"], wl.dt, 0, q["seed"])
    W = Wd + Wb + Wa
    assert np.abs(pr["virial"] - W).max() < 1e-10 * np.abs(W).max()
    assert abs(pr["kinetic"] - 0.5 * (wl.vel ** 2).sum()) < 1e-12 * pr["kinetic"]
    assert abs(pr["pressure"] - oracle.pressure(wl.vel, wl.box, W)) < 1e-10 * abs(pr["pressure"])
    # harmonic bonds virial (the configured polymer model)
    pr_h = md.pressure(B.step_desc("polymer", wl.dt, q))
    Wh = oracle.forces_bonds_kind(wl.pos, wl.box, wl.bonds, "harmonic", q["bond_k"], q["bond_r0"])[2]
    assert np.abs(pr_h["virial"] - (Wd + Wh)).max() < 1e-10 * np.abs(Wd + Wh).max()
    # one md_step with DPD + FENE + angles against the plain sequence of oracle calls
    ms = B.from_workload(wl)
    ms.set_angles(ang)
    ms.step(desc, 1)
    pos, vel, _ = ms.get_state()

    def total_force(x, v, step):
        Ft = oracle.forces_dpd(x, v, wl.box, wl.rc, q["A"], q["gamma"], q["kT"], wl.dt, step, q["seed"])
        oracle.forces_bonds_kind(x, wl.box, wl.bonds, "fene", k_f, r0_f, force=Ft)
        oracle.forces_angles(x, wl.box, ang, k_a, th0, force=Ft)
        return Ft
    v = wl.vel + 0.5 * wl.dt * total_force(wl.pos, wl.vel, 0)
    x = oracle.wrap(wl.pos + wl.dt * v, wl.box)
    assert np.abs(min_image_diff(pos, x, wl.box)).max() < 1e-12
    v2 = v + 0.5 * wl.dt * total_force(x, v, 1)
    assert np.abs(vel - v2).max() < 1e-10
    # clearing the angles switches the term off
    ms.set_angles(None)
    ms.set_state(wl.pos, wl.vel)                       # (forces are accumulated: start from a cleared force array)
    ms.build_cells(); ms.forces_angles(k_a, th0)
    assert np.abs(ms.get_forces()[0]).max() == 0.0


def test_lj_and_dpd_pressure_at_scale_and_after_steps():
    """Pressure of the LJ liquid (mixed-precision context: the virial is fp64 either way) after md_step, list valid but
    not fresh, against the oracle at the same positions; ideal-gas limit with the forces off."""
    wl = inputs.lj_fcc(8, rc=3.0, r_buff=0.4, kT=1.2, jitter=0.05, pos_seed=2, vel_seed=3)       # N = 2048
    desc = B.step_desc("lj", wl.dt, wl.params)
    md = B.from_workload(wl, precision=B.MD_MIXED)
    md.step(desc, 7)
    pos, vel, _ = md.get_state()
    pr = md.pressure(desc)
    W = oracle.virial_pair(pos, wl.box, wl.rc, "lj", (1.0, 1.0))
    assert np.abs(pr["virial"] - W).max() < 1e-10 * np.abs(W).max()
    assert abs(pr["pressure"] - oracle.pressure(vel, wl.box, W)) < 1e-10 * abs(pr["pressure"])
    none = md.pressure(B.step_desc("none", wl.dt, {}))
    assert np.abs(none["virial"]).max() == 0.0
    assert abs(none["pressure"] - 2.0 * none["kinetic"] / (3.0 * none["volume"])) < 1e-15
    md.step(desc, 3)                                    # the pressure call left the run untouched
    ref = B.from_workload(wl, precision=B.MD_MIXED); ref.step(desc, 10)
    assert np.array_equal(md.get_state()[0], ref.get_state()[0])


@pytest.mark.parametrize("sign,n", [(1, 1), (-1, 2), (1, 3)])
def test_dihedrals_forces_energy_virial_and_step(sign, n):
    """R35 through the C-ABI: md_forces_dihedrals alone, its virial inside md_pressure, and one md_step of the polymer model
    with bonds + angles + dihedrals against the plain sequence of oracle calls."""
    wl = inputs.polymer_melt(40, chain_len=32, start_seed=16, walk_seed=17, vel_seed=18)          # N = 1280
    dih = _chain_dihedrals(40, 32)
    ang = _chain_angles(40, 32)
    k_d, k_a, th0 = 6.0, 8.0, 2.0
    md = B.from_workload(wl)
    md.set_dihedrals(dih)
    md.build_cells()
    md.forces_dihedrals(k_d, sign, n)
    F, E = md.get_forces()
    Fr, Er, Wr = oracle.forces_dihedrals(wl.pos, wl.box, dih, k_d, sign, n)
    assert np.abs(Fr).max() > 1.0                          # the term is really there
    assert force_rel_err(F, Fr) < 1e-10 and np.abs(E - Er).max() < 1e-11 * np.abs(Er).max()
    assert abs(F.sum(axis=0)).max() < 1e-10                # every quadruplet's four forces cancel
    # the dihedral virial alone, then together with DPD + harmonic bonds + angles
    d_only = B.step_desc("none", wl.dt, dict(dihedral_k=k_d, dihedral_sign=sign, dihedral_n=n))
    assert d_only.flags == B.MD_F_DIHEDRALS
    pr = md.pressure(d_only)
    assert np.abs(pr["virial"] - Wr).max() < 1e-10 * np.abs(Wr).max()
    q = wl.params
    prm = dict(q, angle_k=k_a, angle_theta0=th0, dihedral_k=k_d, dihedral_sign=sign, dihedral_n=n)
    desc = B.step_desc("polymer", wl.dt, prm)
    assert desc.flags == B.MD_F_DPD | B.MD_F_BONDS | B.MD_F_ANGLES | B.MD_F_DIHEDRALS
    md.set_angles(ang)
    pr = md.pressure(desc)
    Wd = oracle.virial_dpd(wl.pos, wl.vel, wl.box, wl.rc, q["A"], q["gamma"], q["kT"], wl.dt, 0, q["seed"])
    Wb = oracle.forces_bonds_kind(wl.pos, wl.box, wl.bonds, "harmonic", q["bond_k"], q["bond_r0"])[2]
    Wa = oracle.forces_angles(wl.pos, wl.box, ang, k_a, th0)[2]
    W = Wd + Wb + Wa + Wr
    assert np.abs(pr["virial"] - W).max() < 1e-10 * np.abs(W).max()
    # one md_step (batch scheduler, the default) and the same step with the synchronous scheduler
    outs = []
    for sched in (B.MD_SCHED_BATCH, B.MD_SCHED_SYNC):
        ms = B.from_workload(wl, sched=sched)
        ms.set_angles(ang)
        ms.set_dihedrals(dih)
        ms.step(desc, 1)
        outs.append(ms.get_state())
    pos, vel, _ = outs[0]
    assert np.array_equal(pos, outs[1][0]) and np.array_equal(vel, outs[1][1])

    def total_force(x, v, step):
        Ft = oracle.forces_dpd(x, v, wl.box, wl.rc, q["A"], q["gamma"], q["kT"], wl.dt, step, q["seed"])
        oracle.forces_bonds_kind(x, wl.box, wl.bonds, "harmonic", q["bond_k"], q["bond_r0"], force=Ft)
        oracle.forces_angles(x, wl.box, ang, k_a, th0, force=Ft)
        oracle.forces_dihedrals(x, wl.box, dih, k_d, sign, n, force=Ft)
        return Ft
    v = wl.vel + 0.5 * wl.dt * total_force(wl.pos, wl.vel, 0)
    x = oracle.wrap(wl.pos + wl.dt * v, wl.box)
    assert np.abs(min_image_diff(pos, x, wl.box)).max() < 1e-12
    v2 = v + 0.5 * wl.dt * total_force(x, v, 1)
    assert np.abs(vel - v2).max() < 1e-10


def test_dihedrals_argument_checks_and_clear():
    wl = inputs.polymer_melt(40, chain_len=8, start_seed=1, walk_seed=2, vel_seed=3)          # N = 320
    md = B.from_workload(wl)
    with pytest.raises(B.MDError):
        md.set_dihedrals(np.array([[0, 1, 2, wl.N]], dtype=np.uint32))         # tag out of range
    with pytest.raises(B.MDError):
        md.set_dihedrals(np.array([[0, 1, 2, 1]], dtype=np.uint32))            # repeated tag
    md.set_dihedrals(_chain_dihedrals(40, 8))
    md.build_cells()
    with pytest.raises(B.MDError):
        md.forces_dihedrals(1.0, 0, 1)                                         # sign must be +-1
    with pytest.raises(B.MDError):
        md.forces_dihedrals(1.0, 1, 0)                                         # n >= 1
    md.forces_dihedrals(2.0, 1, 1)
    assert np.abs(md.get_forces()[0]).max() > 0.0
    md.set_dihedrals(None)
    md.set_state(wl.pos, wl.vel)
    md.build_cells(); md.forces_dihedrals(2.0, 1, 1)
    assert np.abs(md.get_forces()[0]).max() == 0.0


def test_langevin_force_and_steps_against_the_oracle():
    """R36: md_forces_langevin on top of an LJ evaluation (same Philox words as the oracle: 1e-13), md_step with LJ +
    Langevin for 6 steps against oracle.Sim, every scheduler bit-identical, argument checks."""
    wl = inputs.lj_fcc(6, rc=2.5, r_buff=0.4, kT=1.0, jitter=0.06, pos_seed=9, vel_seed=10)      # N = 864
    g, kT, seed = 1.5, 1.3, (0xabcdef << 32) | 1234
    md = B.from_workload(wl)
    md.build_nlist()
    md.forces_lj(1.0, 1.0, 1)
    md.forces_langevin(g, kT, wl.dt, (1 << 33) + 7, seed)
    F, _ = md.get_forces()
    Fr = oracle.forces_lj(wl.pos, wl.box, wl.rc, 1.0, 1.0, 1)[0]
    FL = oracle.forces_langevin(wl.vel, g, kT, wl.dt, (1 << 33) + 7, seed)
    assert np.abs(FL).max() > 10.0
    assert force_rel_err(F, Fr + FL) < 1e-10
    # the thermostat term alone: identical words, identical operations
    md.set_state(wl.pos, wl.vel)
    md.build_cells()
    md.forces_langevin(g, kT, wl.dt, 3, seed)
    assert np.abs(md.get_forces()[0] - oracle.forces_langevin(wl.vel, g, kT, wl.dt, 3, seed)).max() < 1e-13
    prm = dict(wl.params, langevin=dict(gamma=g, kT=kT, seed=seed))
    desc = B.step_desc("lj", wl.dt, prm)
    assert desc.flags == B.MD_F_LJ | B.MD_F_LANGEVIN
    outs = []
    for sched in (B.MD_SCHED_BATCH, B.MD_SCHED_SPECULATIVE, B.MD_SCHED_SYNC):
        ms = B.from_workload(wl, sched=sched)
        ms.step(desc, 6)
        outs.append(ms.get_state())
    for o in outs[1:]:
        assert np.array_equal(o[0], outs[0][0]) and np.array_equal(o[1], outs[0][1])
    sim = oracle.Sim(wl.pos, wl.vel, wl.box, wl.rc, wl.r_buff,
                     {"lj": dict(epsilon=1.0, sigma=1.0, energy_shift=1), "langevin": dict(gamma=g, kT=kT, seed=seed)})
    sim.run(6, wl.dt)
    assert np.abs(min_image_diff(outs[0][0], sim.pos, wl.box)).max() < 1e-11
    assert np.abs(outs[0][1] - sim.vel).max() < 1e-10
    with pytest.raises(B.MDError):
        md.forces_langevin(-1.0, kT, wl.dt, 0, 0)
    with pytest.raises(B.MDError):
        md.forces_langevin(g, kT, 0.0, 0, 0)
    with pytest.raises(B.MDError):
        B.from_workload(wl).step(B.step_desc("lj", wl.dt, prm, nvt=dict(kT=1.0, tau=0.5)), 1)


def test_langevin_free_particles_closed_forms_on_the_device():
    """No other force: exact per-step decay of the velocities at kT = 0 and the stationary variance of the discrete scheme
    at kT > 0 (the closed forms the oracle is pinned with), over 4e5 particles."""
    N, box = 400000, 120.0
    rng = np.random.default_rng(11)
    pos = rng.uniform(0, box, size=(N, 3))
    v0 = rng.normal(size=(N, 3))
    dt, g = 0.01, 3.0
    a = g * dt
    md = B.MD(box, N, 1.0, 0.4)
    md.set_state(pos, v0)
    md.step(B.step_desc("none", dt, dict(langevin=dict(gamma=g, kT=0.0, seed=1))), 10)
    assert np.abs(md.get_state()[1] - v0 * (1 - a / 2) ** 2 * (1 - a) ** 9).max() < 1e-12
    kT, g, dt = 1.5, 5.0, 0.02
    a = g * dt
    md = B.MD(box, N, 1.0, 0.4)
    md.set_state(pos, np.zeros((N, 3)))
    md.step(B.step_desc("none", dt, dict(langevin=dict(gamma=g, kT=kT, seed=7))), 300)
    var_full = kT / (1 - a / 2) * (1 - a / 2) ** 2 + (dt / 2) ** 2 * (2 * g * kT / dt)
    v = md.get_state()[1]
    assert abs((v ** 2).mean() / var_full - 1.0) < 4.0 * math.sqrt(2.0 / (3 * N))
    assert np.abs(v.mean(axis=0)).max() < 4.0 * math.sqrt(var_full / N)


@pytest.mark.parametrize("order", [B.MD_ORDER_MORTON, B.MD_ORDER_LEX])
def test_tabulated_pair_potential_forces_energies_virial_and_step(order):
    """R37 through the C-ABI: a random table (forces and energies 1e-10 of the oracle's, same interpolation), a table of the
    LJ closed forms against the analytic LJ kernel at the interpolation error, virial, md_step, argument checks."""
    wl = inputs.lj_fcc(7, rc=2.5, r_buff=0.4, kT=1.0, jitter=0.08, pos_seed=13, vel_seed=14)      # N = 1372
    r_min, r_max, M = 0.7, 2.3, 257
    rng = np.random.default_rng(4)
    U, F = rng.normal(size=M), 5.0 * rng.normal(size=M)
    Fr, Er, Wr = oracle.pair_table(wl.pos, wl.box, r_min, r_max, U, F)
    for w in (1, 4, 8):
        md = B.from_workload(wl, order=order)
        md.set_launch(B.MD_K_LJ, 128, w)
        md.set_pair_table(r_min, r_max, U, F)
        md.build_nlist()
        md.forces_pair("table")
        Fo, E = md.get_forces()
        assert force_rel_err(Fo, Fr) < 1e-10 and np.abs(E - Er).max() < 1e-11 * np.abs(Er).max()
    desc = B.step_desc("pair", wl.dt, dict(pair_kind="table"))
    pr = md.pressure(desc)
    assert np.abs(pr["virial"] - Wr).max() < 1e-10 * np.abs(Wr).max()
    # LJ closed forms in a fine table: the analytic kernel within the interpolation error
    rk = np.linspace(0.8, wl.rc, 6801)
    md.set_pair_table(0.8, wl.rc, 4 * (rk ** -12 - rk ** -6), 24 * (2 * rk ** -13 - rk ** -7))
    md.forces_pair("table")
    Ft = md.get_forces()[0]
    md.forces_pair("lj", (1.0, 1.0), 0)
    assert np.abs(Ft - md.get_forces()[0]).max() < 2e-4
    # one md_step with the random table against the oracle sequence
    ms = B.from_workload(wl, order=order)
    ms.set_pair_table(r_min, r_max, U, F)
    ms.step(desc, 1)
    pos, vel, _ = ms.get_state()
    v = wl.vel + 0.5 * wl.dt * Fr
    x = oracle.wrap(wl.pos + wl.dt * v, wl.box)
    assert np.abs(min_image_diff(pos, x, wl.box)).max() < 1e-12
    v2 = v + 0.5 * wl.dt * oracle.pair_table(x, wl.box, r_min, r_max, U, F)[0]
    assert np.abs(vel - v2).max() < 1e-11
    # argument checks: r_max beyond the cut-off, one-point table, no table set
    with pytest.raises(B.MDError):
        ms.set_pair_table(0.5, wl.rc + 0.1, U, F)
    with pytest.raises(B.MDError):
        ms.set_pair_table(0.5, 2.0, U[:1], F[:1])
    ms.set_pair_table(0, 0, None, None)
    with pytest.raises(B.MDError):
        ms.forces_pair("table")
    with pytest.raises(B.MDError):
        ms.step(desc, 1)


def test_tabulated_bonds_forces_energy_virial_and_step():
    """R38 through the C-ABI: md_forces_bond_table with a random table (1e-10 of the oracle's, same interpolation), the table
    of the configured harmonic bond against md_forces_bonds, the virial with DPD, one md_step, NaN for a bond that left the
    table, argument checks."""
    wl = inputs.polymer_melt(40, chain_len=32, start_seed=26, walk_seed=27, vel_seed=28)          # N = 1280, bond step 0.97
    r_min, r_max, M = 0.3, 1.9, 129
    rng = np.random.default_rng(6)
    U, F = rng.normal(size=M), 8.0 * rng.normal(size=M)
    md = B.from_workload(wl)
    md.set_bond_table(r_min, r_max, U, F)
    md.build_cells()
    md.forces_bond_table()
    Fo, E = md.get_forces()
    Fr, Er, Wr = oracle.bond_table(wl.pos, wl.box, wl.bonds, r_min, r_max, U, F)
    assert np.isfinite(Fr).all() and np.abs(Fr).max() > 1.0
    assert force_rel_err(Fo, Fr) < 1e-10 and np.abs(E - Er).max() < 1e-11 * np.abs(Er).max()
    # the harmonic bond as a table: forces equal to the analytic kernel's to rounding
    q = wl.params
    rk = np.linspace(r_min, r_max, M)
    md.set_bond_table(r_min, r_max, 0.5 * q["bond_k"] * (rk - q["bond_r0"]) ** 2, -q["bond_k"] * (rk - q["bond_r0"]))
    md.set_state(wl.pos, wl.vel); md.build_cells(); md.forces_bond_table()
    Ft = md.get_forces()[0]
    md.set_state(wl.pos, wl.vel); md.build_cells(); md.forces_bonds(q["bond_k"], q["bond_r0"])
    assert np.abs(Ft - md.get_forces()[0]).max() < 1e-10
    # virial of DPD + tabulated bonds, then one md_step against the oracle sequence
    md.set_bond_table(r_min, r_max, U, F)
    desc = B.step_desc("polymer", wl.dt, dict(q, bond_kind="table"))
    assert desc.flags == B.MD_F_DPD | B.MD_F_BONDS and desc.bond_kind == 2
    pr = md.pressure(desc)
    Wd = oracle.virial_dpd(wl.pos, wl.vel, wl.box, wl.rc, q["A"], q["gamma"], q["kT"], wl.dt, 0, q["seed"])
    assert np.abs(pr["virial"] - (Wd + Wr)).max() < 1e-10 * np.abs(Wd + Wr).max()
    ms = B.from_workload(wl)
    ms.set_bond_table(r_min, r_max, U, F)
    ms.step(desc, 1)
    pos, vel, _ = ms.get_state()

    def total_force(x, v, step):
        Ft_ = oracle.forces_dpd(x, v, wl.box, wl.rc, q["A"], q["gamma"], q["kT"], wl.dt, step, q["seed"])
        oracle.bond_table(x, wl.box, wl.bonds, r_min, r_max, U, F, force=Ft_)
        return Ft_
    v = wl.vel + 0.5 * wl.dt * total_force(wl.pos, wl.vel, 0)
    x = oracle.wrap(wl.pos + wl.dt * v, wl.box)
    assert np.abs(min_image_diff(pos, x, wl.box)).max() < 1e-12
    assert np.abs(vel - (v + 0.5 * wl.dt * total_force(x, v, 1))).max() < 1e-10
    # a bond stretched beyond the table (chain end 0 pulled to 1.5 from its neighbour, table ends at 1.3): its two ends
    # are NaN, every other particle keeps its value, as in the oracle
    pos2 = wl.pos.copy()
    dvec = min_image_diff(pos2[0:1], pos2[1:2], wl.box)[0]
    pos2[0] = pos2[1] + 1.5 * dvec / np.linalg.norm(dvec)
    pos2 = oracle.wrap(pos2, wl.box)
    md.set_bond_table(r_min, 1.3, U, F)
    md.set_state(pos2, wl.vel); md.build_cells(); md.forces_bond_table()
    Fn = md.get_forces()[0]
    Fnr = oracle.bond_table(pos2, wl.box, wl.bonds, r_min, 1.3, U, F)[0]
    assert np.isnan(Fn[:2]).all() and np.isnan(Fnr[:2]).all() and np.isfinite(Fn[2:]).all()
    assert force_rel_err(Fn[2:], Fnr[2:]) < 1e-10
    # argument checks
    with pytest.raises(B.MDError):
        md.set_bond_table(1.0, 0.5, U, F)
    with pytest.raises(B.MDError):
        md.set_bond_table(0.5, 1.0, U[:1], F[:1])
    md.set_bond_table(0, 0, None, None)
    with pytest.raises(B.MDError):
        md.forces_bond_table()
    with pytest.raises(B.MDError):
        md.step(desc, 1)


def test_mtk_nvt_single_factors_steps_and_reversal():
    """Martyna-Tobias-Klein NVT (R39): md_mtk_thermostat_half + the NVE halves against the oracle's factors, md_step with
    MD_F_MTK against oracle.Sim over 40 steps with rebuilds, every scheduler bit-identical, the NVE limit, and the time
    reversal the factorisation guarantees, on the device."""
    wl = inputs.lj_fcc(6, rc=2.5, r_buff=0.4, kT=0.7, jitter=0.08, pos_seed=3, vel_seed=4)       # N = 864
    kT0, tau, dt = 1.2, 0.4, wl.dt
    nvt = dict(kT=kT0, tau=tau, scheme="mtk")
    # --- one step, factor by factor
    md = B.from_workload(wl)
    md.build_nlist(); md.forces_lj()
    md.set_thermostat(0.05, -0.01)
    sim = oracle.Sim(wl.pos, wl.vel, wl.box, wl.rc, wl.r_buff, {"lj": wl.params}, nvt=nvt)
    sim.xi, sim.eta = 0.05, -0.01
    sim.compute_forces(dt, 0)
    md.mtk_thermostat_half(dt, kT0, tau)
    sim.xi, sim.eta = oracle.mtk_thermostat_half(sim.vel, dt, kT0, tau, sim.xi, sim.eta)
    _, vel, _ = md.get_state()
    gxi, geta = md.get_thermostat()
    assert np.abs(vel - sim.vel).max() < 1e-13 and abs(gxi - sim.xi) < 1e-13 and abs(geta - sim.eta) < 1e-14
    assert abs(sim.xi - 0.05) > 1e-4                                  # the factor did something
    md.integrate_nve(dt, 1)
    oracle.vv_half1(sim.pos, sim.vel, sim.image, sim.force, sim.box, dt)
    if md.needs_rebuild():
        md.build_cells()
    md.build_nlist(); md.forces_lj()
    sim.compute_forces(dt, 1)
    md.integrate_nve(dt, 2)
    oracle.vv_half2(sim.vel, sim.force, dt)
    md.mtk_thermostat_half(dt, kT0, tau)
    sim.xi, sim.eta = oracle.mtk_thermostat_half(sim.vel, dt, kT0, tau, sim.xi, sim.eta)
    pos, vel, img = md.get_state()
    assert np.abs(min_image_diff(pos, sim.pos, wl.box)).max() < 1e-12 and np.array_equal(img, sim.image)
    assert np.abs(vel - sim.vel).max() < 1e-11
    gxi, geta = md.get_thermostat()
    assert abs(gxi - sim.xi) < 1e-12 and abs(geta - sim.eta) < 1e-13
    # --- md_step over 40 steps with rebuilds, the three schedulers
    desc = B.step_desc("lj", dt, wl.params, nvt=nvt)
    assert desc.flags == B.MD_F_LJ | B.MD_F_MTK
    sim2 = oracle.Sim(wl.pos, wl.vel, wl.box, wl.rc, wl.r_buff, {"lj": wl.params}, nvt=nvt).run(40, dt)
    outs = []
    for sched in (B.MD_SCHED_BATCH, B.MD_SCHED_SPECULATIVE, B.MD_SCHED_SYNC):
        m = B.from_workload(wl, sched=sched)
        m.step(desc, 17); m.step(desc, 23)                            # two calls: no merged factor across the boundary
        outs.append((m.get_state(), m.get_thermostat(), m.stats()))
    (pos, vel, _), (gxi, geta), st = outs[0]
    assert np.abs(min_image_diff(pos, sim2.pos, wl.box)).max() < 1e-9      # Lyapunov growth from 1e-16 over 40 steps
    assert np.abs(vel - sim2.vel).max() < 1e-8
    assert abs(gxi - sim2.xi) < 1e-10 and abs(geta - sim2.eta) < 1e-10 and sim2.xi < 0.0
    assert st["rebuilds"] >= 2 and st["dangerous_builds"] == 0
    for o in outs[1:]:
        assert np.array_equal(o[0][0], pos) and np.array_equal(o[0][1], vel) and o[1] == (gxi, geta)
    # --- thermostat off (tau huge): NVE
    a = B.from_workload(wl); b = B.from_workload(wl)
    a.step(B.step_desc("lj", dt, wl.params), 10)
    b.step(B.step_desc("lj", dt, wl.params, nvt=dict(kT=kT0, tau=1e150, scheme="mtk")), 10)
    pa, va, _ = a.get_state(); pb, vb, _ = b.get_state()
    assert np.abs(min_image_diff(pa, pb, wl.box)).max() < 1e-13 and np.abs(va - vb).max() < 1e-13
    # --- time reversal on the device: 30 steps forward, v and xi negated, 30 steps: back at the start
    r = B.from_workload(wl)
    r.step(desc, 30)
    p1, v1, _ = r.get_state()
    xi1, eta1 = r.get_thermostat()
    assert np.abs(min_image_diff(p1, wl.pos, wl.box)).max() > 0.05
    r.set_state(p1, -v1, None, 30)
    r.set_thermostat(-xi1, eta1)
    r.step(desc, 30)
    p2, v2, _ = r.get_state()
    xi2, eta2 = r.get_thermostat()
    assert np.abs(min_image_diff(p2, wl.pos, wl.box)).max() < 1e-10 and np.abs(v2 + wl.vel).max() < 1e-10
    assert abs(xi2) < 1e-11 and abs(eta2) < 1e-11
    # --- argument checks
    with pytest.raises(B.MDError):
        r.mtk_thermostat_half(dt, -1.0, tau)
    bad = B.step_desc("lj", dt, dict(wl.params, langevin=dict(gamma=1.0, kT=1.0, seed=1)), nvt=nvt)
    with pytest.raises(B.MDError):
        r.step(bad, 1)


def test_degenerate_and_empty_bonded_terms():
    """Collinear triplets and quadruplets are skipped on the device exactly as in the oracle (no force, no NaN), next to regular
    terms in the same call; empty term lists and particles without terms are no-ops."""
    wl = inputs.lj_fcc(6, rc=2.5, r_buff=0.4, kT=1.0, jitter=0.05, pos_seed=31, vel_seed=32)      # N = 864
    pos = wl.pos.copy()
    base = pos[10].copy()
    for k, x in enumerate((0.0, 1.0, 2.1)):                              # particles 10, 11, 12 on a line along x
        pos[10 + k] = base + [x, 0.0, 0.0]
    pos[13] = base + [3.0, 0.5, 0.0]
    pos = oracle.wrap(pos, wl.box)
    ang = np.array([[10, 11, 12], [11, 12, 13], [20, 21, 22], [12, 11, 10]], dtype=np.uint32)
    dih = np.array([[10, 11, 12, 13], [13, 12, 11, 10], [20, 21, 22, 23], [30, 40, 50, 60]], dtype=np.uint32)
    md = B.MD(wl.box, wl.N, wl.rc, wl.r_buff)
    md.set_state(pos, wl.vel)
    md.set_angles(ang); md.set_dihedrals(dih)
    md.build_cells()
    md.forces_angles(6.0, 1.9); md.forces_dihedrals(2.5, -1, 3)
    F, E = md.get_forces()
    Fr, Er, _ = oracle.forces_angles(pos, wl.box, ang, 6.0, 1.9)
    oracle.forces_dihedrals(pos, wl.box, dih, 2.5, -1, 3, force=Fr, energy=Er)
    assert np.isfinite(F).all() and np.isfinite(Fr).all()
    assert force_rel_err(F, Fr) < 1e-10 and np.abs(E - Er).max() < 1e-11 * np.abs(Er).max()
    assert np.abs(Fr[10]).max() == 0.0 and np.abs(F[10]).max() == 0.0    # 10 only takes part in skipped terms ...
    assert np.abs(F[13]).max() > 0.0                                     # ... 13 also in the regular angle (11, 12, 13)
    untouched = np.setdiff1d(np.arange(wl.N), np.unique(np.concatenate([ang.ravel(), dih.ravel()])))
    assert np.abs(F[untouched]).max() == 0.0
    pr = md.pressure(B.step_desc("none", wl.dt, dict(angle_k=6.0, angle_theta0=1.9, dihedral_k=2.5, dihedral_sign=-1, dihedral_n=3)))
    Wr = oracle.forces_angles(pos, wl.box, ang, 6.0, 1.9)[2] + oracle.forces_dihedrals(pos, wl.box, dih, 2.5, -1, 3)[2]
    assert np.isfinite(pr["virial"]).all() and np.abs(pr["virial"] - Wr).max() < 1e-10 * np.abs(Wr).max()
    # empty lists: the calls and the step flags are no-ops
    md.set_angles(None); md.set_dihedrals(None); md.set_bonds(None)
    md.set_state(pos, wl.vel); md.build_cells()
    md.forces_angles(6.0, 1.9); md.forces_dihedrals(2.5, -1, 3); md.forces_bonds(1.0, 1.0); md.forces_fene(1.0, 1.5)
    assert np.abs(md.get_forces()[0]).max() == 0.0
