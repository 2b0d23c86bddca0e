"""CPU oracle -- TEST INFRASTRUCTURE ONLY (see md_oracle.c header).

Thin ctypes access to oracle/liboracle.so plus the velocity-Verlet driver loop written in the order of
DESIGN.md "The path".  Imports nothing from the CUDA package; only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs may import this.
"""
from __future__ import annotations

import ctypes as C
import numpy as np

from . import build as _build

_lib = None

_dp = C.POINTER(C.c_double)
_u32p = C.POINTER(C.c_uint32)
_i32p = C.POINTER(C.c_int32)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.orc_neighbor_pairs.restype = C.c_uint64
        L.orc_needs_rebuild.restype = C.c_int
        L.orc_dpd_theta.restype = C.c_double
        L.orc_dpd_theta.argtypes = [C.c_uint32, C.c_uint32, C.c_uint64, C.c_uint64]
        _lib = L
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def _u(a):
    a = np.ascontiguousarray(a, dtype=np.uint32)
    return a, a.ctypes.data_as(_u32p)


def _box(box):
    b = np.ascontiguousarray(np.broadcast_to(np.asarray(box, dtype=np.float64), (3,)))
    return b, b.ctypes.data_as(_dp)


def wrap(pos, box, image=None):
    pos = np.array(pos, dtype=np.float64, order="C")
    b, bp = _box(box)
    ip = image.ctypes.data_as(_i32p) if image is not None else None
    lib().orc_wrap(pos.ctypes.data_as(_dp), ip, C.c_uint64(pos.shape[0]), bp)
    return pos


def cell_dims(box, r_list):
    b, bp = _box(box)
    dims = np.zeros(3, dtype=np.uint32)
    lib().orc_cell_dims(bp, C.c_double(r_list), dims.ctypes.data_as(_u32p))
    return dims


def cell_assign(pos, box, r_list):
    pos, pp = _d(pos)
    b, bp = _box(box)
    N = pos.shape[0]
    cell = np.zeros(N, dtype=np.uint32)
    dims = np.zeros(3, dtype=np.uint32)
    lib().orc_cell_assign(pp, C.c_uint64(N), bp, C.c_double(r_list), cell.ctypes.data_as(_u32p),
                          dims.ctypes.data_as(_u32p))
    return cell, dims


def neighbor_pairs(pos, box, r_list):
    """All unordered tag pairs (a<b) within r_list, shape (n_pairs, 2), lexicographically sorted."""
    pos, pp = _d(pos)
    b, bp = _box(box)
    N = pos.shape[0]
    n = lib().orc_neighbor_pairs(pp, C.c_uint64(N), bp, C.c_double(r_list), None, C.c_uint64(0))
    pairs = np.zeros((n, 2), dtype=np.uint32)
    n2 = lib().orc_neighbor_pairs(pp, C.c_uint64(N), bp, C.c_double(r_list), pairs.ctypes.data_as(_u32p),
                                  C.c_uint64(n))
    assert n2 == n
    return pairs


def needs_rebuild(pos, pos_ref, box, r_buff) -> bool:
    pos, pp = _d(pos)
    ref, rp = _d(pos_ref)
    b, bp = _box(box)
    return bool(lib().orc_needs_rebuild(pp, rp, C.c_uint64(pos.shape[0]), bp, C.c_double(r_buff)))


def forces_lj(pos, box, rc, epsilon=1.0, sigma=1.0, energy_shift=1):
    pos, pp = _d(pos)
    b, bp = _box(box)
    N = pos.shape[0]
    F = np.zeros((N, 3))
    E = np.zeros(N)
    lib().orc_forces_lj(pp, C.c_uint64(N), bp, C.c_double(rc), C.c_double(epsilon), C.c_double(sigma),
                        C.c_int(energy_shift), F.ctypes.data_as(_dp), E.ctypes.data_as(_dp))
    return F, E


def philox4x32_10(ctr, key):
    c, cp = _u(ctr)
    k, kp = _u(key)
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(cp, kp, out.ctypes.data_as(_u32p))
    return out


def dpd_theta(tag_a, tag_b, step, seed) -> float:
    return float(lib().orc_dpd_theta(int(tag_a), int(tag_b), int(step), int(seed)))


def forces_dpd(pos, vel, box, rc, A, gamma, kT, dt, step, seed):
    pos, pp = _d(pos)
    vel, vp = _d(vel)
    b, bp = _box(box)
    N = pos.shape[0]
    F = np.zeros((N, 3))
    lib().orc_forces_dpd(pp, vp, C.c_uint64(N), bp, C.c_double(rc), C.c_double(A), C.c_double(gamma),
                         C.c_double(kT), C.c_double(dt), C.c_uint64(step), C.c_uint64(seed),
                         F.ctypes.data_as(_dp))
    return F


def forces_bonds(pos, box, bonds, k, r0, force=None, energy=None):
    """Accumulates into force/energy (fresh zero arrays if None); returns (force, energy)."""
    pos, pp = _d(pos)
    b, bp = _box(box)
    N = pos.shape[0]
    bonds = np.ascontiguousarray(bonds, dtype=np.uint32).reshape(-1, 2)
    ta, tap = _u(bonds[:, 0])
    tb, tbp = _u(bonds[:, 1])
    F = np.zeros((N, 3)) if force is None else force
    E = np.zeros(N) if energy is None else energy
    assert F.flags.c_contiguous and F.dtype == np.float64
    lib().orc_forces_bonds(pp, C.c_uint64(N), bp, tap, tbp, C.c_uint64(bonds.shape[0]), C.c_double(k),
                           C.c_double(r0), F.ctypes.data_as(_dp), E.ctypes.data_as(_dp))
    return F, E


# ---- virial / pressure and further force fields (md_oracle_ext.c) ------------------------------------
PAIR_KINDS = {"lj": 0, "yukawa": 1, "gaussian": 2, "morse": 3}


def _p4(params):
    p = np.zeros(4)
    p[:len(params)] = params
    return p, p.ctypes.data_as(_dp)


def pair_forces(pos, box, rc, kind, params, energy_shift=1):
    """kind: "lj" (eps, sigma) | "yukawa" (eps, kappa) | "gaussian" (eps, sigma) | "morse" (D0, alpha, r0)."""
    pos, pp = _d(pos)
    b, bp = _box(box)
    p, ppar = _p4(params)
    N = pos.shape[0]
    F = np.zeros((N, 3)); E = np.zeros(N)
    lib().orc_pair_forces(pp, C.c_uint64(N), bp, C.c_double(rc), C.c_int(PAIR_KINDS[kind]), ppar, C.c_int(energy_shift),
                          F.ctypes.data_as(_dp), E.ctypes.data_as(_dp))
    return F, E


def pair_table(pos, box, r_min, r_max, U, F):
    """Tabulated pair potential (R37): U, F = -dU/dr at M evenly spaced radii in [r_min, r_max], linear interpolation.
    Returns (force, energy, virial)."""
    pos, pp = _d(pos)
    b, bp = _box(box)
    U, Up = _d(U)
    F, Fp = _d(F)
    assert U.shape == F.shape and U.ndim == 1 and U.shape[0] >= 2
    N = pos.shape[0]
    Fo = np.zeros((N, 3)); E = np.zeros(N); W = np.zeros(6)
    lib().orc_pair_table(pp, C.c_uint64(N), bp, C.c_double(r_min), C.c_double(r_max), C.c_uint64(U.shape[0]), Up, Fp,
                         Fo.ctypes.data_as(_dp), E.ctypes.data_as(_dp), W.ctypes.data_as(_dp))
    return Fo, E, W


def probe_pair_forces(pos, box, rc, kind, params, probes, energy_shift=1, table=None):
    """Force and energy of the probe particles against all N (O(M N)); kind as pair_forces, or "table" with
    table = (r_min, r_max, U, F) (R37)."""
    pos, pp = _d(pos)
    b, bp = _box(box)
    pr, prp = _u(probes)
    M = pr.shape[0]
    Fo = np.zeros((M, 3)); E = np.zeros(M)
    if kind == "table":
        r_min, r_max, U, F = table
        U, Up = _d(U); F, Fp = _d(F)
        p, ppar = _p4(())
        lib().orc_probe_pair_forces(pp, C.c_uint64(pos.shape[0]), bp, C.c_double(rc), C.c_int(4), ppar, C.c_int(0),
                                    C.c_double(r_min), C.c_double(r_max), C.c_uint64(U.shape[0]), Up, Fp, prp, C.c_uint64(M),
                                    Fo.ctypes.data_as(_dp), E.ctypes.data_as(_dp))
    else:
        p, ppar = _p4(params)
        lib().orc_probe_pair_forces(pp, C.c_uint64(pos.shape[0]), bp, C.c_double(rc), C.c_int(PAIR_KINDS[kind]), ppar,
                                    C.c_int(energy_shift), C.c_double(0.0), C.c_double(0.0), C.c_uint64(0), None, None, prp,
                                    C.c_uint64(M), Fo.ctypes.data_as(_dp), E.ctypes.data_as(_dp))
    return Fo, E


def virial_pair(pos, box, rc, kind, params):
    """W (xx, yy, zz, xy, xz, yz) = sum over pairs of d (x) F."""
    pos, pp = _d(pos)
    b, bp = _box(box)
    p, ppar = _p4(params)
    W = np.zeros(6)
    lib().orc_virial_pair(pp, C.c_uint64(pos.shape[0]), bp, C.c_double(rc), C.c_int(PAIR_KINDS[kind]), ppar,
                          W.ctypes.data_as(_dp))
    return W


def virial_dpd(pos, vel, box, rc, A, gamma, kT, dt, step, seed):
    pos, pp = _d(pos)
    vel, vp = _d(vel)
    b, bp = _box(box)
    W = np.zeros(6)
    lib().orc_virial_dpd(pp, vp, C.c_uint64(pos.shape[0]), bp, C.c_double(rc), C.c_double(A), C.c_double(gamma),
                         C.c_double(kT), C.c_double(dt), C.c_uint64(step), C.c_uint64(seed), W.ctypes.data_as(_dp))
    return W


def forces_bonds_kind(pos, box, bonds, kind, k, r0, force=None, energy=None, virial=None):
    """kind: "harmonic" | "fene".  Accumulates into force / energy / virial (fresh zero arrays if None)."""
    pos, pp = _d(pos)
    b, bp = _box(box)
    N = pos.shape[0]
    bonds = np.ascontiguousarray(bonds, dtype=np.uint32).reshape(-1, 2)
    ta, tap = _u(bonds[:, 0])
    tb, tbp = _u(bonds[:, 1])
    F = np.zeros((N, 3)) if force is None else force
    E = np.zeros(N) if energy is None else energy
    W = np.zeros(6) if virial is None else virial
    lib().orc_forces_bonds_kind(pp, C.c_uint64(N), bp, tap, tbp, C.c_uint64(bonds.shape[0]),
                                C.c_int({"harmonic": 0, "fene": 1}[kind]), C.c_double(k), C.c_double(r0),
                                F.ctypes.data_as(_dp), E.ctypes.data_as(_dp), W.ctypes.data_as(_dp))
    return F, E, W


def bond_table(pos, box, bonds, r_min, r_max, U, F, force=None, energy=None, virial=None):
    """Tabulated bonds (R38): U, F = -dU/dr at len(U) evenly spaced lengths in [r_min, r_max], linear interpolation; a bond
    outside [r_min, r_max) gives NaN.  Accumulates; returns (force, energy, virial)."""
    pos, pp = _d(pos)
    b, bp = _box(box)
    N = pos.shape[0]
    bonds = np.ascontiguousarray(bonds, dtype=np.uint32).reshape(-1, 2)
    ta, tap = _u(bonds[:, 0])
    tb, tbp = _u(bonds[:, 1])
    U, Up = _d(U)
    F, Fp = _d(F)
    assert U.shape == F.shape and U.ndim == 1 and U.shape[0] >= 2
    Fo = np.zeros((N, 3)) if force is None else force
    E = np.zeros(N) if energy is None else energy
    W = np.zeros(6) if virial is None else virial
    lib().orc_bond_table(pp, C.c_uint64(N), bp, tap, tbp, C.c_uint64(bonds.shape[0]), C.c_double(r_min), C.c_double(r_max),
                         C.c_uint64(U.shape[0]), Up, Fp, Fo.ctypes.data_as(_dp), E.ctypes.data_as(_dp), W.ctypes.data_as(_dp))
    return Fo, E, W


def forces_angles(pos, box, angles, k, theta0, force=None, energy=None, virial=None):
    """angles: (n, 3) tags (a, b, c), b the vertex.  Accumulates; returns (force, energy, virial)."""
    pos, pp = _d(pos)
    b, bp = _box(box)
    N = pos.shape[0]
    ang = np.ascontiguousarray(angles, dtype=np.uint32).reshape(-1, 3)
    ta, tap = _u(ang[:, 0]); tb, tbp = _u(ang[:, 1]); tc, tcp = _u(ang[:, 2])
    F = np.zeros((N, 3)) if force is None else force
    E = np.zeros(N) if energy is None else energy
    W = np.zeros(6) if virial is None else virial
    lib().orc_forces_angles(pp, C.c_uint64(N), bp, tap, tbp, tcp, C.c_uint64(ang.shape[0]), C.c_double(k),
                            C.c_double(theta0), F.ctypes.data_as(_dp), E.ctypes.data_as(_dp), W.ctypes.data_as(_dp))
    return F, E, W


def dihedral_angle(xa, xb, xc, xd, box) -> float:
    b, bp = _box(box)
    L = lib()
    L.orc_dihedral_angle.restype = C.c_double
    arrs = [np.ascontiguousarray(x, dtype=np.float64) for x in (xa, xb, xc, xd)]
    return float(L.orc_dihedral_angle(*[x.ctypes.data_as(_dp) for x in arrs], bp))


def forces_dihedrals(pos, box, dihedrals, k, s, n, force=None, energy=None, virial=None):
    """dihedrals: (m, 4) tags (a, b, c, d); U = k/2 (1 + s cos(n phi)).  Accumulates; returns (force, energy, virial)."""
    pos, pp = _d(pos)
    b, bp = _box(box)
    N = pos.shape[0]
    q = np.ascontiguousarray(dihedrals, dtype=np.uint32).reshape(-1, 4)
    t = [_u(q[:, i]) for i in range(4)]
    F = np.zeros((N, 3)) if force is None else force
    E = np.zeros(N) if energy is None else energy
    W = np.zeros(6) if virial is None else virial
    lib().orc_forces_dihedrals(pp, C.c_uint64(N), bp, t[0][1], t[1][1], t[2][1], t[3][1], C.c_uint64(q.shape[0]),
                               C.c_double(k), C.c_int(int(s)), C.c_int(int(n)), F.ctypes.data_as(_dp),
                               E.ctypes.data_as(_dp), W.ctypes.data_as(_dp))
    return F, E, W


def langevin_u(tag, step, seed):
    """(u_x, u_y, u_z), uniform on (-1, 1), of particle `tag` at `step` (R36)."""
    u = np.zeros(3)
    lib().orc_langevin_u(C.c_uint32(int(tag)), C.c_uint64(int(step)), C.c_uint64(int(seed)), u.ctypes.data_as(_dp))
    return u


def forces_langevin(vel, gamma, kT, dt, step, seed, force=None):
    """F_a += -gamma v_a + sqrt(6 gamma kT / dt) u_a(step)  (R36).  Accumulates; returns force."""
    vel, vp = _d(vel)
    N = vel.shape[0]
    F = np.zeros((N, 3)) if force is None else force
    lib().orc_forces_langevin(vp, C.c_uint64(N), C.c_double(gamma), C.c_double(kT), C.c_double(dt), C.c_uint64(int(step)),
                              C.c_uint64(int(seed)), F.ctypes.data_as(_dp))
    return F


def pressure(vel, box, W, mass=None):
    """P = (2 K + tr W) / (3 V)  (virial theorem, R32)."""
    m = 1.0 if mass is None else np.asarray(mass)[:, None]
    K = 0.5 * float(np.sum(m * np.asarray(vel) ** 2))
    return (2.0 * K + W[0] + W[1] + W[2]) / (3.0 * float(np.prod(np.broadcast_to(box, (3,)))))


def vv_half1(pos, vel, image, force, box, dt, mass=None):
    """In place on pos, vel, image (C-contiguous float64 / int32 arrays)."""
    b, bp = _box(box)
    N = pos.shape[0]
    for a in (pos, vel, force):
        assert a.flags.c_contiguous and a.dtype == np.float64
    mp = None
    if mass is not None:
        mass, mp = _d(mass)
    ip = image.ctypes.data_as(_i32p) if image is not None else None
    lib().orc_vv_half1(pos.ctypes.data_as(_dp), vel.ctypes.data_as(_dp), ip, force.ctypes.data_as(_dp), mp,
                       C.c_uint64(N), bp, C.c_double(dt))


def vv_half2(vel, force, dt, mass=None):
    N = vel.shape[0]
    assert vel.flags.c_contiguous and force.flags.c_contiguous
    mp = None
    if mass is not None:
        mass, mp = _d(mass)
    lib().orc_vv_half2(vel.ctypes.data_as(_dp), force.ctypes.data_as(_dp), mp, C.c_uint64(N), C.c_double(dt))


def probe_nlist(pos, box, r_list, probes, row_stride=512):
    pos, pp = _d(pos)
    b, bp = _box(box)
    pr, prp = _u(probes)
    M = pr.shape[0]
    counts = np.zeros(M, dtype=np.uint32)
    nbrs = np.full((M, row_stride), 0xFFFFFFFF, dtype=np.uint32)
    lib().orc_probe_nlist(pp, C.c_uint64(pos.shape[0]), bp, C.c_double(r_list), prp, C.c_uint64(M),
                          counts.ctypes.data_as(_u32p), nbrs.ctypes.data_as(_u32p), C.c_uint64(row_stride))
    return counts, nbrs


def probe_forces_lj(pos, box, rc, probes, epsilon=1.0, sigma=1.0, energy_shift=1):
    pos, pp = _d(pos)
    b, bp = _box(box)
    pr, prp = _u(probes)
    M = pr.shape[0]
    F = np.zeros((M, 3))
    E = np.zeros(M)
    lib().orc_probe_forces_lj(pp, C.c_uint64(pos.shape[0]), bp, C.c_double(rc), C.c_double(epsilon),
                              C.c_double(sigma), C.c_int(energy_shift), prp, C.c_uint64(M),
                              F.ctypes.data_as(_dp), E.ctypes.data_as(_dp))
    return F, E


def probe_forces_dpd(pos, vel, box, rc, A, gamma, kT, dt, step, seed, probes):
    pos, pp = _d(pos)
    vel, vp = _d(vel)
    b, bp = _box(box)
    pr, prp = _u(probes)
    M = pr.shape[0]
    F = np.zeros((M, 3))
    lib().orc_probe_forces_dpd(pp, vp, C.c_uint64(pos.shape[0]), bp, C.c_double(rc), C.c_double(A),
                               C.c_double(gamma), C.c_double(kT), C.c_double(dt), C.c_uint64(step),
                               C.c_uint64(seed), prp, C.c_uint64(M), F.ctypes.data_as(_dp))
    return F


# ------------------------------------------------------------------------------------------------------
# NVT: Nose-Hoover thermostat (SURVEY.md 8(f) row 1; "NVT ... Nose-Hoover" PAPER.md:63, :208, :214; the paper prints
# no equations -> DESIGN.md R30).  Equations of motion: dx/dt = v, dv/dt = F/m - xi v, dxi/dt = (T_inst/T0 - 1)/tau^2,
# deta/dt = xi, T_inst = 2 K / g with g = 3N - 3 (R18).  Velocity-Verlet discretisation, step by step, plain numpy:
#   half 1:      v <- (v + (dt/2) F/m) / (1 + (dt/2) xi) ;  x <- x + dt v ;  wrap
#   thermostat:  K' = sum 1/2 m v^2 ;  xi_old = xi ;  xi <- xi + (dt/tau^2) (2K'/(g kT0) - 1) ;  eta <- eta + (dt/2)(xi + xi_old)
#   forces at the new x
#   half 2:      v <- v + (dt/2) (F/m - xi v)
# Conserved: K + U + g kT0 (tau^2 xi^2 / 2 + eta).
# ------------------------------------------------------------------------------------------------------
def nvt_half1(pos, vel, image, force, box, dt, xi, mass=None):
    """In place on pos, vel, image (C-contiguous float64 / int32)."""
    m = 1.0 if mass is None else np.asarray(mass, dtype=np.float64)[:, None]
    vel[:] = (vel + (0.5 * dt * force) / m) / (1.0 + 0.5 * dt * xi)
    pos += dt * vel
    b = np.asarray(box, dtype=np.float64)
    hi = pos >= 0.5 * b
    lo = pos < -0.5 * b
    pos[hi] -= np.broadcast_to(b, pos.shape)[hi]
    pos[lo] += np.broadcast_to(b, pos.shape)[lo]
    image[hi] += 1
    image[lo] -= 1


def nvt_thermostat(vel, dt, kT, tau, xi, eta, mass=None):
    """Returns (xi_new, eta_new, K) from the velocities left by half 1."""
    m = 1.0 if mass is None else np.asarray(mass, dtype=np.float64)[:, None]
    K = 0.5 * float(np.sum(m * vel * vel))
    g = 3 * vel.shape[0] - 3
    xi_new = xi + (dt / (tau * tau)) * (2.0 * K / (g * kT) - 1.0)
    eta_new = eta + 0.5 * dt * (xi_new + xi)
    return xi_new, eta_new, K


def nvt_half2(vel, force, dt, xi, mass=None):
    m = 1.0 if mass is None else np.asarray(mass, dtype=np.float64)[:, None]
    vel += 0.5 * dt * (force / m - xi * vel)


# ------------------------------------------------------------------------------------------------------
# NVT, second scheme: the explicit reversible Martyna-Tobias-Klein update ("NVT (Nose-Hoover, then
# MTK)"; ensembles "implement the Velocity-Verlet or the symplectic Martyna-Tobias-Klein update equations";
# no equations printed -> DESIGN.md R39).  Same equations of motion as above with one thermostat (chain length 1),
# Q = g kT0 tau^2, integrated by the symmetric Trotter factorisation of Martyna, Tuckerman, Tobias & Klein (1996):
#   step = T(dt/2)  kick(dt/2)  drift(dt)  [forces]  kick(dt/2)  T(dt/2),
#   T(dt/2):  G = (2K - g kT0)/Q ; xi += (dt/4) G ; s = exp(-xi dt/2) ; v <- s v ; K <- s^2 K ; eta += xi dt/2 ;
#             G = (2K - g kT0)/Q ; xi += (dt/4) G
# (each factor is the exact flow of its part, so the step is time-reversible and second order).  Conserved quantity as
# above.  kick and drift are vv_half1 / vv_half2.
# ------------------------------------------------------------------------------------------------------
def mtk_thermostat_half(vel, dt, kT, tau, xi, eta, mass=None):
    """T(dt/2) in place on vel; returns (xi, eta)."""
    m = 1.0 if mass is None else np.asarray(mass, dtype=np.float64)[:, None]
    g = 3 * vel.shape[0] - 3
    Q = g * kT * tau * tau
    K = 0.5 * float(np.sum(m * vel * vel))
    xi = xi + 0.25 * dt * (2.0 * K - g * kT) / Q
    s = float(np.exp(-0.5 * dt * xi))
    vel *= s
    K = K * s * s
    eta = eta + 0.5 * dt * xi
    xi = xi + 0.25 * dt * (2.0 * K - g * kT) / Q
    return xi, eta


# ------------------------------------------------------------------------------------------------------
# The step loop, in the order of DESIGN.md "The path" (S6a -> S3 -> [S1,S2] -> S4 (+S5) -> S6b).
# ------------------------------------------------------------------------------------------------------
class Sim:
    """Plain MD driver on top of the O(N^2) routines.

    what: dict with any of
       lj    = dict(epsilon, sigma, energy_shift)
       dpd   = dict(A, gamma, kT, seed)
       bonds = dict(k, r0)  (+ self.bonds array)
       langevin = dict(gamma, kT, seed)   (R36)
    Forces never depend on a neighbour list here (all pairs); the rebuild trigger (O3) is evaluated
    only to log WHEN the CUDA path must rebuild.
    """

    def __init__(self, pos, vel, box, rc, r_buff, what, bonds=None, mass=None, step0=0, nvt=None):
        self.nvt = nvt                       # None = NVE; dict(kT, tau) = Nose-Hoover (R30); + scheme="mtk": R39
        self.xi, self.eta = 0.0, 0.0
        self.box = np.ascontiguousarray(np.broadcast_to(np.asarray(box, dtype=np.float64), (3,)))
        self.pos = wrap(pos, self.box)
        self.vel = np.array(vel, dtype=np.float64, order="C")
        self.N = self.pos.shape[0]
        self.image = np.zeros((self.N, 3), dtype=np.int32)
        self.rc, self.r_buff = float(rc), float(r_buff)
        self.what = what
        self.bonds = bonds
        self.mass = mass
        self.step = int(step0)
        self.pos_ref = self.pos.copy()
        self.rebuild_steps = []
        self.force = None
        self.energy = None

    def compute_forces(self, dt, step):
        F = np.zeros((self.N, 3))
        E = np.zeros(self.N)
        if "lj" in self.what:
            p = self.what["lj"]
            F, E = forces_lj(self.pos, self.box, self.rc, p.get("epsilon", 1.0), p.get("sigma", 1.0),
                             p.get("energy_shift", 1))
        if "dpd" in self.what:
            p = self.what["dpd"]
            F = F + forces_dpd(self.pos, self.vel, self.box, self.rc, p["A"], p["gamma"], p["kT"], dt, step,
                               p["seed"])
        if "bonds" in self.what:
            p = self.what["bonds"]
            F = np.ascontiguousarray(F)
            forces_bonds(self.pos, self.box, self.bonds, p["k"], p["r0"], F, E)
        if "langevin" in self.what:
            p = self.what["langevin"]
            F = np.ascontiguousarray(F)
            forces_langevin(self.vel, p["gamma"], p["kT"], dt, step, p["seed"], F)
        self.force, self.energy = np.ascontiguousarray(F), E
        return self.force

    def run(self, n_steps, dt):
        if self.force is None:
            self.compute_forces(dt, self.step)          # DESIGN.md R16: F(t0) before the first half-kick
        for _ in range(n_steps):
            mtk = self.nvt is not None and self.nvt.get("scheme") == "mtk"
            if mtk:
                self.xi, self.eta = mtk_thermostat_half(self.vel, dt, self.nvt["kT"], self.nvt["tau"], self.xi, self.eta,
                                                        self.mass)
            if self.nvt is None or mtk:
                vv_half1(self.pos, self.vel, self.image, self.force, self.box, dt, self.mass)
            else:
                nvt_half1(self.pos, self.vel, self.image, self.force, self.box, dt, self.xi, self.mass)
                self.xi_half1 = self.xi
                self.xi, self.eta, _ = nvt_thermostat(self.vel, dt, self.nvt["kT"], self.nvt["tau"], self.xi, self.eta,
                                                      self.mass)
            if needs_rebuild(self.pos, self.pos_ref, self.box, self.r_buff):
                self.pos_ref = self.pos.copy()
                self.rebuild_steps.append(self.step + 1)
            self.compute_forces(dt, self.step + 1)      # DESIGN.md R15: hash counter = step being completed
            if self.nvt is None or mtk:
                vv_half2(self.vel, self.force, dt, self.mass)
            else:
                nvt_half2(self.vel, self.force, dt, self.xi, self.mass)
            if mtk:
                self.xi, self.eta = mtk_thermostat_half(self.vel, dt, self.nvt["kT"], self.nvt["tau"], self.xi, self.eta,
                                                        self.mass)
            self.step += 1
        return self

    def nvt_conserved(self):
        """K + U + g kT0 (tau^2 xi^2 / 2 + eta) (R30)."""
        g = 3 * self.N - 3
        return (self.kinetic_energy() + self.potential_energy()
                + g * self.nvt["kT"] * (0.5 * self.nvt["tau"] ** 2 * self.xi ** 2 + self.eta))

    def kinetic_energy(self):
        m = 1.0 if self.mass is None else np.asarray(self.mass)[:, None]
        return 0.5 * float(np.sum(m * self.vel * self.vel))

    def potential_energy(self):
        return float(np.sum(self.energy))
