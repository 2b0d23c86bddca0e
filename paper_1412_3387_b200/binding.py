"""Thin Python binding of the C-ABI in include/b200md.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of csrc/libb200md.so; this module converts numpy arrays /
torch tensors to raw pointers and calls the functions of the same name.  There is no fallback: if the shared
library is missing or no CUDA device is present the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libb200md.so")

MD_FP64, MD_MIXED = 0, 1
MD_ORDER_LEX, MD_ORDER_MORTON, MD_ORDER_HILBERT = 0, 1, 2
MD_F_LJ, MD_F_DPD, MD_F_BONDS, MD_F_NVT, MD_F_PAIR, MD_F_ANGLES, MD_F_DIHEDRALS, MD_F_LANGEVIN, MD_F_MTK = 1, 2, 4, 8, 16, 32, 64, 128, 256
PAIR_KINDS = {"lj": 0, "yukawa": 1, "gaussian": 2, "morse": 3, "table": 4}
BOND_KINDS = {"harmonic": 0, "fene": 1, "table": 2}
MD_SCHED_SYNC, MD_SCHED_SPECULATIVE, MD_SCHED_BATCH = 0, 1, 2
MD_OPT_TILE_BRICK, MD_OPT_ACC_BLOCK, MD_OPT_RETUNE_PERIOD, MD_OPT_PROFILE_STRIDE = 1, 2, 4, 8
MD_N_KERNELS = 8
MD_K_NLIST, MD_K_LJ, MD_K_DPD, MD_K_BONDS, MD_K_INTEGRATE, MD_K_CELLS = 0, 1, 2, 3, 4, 5
KERNEL_NAMES = {MD_K_NLIST: "nlist", MD_K_LJ: "lj", MD_K_DPD: "dpd", MD_K_BONDS: "bonds",
                MD_K_INTEGRATE: "integrate", MD_K_CELLS: "cells"}

EXPORTS = ["md_create", "md_workspace_bytes", "md_set_workspace", "md_configure", "md_destroy", "md_last_error", "md_set_state", "md_set_bonds",
           "md_get_state", "md_get_forces", "md_build_cells", "md_get_cells", "md_build_nlist", "md_get_nlist",
           "md_get_nlist_rows", "md_forces_lj", "md_forces_dpd", "md_forces_bonds", "md_forces_pair", "md_set_pair_table", "md_set_bond_table", "md_forces_bond_table", "md_forces_fene", "md_set_angles", "md_forces_angles",
           "md_set_dihedrals", "md_forces_dihedrals", "md_forces_langevin", "md_pressure",
           "md_integrate_nve",
           "md_needs_rebuild", "md_step", "md_tune", "md_tune_rbuff", "md_set_option", "md_set_launch", "md_get_stats", "md_set_profiling",
           "md_debug_philox", "md_debug_peak", "md_struct_size", "md_thermo", "md_integrate_nvt", "md_set_thermostat", "md_get_thermostat", "md_mtk_thermostat_half",
           "md_kinetic_noalloc", "md_noalloc_last_error"]


class md_step_desc(C.Structure):
    _fields_ = [("flags", C.c_uint32), ("lj_energy_shift", C.c_int32), ("dt", C.c_double),
                ("lj_epsilon", C.c_double), ("lj_sigma", C.c_double),
                ("dpd_A", C.c_double), ("dpd_gamma", C.c_double), ("dpd_kT", C.c_double),
                ("dpd_seed", C.c_uint64), ("bond_k", C.c_double), ("bond_r0", C.c_double),
                ("nvt_kT", C.c_double), ("nvt_tau", C.c_double),
                ("pair_kind", C.c_int32), ("bond_kind", C.c_int32), ("pair_p", C.c_double * 4),
                ("angle_k", C.c_double), ("angle_theta0", C.c_double),
                ("dihedral_k", C.c_double), ("dihedral_sign", C.c_int32), ("dihedral_n", C.c_int32),
                ("langevin_gamma", C.c_double), ("langevin_kT", C.c_double), ("langevin_seed", C.c_uint64)]


class md_pressure_t(C.Structure):
    _fields_ = [("virial", C.c_double * 6), ("kinetic", C.c_double), ("volume", C.c_double), ("pressure", C.c_double)]


class md_thermo_t(C.Structure):
    _fields_ = [("kinetic", C.c_double), ("potential", C.c_double), ("momentum", C.c_double * 3),
                ("temperature", C.c_double)]


class md_stats(C.Structure):
    _fields_ = [("steps", C.c_uint64), ("rebuilds", C.c_uint64), ("dangerous_builds", C.c_uint64),
                ("nlist_entries", C.c_uint64), ("nlist_capacity", C.c_uint64), ("device_bytes", C.c_uint64),
                ("mean_neighbors", C.c_double), ("dims", C.c_uint32 * 3), ("max_cell_count", C.c_uint32),
                ("block", C.c_int32 * MD_N_KERNELS), ("w", C.c_int32 * MD_N_KERNELS),
                ("tuned_us", C.c_float * MD_N_KERNELS), ("tuner_runs", C.c_uint32), ("launches", C.c_uint32),
                ("stage_ms", C.c_double * MD_N_KERNELS), ("stage_launches", C.c_uint64 * MD_N_KERNELS),
                ("speculative_forces", C.c_uint64), ("wasted_forces", C.c_uint64),
                ("r_buff", C.c_double), ("rbuff_tuned_tps", C.c_double)]


class MDError(RuntimeError):
    pass


_lib = None


def load():
    """Open csrc/libb200md.so (built by `python -m paper_1412_3387_b200.csrc.build`).  Raises if missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise MDError(f"{LIB_PATH} is missing: build it with `python -m paper_1412_3387_b200.csrc.build` "
                      "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, u64, dbl, i32, u32 = C.c_void_p, C.c_uint64, C.c_double, C.c_int, C.c_uint32
    sig = {
        "md_create": [C.POINTER(vp), C.POINTER(dbl), u64, dbl, dbl],
        "md_configure": [vp, i32, vp, i32, i32],
        "md_workspace_bytes": [C.POINTER(dbl), u64, dbl, dbl, i32, C.POINTER(u64)],
        "md_set_workspace": [vp, vp, u64],
        "md_destroy": [vp],
        "md_set_state": [vp, vp, vp, vp, u64],
        "md_set_bonds": [vp, vp, vp, u64],
        "md_get_state": [vp, vp, vp, vp],
        "md_get_forces": [vp, vp, vp],
        "md_build_cells": [vp],
        "md_get_cells": [vp, vp, C.POINTER(u32)],
        "md_build_nlist": [vp],
        "md_get_nlist": [vp, C.POINTER(u64), vp, u64],
        "md_get_nlist_rows": [vp, vp, u32, vp, vp, u32],
        "md_forces_lj": [vp, dbl, dbl, i32],
        "md_forces_dpd": [vp, dbl, dbl, dbl, dbl, u64, u64],
        "md_forces_bonds": [vp, dbl, dbl],
        "md_forces_pair": [vp, i32, C.POINTER(dbl), i32],
        "md_set_pair_table": [vp, dbl, dbl, vp, vp, u64],
        "md_set_bond_table": [vp, dbl, dbl, vp, vp, u64],
        "md_forces_bond_table": [vp],
        "md_forces_fene": [vp, dbl, dbl],
        "md_set_angles": [vp, vp, vp, vp, u64],
        "md_forces_angles": [vp, dbl, dbl],
        "md_set_dihedrals": [vp, vp, vp, vp, vp, u64],
        "md_forces_dihedrals": [vp, dbl, i32, i32],
        "md_forces_langevin": [vp, dbl, dbl, dbl, u64, u64],
        "md_pressure": [vp, C.POINTER(md_step_desc), vp],
        "md_integrate_nve": [vp, dbl, i32],
        "md_needs_rebuild": [vp, C.POINTER(i32)],
        "md_step": [vp, C.POINTER(md_step_desc), u64],
        "md_tune": [vp, C.POINTER(md_step_desc), i32],
        "md_tune_rbuff": [vp, C.POINTER(md_step_desc), C.POINTER(dbl), u32, u64, C.POINTER(dbl)],
        "md_set_launch": [vp, i32, i32, i32],
        "md_set_option": [vp, i32, C.c_int64],
        "md_get_stats": [vp, C.POINTER(md_stats)],
        "md_set_profiling": [vp, i32],
        "md_debug_philox": [vp, vp, vp, vp, u64],
        "md_debug_peak": [vp, i32, C.POINTER(dbl)],
        "md_struct_size": [i32],
        "md_thermo": [vp, vp],
        "md_integrate_nvt": [vp, C.c_double, i32, C.c_double, C.c_double],
        "md_set_thermostat": [vp, C.c_double, C.c_double],
        "md_get_thermostat": [vp, vp, vp],
        "md_mtk_thermostat_half": [vp, dbl, dbl, dbl],
        "md_kinetic_noalloc": [vp, vp, u64, vp, vp],
    }
    for name, args in sig.items():
        fn = getattr(L, name)
        fn.argtypes = args
        fn.restype = C.c_int
    for k, st in enumerate((md_step_desc, md_stats, md_thermo_t, md_pressure_t)):
        if L.md_struct_size(k) != C.sizeof(st):
            raise MDError(f"binding out of date: sizeof({st.__name__}) = {C.sizeof(st)}, library says {L.md_struct_size(k)}")
    L.md_last_error.argtypes = [vp]
    L.md_last_error.restype = C.c_char_p
    L.md_noalloc_last_error.argtypes = []
    L.md_noalloc_last_error.restype = C.c_char_p
    _lib = L
    return L


def _ptr(a):
    """Raw address of a numpy array (host) or torch tensor (host or CUDA); None -> NULL."""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        assert a.flags.c_contiguous, "array must be C-contiguous"
        return a.ctypes.data
    if hasattr(a, "data_ptr"):
        assert a.is_contiguous(), "tensor must be contiguous"
        return a.data_ptr()
    raise TypeError(type(a))


def workspace_bytes(box, N, rc, r_buff, precision=MD_FP64) -> int:
    """md_workspace_bytes: device bytes a context of this problem needs (upper estimate)."""
    b = (C.c_double * 3)(*[float(x) for x in np.broadcast_to(np.asarray(box, dtype=np.float64), (3,))])
    n = C.c_uint64()
    s = load().md_workspace_bytes(b, int(N), float(rc), float(r_buff), int(precision), C.byref(n))
    if s != 0:
        raise MDError(f"md_workspace_bytes -> {s}")
    return int(n.value)


def step_desc(kind: str, dt: float, params: dict, nvt: dict = None) -> md_step_desc:
    """nvt = dict(kT, tau): Nose-Hoover thermostat (MD_F_NVT) instead of NVE."""
    d = md_step_desc()
    d.dt = dt
    d.lj_epsilon, d.lj_sigma, d.lj_energy_shift = 1.0, 1.0, 1
    if kind == "lj":
        d.flags = MD_F_LJ
        d.lj_epsilon = params.get("epsilon", 1.0)
        d.lj_sigma = params.get("sigma", 1.0)
        d.lj_energy_shift = int(params.get("energy_shift", 1))
    elif kind in ("dpd", "polymer"):
        d.flags = MD_F_DPD | (MD_F_BONDS if kind == "polymer" else 0)
        d.dpd_A, d.dpd_gamma, d.dpd_kT = params["A"], params["gamma"], params["kT"]
        d.dpd_seed = int(params["seed"])
        d.bond_k, d.bond_r0 = params.get("bond_k", 0.0), params.get("bond_r0", 0.0)
    elif kind == "bonds":
        d.flags = MD_F_BONDS
        d.bond_k, d.bond_r0 = params["bond_k"], params["bond_r0"]
    elif kind == "pair":   # params: pair_kind ("yukawa" | "gaussian" | "morse" | "lj"), pair_p, energy_shift
        d.flags = MD_F_PAIR
        d.pair_kind = PAIR_KINDS[params["pair_kind"]]
        for i, v in enumerate(params.get("pair_p", ())):
            d.pair_p[i] = float(v)
        d.lj_energy_shift = int(params.get("energy_shift", 1))
    elif kind == "none":
        d.flags = 0
    else:
        raise ValueError(kind)
    if "bond_kind" in params and (d.flags & MD_F_BONDS or params.get("bonds_on")):
        d.flags |= MD_F_BONDS
        d.bond_kind = BOND_KINDS[params["bond_kind"]]
        d.bond_k, d.bond_r0 = params.get("bond_k", 0.0), params.get("bond_r0", 0.0)
    if "angle_k" in params:
        d.flags |= MD_F_ANGLES
        d.angle_k, d.angle_theta0 = float(params["angle_k"]), float(params["angle_theta0"])
    if "dihedral_k" in params:
        d.flags |= MD_F_DIHEDRALS
        d.dihedral_k = float(params["dihedral_k"])
        d.dihedral_sign, d.dihedral_n = int(params.get("dihedral_sign", 1)), int(params.get("dihedral_n", 1))
    if "langevin" in params:       # dict(gamma, kT, seed): Langevin thermostat (R36)
        q = params["langevin"]
        d.flags |= MD_F_LANGEVIN
        d.langevin_gamma, d.langevin_kT, d.langevin_seed = float(q["gamma"]), float(q["kT"]), int(q["seed"])
    if nvt is not None:
        d.flags |= MD_F_MTK if nvt.get("scheme") == "mtk" else MD_F_NVT
        d.nvt_kT, d.nvt_tau = float(nvt["kT"]), float(nvt["tau"])
    return d


class MD:
    """One simulation context (md_ctx).  Methods are 1:1 with the C entry points (md_ prefix dropped)."""

    def __init__(self, box, N, rc, r_buff, precision=MD_FP64, stream=None, order=MD_ORDER_MORTON, sched=MD_SCHED_BATCH,
                 workspace=None):
        """workspace: None (the library allocates), a CUDA uint8 tensor (md_set_workspace), or "torch": a tensor of
        md_workspace_bytes bytes is taken from torch's allocator and kept alive with this object."""
        self.L = load()
        self.N = int(N)
        b = (C.c_double * 3)(*[float(x) for x in np.broadcast_to(np.asarray(box, dtype=np.float64), (3,))])
        h = C.c_void_p()
        s = self.L.md_create(C.byref(h), b, self.N, float(rc), float(r_buff))
        if s != 0:
            raise MDError(f"md_create -> {s}: {self.L.md_last_error(None).decode()}")
        self.h = h
        self.workspace = None
        if isinstance(workspace, str) and workspace == "torch":
            import torch
            workspace = torch.empty(workspace_bytes(box, N, rc, r_buff, precision), dtype=torch.uint8, device="cuda")
        if workspace is not None:
            self.workspace = workspace          # kept alive until close()
            self._chk(self.L.md_set_workspace(self.h, workspace.data_ptr(), workspace.numel() * workspace.element_size()),
                      "md_set_workspace")
        self._chk(self.L.md_configure(self.h, precision, stream, order, sched), "md_configure")

    def _chk(self, s, who):
        if s != 0:
            raise MDError(f"{who} -> {s}: {self.L.md_last_error(self.h).decode()}")

    def close(self):
        if getattr(self, "h", None):
            self.L.md_destroy(self.h)
            self.h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # --- state
    def set_state(self, pos, vel, mass=None, step0=0):
        self._keep = (pos, vel, mass)
        self._chk(self.L.md_set_state(self.h, _ptr(pos), _ptr(vel), _ptr(mass), int(step0)), "md_set_state")

    def set_bonds(self, bonds):
        if bonds is None or len(bonds) == 0:
            self._chk(self.L.md_set_bonds(self.h, None, None, 0), "md_set_bonds")
            return
        b = np.ascontiguousarray(bonds, dtype=np.uint32).reshape(-1, 2)
        ta, tb = np.ascontiguousarray(b[:, 0]), np.ascontiguousarray(b[:, 1])
        self._chk(self.L.md_set_bonds(self.h, _ptr(ta), _ptr(tb), b.shape[0]), "md_set_bonds")

    def get_state(self, pos=None, vel=None, image=None):
        """Fills the given arrays/tensors; with no arguments returns fresh numpy (pos, vel, image)."""
        if pos is None and vel is None and image is None:
            pos = np.empty((self.N, 3)); vel = np.empty((self.N, 3)); image = np.empty((self.N, 3), dtype=np.int32)
        self._chk(self.L.md_get_state(self.h, _ptr(pos), _ptr(vel), _ptr(image)), "md_get_state")
        return pos, vel, image

    def get_forces(self, force=None, energy=None):
        if force is None and energy is None:
            force = np.empty((self.N, 3)); energy = np.empty(self.N)
        self._chk(self.L.md_get_forces(self.h, _ptr(force), _ptr(energy)), "md_get_forces")
        return force, energy

    # --- S1/S2
    def build_cells(self):
        self._chk(self.L.md_build_cells(self.h), "md_build_cells")

    def get_cells(self, cell_of=None):
        dims = (C.c_uint32 * 3)()
        if cell_of is None:
            cell_of = np.empty(self.N, dtype=np.uint32)
        self._chk(self.L.md_get_cells(self.h, _ptr(cell_of), dims), "md_get_cells")
        return cell_of, np.array(list(dims), dtype=np.uint32)

    def build_nlist(self):
        self._chk(self.L.md_build_nlist(self.h), "md_build_nlist")

    def get_nlist(self, device_out=None):
        """Unique pairs (tag_i < tag_j), unordered.  Returns a numpy (n,2) array unless a tensor is supplied."""
        n = C.c_uint64()
        self._chk(self.L.md_get_nlist(self.h, C.byref(n), None, 0), "md_get_nlist")
        if device_out is not None:
            assert device_out.numel() >= 2 * n.value
            self._chk(self.L.md_get_nlist(self.h, C.byref(n), _ptr(device_out), n.value), "md_get_nlist")
            return n.value
        pairs = np.empty((n.value, 2), dtype=np.uint32)
        self._chk(self.L.md_get_nlist(self.h, C.byref(n), _ptr(pairs), n.value), "md_get_nlist")
        return pairs

    def count_nlist(self) -> int:
        """Number of unordered pairs of the exported list (md_get_nlist with pairs = NULL)."""
        n = C.c_uint64()
        self._chk(self.L.md_get_nlist(self.h, C.byref(n), None, 0), "md_get_nlist")
        return int(n.value)

    def get_nlist_rows(self, probe_tags, row_stride=512):
        pr = np.ascontiguousarray(probe_tags, dtype=np.uint32)
        counts = np.empty(pr.shape[0], dtype=np.uint32)
        nbrs = np.empty((pr.shape[0], row_stride), dtype=np.uint32)
        self._chk(self.L.md_get_nlist_rows(self.h, _ptr(pr), pr.shape[0], _ptr(counts), _ptr(nbrs), row_stride),
                  "md_get_nlist_rows")
        return counts, nbrs

    # --- S4/S5/S6
    def forces_lj(self, epsilon=1.0, sigma=1.0, energy_shift=1):
        self._chk(self.L.md_forces_lj(self.h, float(epsilon), float(sigma), int(energy_shift)), "md_forces_lj")

    def forces_dpd(self, A, gamma, kT, dt, step, seed):
        self._chk(self.L.md_forces_dpd(self.h, float(A), float(gamma), float(kT), float(dt), int(step), int(seed)),
                  "md_forces_dpd")

    def forces_bonds(self, k, r0):
        self._chk(self.L.md_forces_bonds(self.h, float(k), float(r0)), "md_forces_bonds")

    def forces_pair(self, kind, p=(), energy_shift=1):
        p = list(p or ())
        arr = (C.c_double * 4)(*([float(x) for x in p] + [0.0] * (4 - len(p))))
        self._chk(self.L.md_forces_pair(self.h, PAIR_KINDS[kind], arr, int(energy_shift)), "md_forces_pair")

    def set_pair_table(self, r_min, r_max, U, F):
        """U, F = -dU/dr at len(U) evenly spaced radii in [r_min, r_max] (R37); None clears."""
        if U is None:
            self._chk(self.L.md_set_pair_table(self.h, 0.0, 0.0, None, None, 0), "md_set_pair_table")
            return
        U = np.ascontiguousarray(U, dtype=np.float64)
        F = np.ascontiguousarray(F, dtype=np.float64)
        if U.shape != F.shape or U.ndim != 1:
            raise ValueError("U and F must be 1-D arrays of the same length")
        self._chk(self.L.md_set_pair_table(self.h, float(r_min), float(r_max), _ptr(U), _ptr(F), U.shape[0]), "md_set_pair_table")

    def set_bond_table(self, r_min, r_max, U, F):
        """U, F = -dU/dr at len(U) evenly spaced bond lengths in [r_min, r_max] (R38); None clears."""
        if U is None:
            self._chk(self.L.md_set_bond_table(self.h, 0.0, 0.0, None, None, 0), "md_set_bond_table")
            return
        U = np.ascontiguousarray(U, dtype=np.float64)
        F = np.ascontiguousarray(F, dtype=np.float64)
        if U.shape != F.shape or U.ndim != 1:
            raise ValueError("U and F must be 1-D arrays of the same length")
        self._chk(self.L.md_set_bond_table(self.h, float(r_min), float(r_max), _ptr(U), _ptr(F), U.shape[0]), "md_set_bond_table")

    def forces_bond_table(self):
        self._chk(self.L.md_forces_bond_table(self.h), "md_forces_bond_table")

    def forces_fene(self, k, r0):
        self._chk(self.L.md_forces_fene(self.h, float(k), float(r0)), "md_forces_fene")

    def set_angles(self, angles):
        if angles is None or len(angles) == 0:
            self._chk(self.L.md_set_angles(self.h, None, None, None, 0), "md_set_angles")
            return
        a = np.ascontiguousarray(angles, dtype=np.uint32).reshape(-1, 3)
        ta, tb, tc = (np.ascontiguousarray(a[:, i]) for i in range(3))
        self._chk(self.L.md_set_angles(self.h, _ptr(ta), _ptr(tb), _ptr(tc), a.shape[0]), "md_set_angles")

    def forces_angles(self, k, theta0):
        self._chk(self.L.md_forces_angles(self.h, float(k), float(theta0)), "md_forces_angles")

    def set_dihedrals(self, dihedrals):
        if dihedrals is None or len(dihedrals) == 0:
            self._chk(self.L.md_set_dihedrals(self.h, None, None, None, None, 0), "md_set_dihedrals")
            return
        a = np.ascontiguousarray(dihedrals, dtype=np.uint32).reshape(-1, 4)
        t = [np.ascontiguousarray(a[:, i]) for i in range(4)]
        self._chk(self.L.md_set_dihedrals(self.h, _ptr(t[0]), _ptr(t[1]), _ptr(t[2]), _ptr(t[3]), a.shape[0]), "md_set_dihedrals")

    def forces_dihedrals(self, k, sign=1, n=1):
        self._chk(self.L.md_forces_dihedrals(self.h, float(k), int(sign), int(n)), "md_forces_dihedrals")

    def forces_langevin(self, gamma, kT, dt, step, seed):
        self._chk(self.L.md_forces_langevin(self.h, float(gamma), float(kT), float(dt), int(step), int(seed)), "md_forces_langevin")

    def pressure(self, desc: md_step_desc) -> dict:
        t = md_pressure_t()
        self._chk(self.L.md_pressure(self.h, C.byref(desc), C.byref(t)), "md_pressure")
        return dict(virial=np.array(list(t.virial)), kinetic=t.kinetic, volume=t.volume, pressure=t.pressure)

    def integrate_nve(self, dt, half):
        self._chk(self.L.md_integrate_nve(self.h, float(dt), int(half)), "md_integrate_nve")

    def mtk_thermostat_half(self, dt, kT, tau):
        self._chk(self.L.md_mtk_thermostat_half(self.h, float(dt), float(kT), float(tau)), "md_mtk_thermostat_half")

    def integrate_nvt(self, dt, half, kT, tau):
        self._chk(self.L.md_integrate_nvt(self.h, float(dt), int(half), float(kT), float(tau)), "md_integrate_nvt")

    def set_thermostat(self, xi, eta):
        self._chk(self.L.md_set_thermostat(self.h, float(xi), float(eta)), "md_set_thermostat")

    def get_thermostat(self):
        xi, eta = C.c_double(), C.c_double()
        self._chk(self.L.md_get_thermostat(self.h, C.byref(xi), C.byref(eta)), "md_get_thermostat")
        return xi.value, eta.value

    def needs_rebuild(self) -> bool:
        f = C.c_int()
        self._chk(self.L.md_needs_rebuild(self.h, C.byref(f)), "md_needs_rebuild")
        return bool(f.value)

    # --- S7/S8
    def step(self, desc: md_step_desc, n_steps: int):
        self._chk(self.L.md_step(self.h, C.byref(desc), int(n_steps)), "md_step")

    def tune(self, desc: md_step_desc, full: bool = False):
        self._chk(self.L.md_tune(self.h, C.byref(desc), int(full)), "md_tune")

    def tune_rbuff(self, desc: md_step_desc, candidates=None, burst_steps=0) -> float:
        """md_tune_rbuff: the skin with the most steps per second among `candidates` (None = 0.5 .. 2 x the current one)."""
        out = C.c_double()
        if candidates is None:
            arr, n = None, 0
        else:
            n = len(candidates)
            arr = (C.c_double * n)(*[float(x) for x in candidates])
        self._chk(self.L.md_tune_rbuff(self.h, C.byref(desc), arr, n, int(burst_steps), C.byref(out)), "md_tune_rbuff")
        return out.value

    def set_profiling(self, on: bool):
        self._chk(self.L.md_set_profiling(self.h, int(on)), "md_set_profiling")

    def set_option(self, option, value):
        self._chk(self.L.md_set_option(self.h, int(option), int(value)), "md_set_option")

    def set_launch(self, kernel, block, w):
        self._chk(self.L.md_set_launch(self.h, kernel, block, w), "md_set_launch")

    def stats(self) -> dict:
        st = md_stats()
        self._chk(self.L.md_get_stats(self.h, C.byref(st)), "md_get_stats")
        d = {k: getattr(st, k) for k in ("steps", "rebuilds", "dangerous_builds", "nlist_entries", "nlist_capacity",
                                         "device_bytes", "mean_neighbors", "max_cell_count", "tuner_runs", "launches",
                                         "speculative_forces", "wasted_forces", "r_buff", "rbuff_tuned_tps")}
        d["dims"] = list(st.dims)
        d["stage_ms"] = {KERNEL_NAMES[k]: st.stage_ms[k] for k in KERNEL_NAMES}
        d["stage_launches"] = {KERNEL_NAMES[k]: st.stage_launches[k] for k in KERNEL_NAMES}
        d["launch"] = {KERNEL_NAMES[k]: dict(block=st.block[k], w=st.w[k], us=st.tuned_us[k]) for k in KERNEL_NAMES}
        return d

    def thermo(self) -> dict:
        t = md_thermo_t()
        self._chk(self.L.md_thermo(self.h, C.byref(t)), "md_thermo")
        return dict(kinetic=t.kinetic, potential=t.potential, momentum=np.array(list(t.momentum)),
                    temperature=t.temperature)

    PEAK_PIPES = {"fp32_fma": 0, "fp32_fma2": 1, "fp64_fma": 2, "int32_mad": 3, "int32_mulhi": 4, "cvt_f32_f64": 5,
                  "rcp_f32": 6, "lds128": 7}

    def debug_peak(self, pipe) -> float:
        """Measured issue rate of one pipe in giga lane-instructions per second (md_debug_peak)."""
        v = C.c_double()
        self._chk(self.L.md_debug_peak(self.h, self.PEAK_PIPES.get(pipe, pipe), C.byref(v)), "md_debug_peak")
        return v.value

    def debug_philox(self, ctr, key):
        ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
        key = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
        out = np.empty_like(ctr)
        self._chk(self.L.md_debug_philox(self.h, _ptr(ctr), _ptr(key), _ptr(out), ctr.shape[0]), "md_debug_philox")
        return out


MD_NOALLOC_MAX_N = 8192 * 4096


def kinetic_noalloc(vel, mass, out4, n=None, stream=None):
    """md_kinetic_noalloc: sum 1/2 m v^2 and sum m v of n particles into out4 (4 doubles), device tensors only, no
    allocation anywhere, no synchronisation.  stream: a raw cudaStream_t value (e.g. torch.cuda.Stream.cuda_stream) or None."""
    L = load()
    if n is None:
        n = vel.shape[0]
    s = L.md_kinetic_noalloc(_ptr(vel), _ptr(mass), int(n), _ptr(out4), C.c_void_p(stream) if stream else None)
    if s != 0:
        raise MDError(f"md_kinetic_noalloc -> {s}: {L.md_noalloc_last_error().decode()}")


def from_workload(w, precision=None, **kw) -> MD:
    """Context for a paper_1412_3387_b200.inputs.Workload, state and bonds uploaded."""
    if precision is None:
        precision = MD_MIXED if w.precision == "mixed" else MD_FP64
    md = MD(w.box, w.N, w.rc, w.r_buff, precision=precision, **kw)
    md.set_state(w.pos, w.vel)
    if w.bonds is not None:
        md.set_bonds(w.bonds)
    return md
