"""ctypes front end of the host-side tree / group / list builder (workload/bhtree.cpp).

Harness input generation (SURVEY.md section 8(a) "H"): Morton-ordered particles, tree cells in
level order, i-groups and the two CSR index lists (EPJ = particle indices, SPJ = cell indices)
that PAPER.md P:77, P:153-156, P:181 describe.  Shared by the CUDA path and the oracle as INPUT.
"""
from __future__ import annotations

import ctypes
import dataclasses
import os

import numpy as np

from .. import build as _build
from .generators import Config, make_particles, make_sph_fields

_lib = None


def _load():
    global _lib
    if _lib is None:
        path = _build.build_workload()
        lib = ctypes.CDLL(path)
        vp, i64, i32, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double
        lib.bh_build.restype = vp
        lib.bh_build.argtypes = [i64, vp, ctypes.c_int, ctypes.c_int]
        lib.bh_free.argtypes = [vp]
        lib.bh_n_cell.restype = i64
        lib.bh_n_cell.argtypes = [vp]
        lib.bh_n_group.restype = i64
        lib.bh_n_group.argtypes = [vp]
        lib.bh_n_level.restype = i32
        lib.bh_n_level.argtypes = [vp]
        lib.bh_get_tree.argtypes = [vp] * 7
        lib.bh_get_groups.argtypes = [vp] * 4
        lib.bh_build_lists.restype = ctypes.c_int
        lib.bh_build_lists.argtypes = [vp, dbl, vp, vp, ctypes.POINTER(i64), ctypes.POINTER(i64)]
        lib.bh_get_lists.argtypes = [vp, vp, vp]
        lib.bh_build_neighbour_lists.restype = ctypes.c_int
        lib.bh_build_neighbour_lists.argtypes = [vp, vp, dbl, vp, vp, ctypes.POINTER(i64)]
        lib.bh_pack_data_lists.argtypes = [i64, i64] + [vp] * 8
        _lib = lib
    return _lib


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


@dataclasses.dataclass
class Workload:
    """Everything one force evaluation needs, in tree (Morton) order."""
    cfg: Config
    posm: np.ndarray        # [N,4] float32 (x,y,z,m), Morton order
    vel: np.ndarray | None  # [N,3] float64, Morton order (configs with velocities)
    perm: np.ndarray        # [N] int32: Morton position -> generator index
    cells: np.ndarray       # [n_cell,4] int32 (first_ptcl, n_ptcl, first_child, n_child), level order
    geom: np.ndarray        # [n_cell,4] float64 (centre xyz, side) -- builder geometry, not uploaded
    level: np.ndarray       # [n_cell] int32
    level_first: np.ndarray  # [n_level+1] int32
    root: np.ndarray        # [4] float64 (centre xyz, side)
    grp_cell: np.ndarray    # [n_group] int32
    grp_first: np.ndarray   # [n_group] int32
    grp_n: np.ndarray       # [n_group] int32
    epj_off: np.ndarray     # [n_group+1] int64
    epj_id: np.ndarray      # [E_epj] int32 particle indices
    spj_off: np.ndarray     # [n_group+1] int64
    spj_id: np.ndarray      # [E_spj] int32 cell indices
    theta: float
    sph: np.ndarray | None = None  # [N,4] float32 (h, u, 0, 0), Morton order: short-range workload (NEXT-4) only
    skin: float = 0.0              # neighbour lists were built with search radii 2 (1 + skin) h

    @property
    def n(self) -> int:
        return int(self.posm.shape[0])

    @property
    def n_cell(self) -> int:
        return int(self.cells.shape[0])

    @property
    def n_group(self) -> int:
        return int(self.grp_first.shape[0])

    @property
    def n_list(self) -> np.ndarray:
        return (np.diff(self.epj_off) + np.diff(self.spj_off)).astype(np.int64)

    @property
    def n_entry(self) -> int:
        return int(self.epj_off[-1] + self.spj_off[-1])

    @property
    def interactions(self) -> int:
        """I = sum_g n_i(g) * n_list(g): the paper's n<n_list>."""
        return int(np.sum(self.grp_n.astype(np.int64) * self.n_list))


def build_tree_and_lists(posm: np.ndarray, n_leaf: int, n_grp: int, theta: float, cfg: Config | None = None,
                         vel: np.ndarray | None = None, sph: np.ndarray | None = None, skin: float = 0.0) -> Workload:
    """sph ([N,4] float32 (h, u, ., .) in the caller's order) switches the list walk to the short-range neighbour
    search (reading S24): EPJ lists only, search radii 2 (1 + skin) h; theta is then ignored."""
    lib = _load()
    posm = np.ascontiguousarray(posm, dtype=np.float32)
    n = posm.shape[0]
    if sph is not None:
        sph = np.ascontiguousarray(sph, dtype=np.float32)
        if sph.shape != (n, 4):
            raise ValueError("sph must be [N,4]")
    h = lib.bh_build(n, _p(posm), int(n_leaf), int(n_grp))
    if not h:
        raise ValueError("bh_build rejected its arguments")
    try:
        n_cell, n_group, n_level = lib.bh_n_cell(h), lib.bh_n_group(h), lib.bh_n_level(h)
        perm = np.empty(n, np.int32)
        cells = np.empty((n_cell, 4), np.int32)
        geom = np.empty((n_cell, 4), np.float64)
        level = np.empty(n_cell, np.int32)
        level_first = np.empty(n_level + 1, np.int32)
        root = np.empty(4, np.float64)
        lib.bh_get_tree(h, _p(perm), _p(cells), _p(geom), _p(level), _p(level_first), _p(root))
        grp_cell = np.empty(n_group, np.int32)
        grp_first = np.empty(n_group, np.int32)
        grp_n = np.empty(n_group, np.int32)
        lib.bh_get_groups(h, _p(grp_cell), _p(grp_first), _p(grp_n))
        epj_off = np.empty(n_group + 1, np.int64)
        spj_off = np.empty(n_group + 1, np.int64)
        e_epj, e_spj = ctypes.c_int64(0), ctypes.c_int64(0)
        if sph is None:
            rc = lib.bh_build_lists(h, float(theta), _p(epj_off), _p(spj_off), ctypes.byref(e_epj), ctypes.byref(e_spj))
        else:
            hsml = np.ascontiguousarray(sph[:, 0])
            rc = lib.bh_build_neighbour_lists(h, _p(hsml), float(skin), _p(epj_off), _p(spj_off), ctypes.byref(e_epj))
        if rc != 0:
            raise ValueError("bh_build_lists failed")
        epj_id = np.empty(e_epj.value, np.int32)
        spj_id = np.empty(e_spj.value, np.int32)
        lib.bh_get_lists(h, _p(epj_id), _p(spj_id))
    finally:
        lib.bh_free(h)
    return Workload(cfg=cfg, posm=np.ascontiguousarray(posm[perm]), vel=None if vel is None else np.ascontiguousarray(vel[perm]),
                    perm=perm, cells=cells, geom=geom, level=level, level_first=level_first, root=root,
                    grp_cell=grp_cell, grp_first=grp_first, grp_n=grp_n,
                    epj_off=epj_off, epj_id=epj_id, spj_off=spj_off, spj_id=spj_id, theta=float(theta),
                    sph=None if sph is None else np.ascontiguousarray(sph[perm]), skin=float(skin))


def pack_data_lists(w: Workload, g0: int, g1: int, posm: np.ndarray, spj: np.ndarray, out: np.ndarray | None = None):
    """Method G1's host-side packing (Fig. 2): the j RECORDS of groups [g0, g1) -- EPJ from posm [N,4], then SPJ
    from spj [n_cell,4] (the monopoles as the device refresh made them) -- gathered into one contiguous float32 [E,4] array
    (out, e.g. a pinned buffer viewed as numpy) plus the int64 run offsets.  Returns (records, joff)."""
    lib = _load()
    n_e = int(w.epj_off[g1] - w.epj_off[g0] + w.spj_off[g1] - w.spj_off[g0])
    if out is None:
        out = np.empty((max(1, n_e), 4), np.float32)
    if out.shape[0] < n_e or out.dtype != np.float32 or not out.flags.c_contiguous:
        raise ValueError("out must be a C-contiguous float32 [>= %d, 4] array" % n_e)
    posm = np.ascontiguousarray(posm, dtype=np.float32)
    spj = np.ascontiguousarray(spj, dtype=np.float32)
    joff = np.empty(g1 - g0 + 1, np.int64)
    lib.bh_pack_data_lists(int(g0), int(g1), _p(posm), _p(spj), _p(w.epj_off), _p(w.epj_id), _p(w.spj_off), _p(w.spj_id), _p(out), _p(joff))
    return out[:n_e], joff


def make_workload(cfg: Config, n: int | None = None, theta: float | None = None) -> Workload:
    """Generate a config's particles and build its tree, groups and lists (construction step)."""
    posm, vel = make_particles(cfg, n)
    sph = make_sph_fields(cfg, posm) if cfg.kind.startswith("sph_") else None
    return build_tree_and_lists(posm, cfg.n_leaf, cfg.n_grp, cfg.theta if theta is None else theta, cfg=cfg, vel=vel,
                                sph=sph, skin=cfg.skin)
