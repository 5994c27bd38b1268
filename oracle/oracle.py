"""ctypes front end of oracle/mwf_oracle.c (fp64 CPU oracle; test infrastructure only)."""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mwf_oracle.c")
_SRC_SPH = os.path.join(_HERE, "sph_oracle.c")
_SO = os.path.join(_HERE, "libmwf_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc -O2 -fopenmp (no fast-math, no intrinsics)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC_SPH)):
        r = subprocess.run(["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", "-o", _SO, _SRC, _SRC_SPH, "-lm"],
                           capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError("oracle build failed:\n" + r.stderr)
    return _SO


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        vp, i64, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double
        lib.orc_num_threads.restype = ctypes.c_int
        lib.orc_set_num_threads.argtypes = [ctypes.c_int]
        lib.orc_monopoles.argtypes = [i64, vp, vp, vp]
        lib.orc_forces.argtypes = [i64, vp, vp, vp, vp, vp, vp, vp, vp, vp, dbl, dbl, vp, vp]
        lib.orc_direct.argtypes = [i64, vp, dbl, dbl, vp, vp]
        lib.orc_quadrupoles.argtypes = [i64, vp, vp, vp, vp]
        lib.orc_forces_quad.argtypes = [i64, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, dbl, dbl, vp, vp]
        lib.orc_kick_drift.argtypes = [i64, vp, vp, vp, dbl, vp, vp]
        lib.orc_kick.argtypes = [i64, vp, vp, dbl, vp]
        lib.orc_sph_w.restype = dbl
        lib.orc_sph_w.argtypes = [dbl, dbl]
        lib.orc_sph_dwdr.restype = dbl
        lib.orc_sph_dwdr.argtypes = [dbl, dbl]
        lib.orc_sph_density.argtypes = [i64, vp, vp, vp, vp, vp, vp, vp, dbl, vp, vp]
        lib.orc_sph_density_direct.argtypes = [i64, vp, vp, vp]
        lib.orc_sph_hydro.argtypes = [i64, vp, vp, vp, vp, vp, vp, vp, vp, vp]
        lib.orc_sph_hydro_direct.argtypes = [i64, vp, vp, vp, vp]
        _lib = lib
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def num_threads() -> int:
    return int(_load().orc_num_threads())


def set_num_threads(n: int) -> None:
    _load().orc_set_num_threads(int(n))


def _c(a, dt):
    a = np.ascontiguousarray(a, dtype=dt)
    return a


def monopoles(cells: np.ndarray, posm: np.ndarray) -> np.ndarray:
    """[n_cell,4] float64 (X_c xyz, M_c) from the fp32 particle array."""
    cells = _c(cells, np.int32)
    posm = _c(posm, np.float32)
    mom = np.empty((cells.shape[0], 4), np.float64)
    _load().orc_monopoles(cells.shape[0], _p(cells), _p(posm), _p(mom))
    return mom


def quadrupoles(cells: np.ndarray, posm: np.ndarray, mom: np.ndarray) -> np.ndarray:
    """[n_cell,6] float64 (Qxx, Qyy, Qzz, Qxy, Qxz, Qyz): second moments about the centres of mass in `mom`."""
    cells = _c(cells, np.int32)
    posm = _c(posm, np.float32)
    mom = _c(mom, np.float64)
    quad = np.empty((cells.shape[0], 6), np.float64)
    _load().orc_quadrupoles(cells.shape[0], _p(cells), _p(posm), _p(mom), _p(quad))
    return quad


def forces(posm, mom, grp_first, grp_n, epj_off, epj_id, spj_off, spj_id, eps: float, G: float = 1.0, groups=None, quad=None):
    """acc [N,3], pot [N] in float64 for the selected groups (all when `groups` is None); particles of
    other groups are left NaN.  quad (from `quadrupoles`): SPJ entries act through monopole and quadrupole."""
    posm = _c(posm, np.float32)
    mom = _c(mom, np.float64)
    grp_first, grp_n = _c(grp_first, np.int32), _c(grp_n, np.int32)
    epj_off, spj_off = _c(epj_off, np.int64), _c(spj_off, np.int64)
    epj_id, spj_id = _c(epj_id, np.int32), _c(spj_id, np.int32)
    n = posm.shape[0]
    acc = np.full((n, 3), np.nan)
    pot = np.full(n, np.nan)
    if groups is None:
        n_sel, sel = grp_first.shape[0], None
    else:
        sel = _c(groups, np.int64)
        n_sel = sel.shape[0]
    if quad is not None:
        quad = _c(quad, np.float64)
        _load().orc_forces_quad(n_sel, _p(sel), _p(grp_first), _p(grp_n), _p(epj_off), _p(epj_id), _p(spj_off), _p(spj_id),
                                _p(posm), _p(mom), _p(quad), float(eps), float(G), _p(acc), _p(pot))
        return acc, pot
    _load().orc_forces(n_sel, _p(sel), _p(grp_first), _p(grp_n), _p(epj_off), _p(epj_id), _p(spj_off), _p(spj_id),
                       _p(posm), _p(mom), float(eps), float(G), _p(acc), _p(pot))
    return acc, pot


def direct(posm, eps: float, G: float = 1.0):
    """Plain O(N^2) direct summation: acc [N,3], pot [N] float64."""
    posm = _c(posm, np.float32)
    n = posm.shape[0]
    acc = np.empty((n, 3))
    pot = np.empty(n)
    _load().orc_direct(n, _p(posm), float(eps), float(G), _p(acc), _p(pot))
    return acc, pot


def kick_drift(posm, vel4, accp4, dt: float):
    """Leapfrog kick-drift in fp64 from fp32 state: returns (x[N,3], v[N,3]) with v = v + a dt/2, x = x + v dt."""
    posm, vel4, accp4 = _c(posm, np.float32), _c(vel4, np.float32), _c(accp4, np.float32)
    n = posm.shape[0]
    x, v = np.empty((n, 3)), np.empty((n, 3))
    _load().orc_kick_drift(n, _p(posm), _p(vel4), _p(accp4), float(dt), _p(x), _p(v))
    return x, v


def kick(vel4, accp4, dt: float):
    """Closing half kick in fp64 from fp32 state: v[N,3] = v + a dt/2."""
    vel4, accp4 = _c(vel4, np.float32), _c(accp4, np.float32)
    n = vel4.shape[0]
    v = np.empty((n, 3))
    _load().orc_kick(n, _p(vel4), _p(accp4), float(dt), _p(v))
    return v


# ---- short-range workload (NEXT-4): SPH density and pressure-gradient acceleration, oracle/sph_oracle.c

def sph_w(r: float, h: float) -> float:
    """Cubic-spline kernel W(r, h) in 3-D, support 2h."""
    return float(_load().orc_sph_w(float(r), float(h)))


def sph_dwdr(r: float, h: float) -> float:
    return float(_load().orc_sph_dwdr(float(r), float(h)))


def _sel(groups, grp_first):
    if groups is None:
        return grp_first.shape[0], None
    sel = _c(groups, np.int64)
    return sel.shape[0], sel


def sph_density(posm, sph4, grp_first, grp_n, epj_off, epj_id, gamma: float, groups=None):
    """rho [N], P/rho^2 [N] (float64) over the groups' neighbour lists; sph4 = [N,4] float32 (h, u, rho, P/rho^2),
    of which h and u are read.  Particles of unselected groups are NaN."""
    posm, sph4 = _c(posm, np.float32), _c(sph4, np.float32)
    grp_first, grp_n, epj_off, epj_id = _c(grp_first, np.int32), _c(grp_n, np.int32), _c(epj_off, np.int64), _c(epj_id, np.int32)
    n = posm.shape[0]
    rho, pr2 = np.full(n, np.nan), np.full(n, np.nan)
    n_sel, sel = _sel(groups, grp_first)
    _load().orc_sph_density(n_sel, _p(sel), _p(grp_first), _p(grp_n), _p(epj_off), _p(epj_id), _p(posm), _p(sph4), float(gamma), _p(rho), _p(pr2))
    return rho, pr2


def sph_density_direct(posm, sph4):
    posm, sph4 = _c(posm, np.float32), _c(sph4, np.float32)
    rho = np.empty(posm.shape[0])
    _load().orc_sph_density_direct(posm.shape[0], _p(posm), _p(sph4), _p(rho))
    return rho


def sph_hydro(posm, sph4, grp_first, grp_n, epj_off, epj_id, groups=None):
    """acc [N,3] and scale [N] (sum of the magnitudes of the pair terms) in float64; reads h and P/rho^2 of sph4."""
    posm, sph4 = _c(posm, np.float32), _c(sph4, np.float32)
    grp_first, grp_n, epj_off, epj_id = _c(grp_first, np.int32), _c(grp_n, np.int32), _c(epj_off, np.int64), _c(epj_id, np.int32)
    n = posm.shape[0]
    acc, scale = np.full((n, 3), np.nan), np.full(n, np.nan)
    n_sel, sel = _sel(groups, grp_first)
    _load().orc_sph_hydro(n_sel, _p(sel), _p(grp_first), _p(grp_n), _p(epj_off), _p(epj_id), _p(posm), _p(sph4), _p(acc), _p(scale))
    return acc, scale


def sph_hydro_direct(posm, sph4):
    posm, sph4 = _c(posm, np.float32), _c(sph4, np.float32)
    n = posm.shape[0]
    acc, scale = np.empty((n, 3)), np.empty(n)
    _load().orc_sph_hydro_direct(n, _p(posm), _p(sph4), _p(acc), _p(scale))
    return acc, scale
