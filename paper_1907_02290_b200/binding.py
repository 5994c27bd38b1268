"""Thin Python binding of the C-ABI CUDA library (include/mwf.h, csrc/libmwf.so).

Argument marshalling only: every step of the path runs in the library's kernels.  PyTorch supplies the
device arena, the streams and pinned host buffers; the calls carry the names of the C entry points
without the `mwf_` prefix.  There is no CPU fallback: a missing library or a non-CUDA environment raises.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from . import build as _build

MAKE_LIST, MAKE_LIST_FOR_REUSE, REUSE_LIST = 0, 1, 2
OK, EINVAL, ESTATE, ERANGE, ENOMEM, ECUDA = 0, -1, -2, -3, -4, -5
MAX_TAG = 16

# every symbol include/mwf.h declares (tests check that the library exports exactly these)
SYMBOLS = (
    "mwf_arena_bytes", "mwf_create", "mwf_destroy", "mwf_set_tag_stream", "mwf_set_particles", "mwf_get_particles",
    "mwf_set_tree", "mwf_set_lists", "mwf_begin_step", "mwf_refresh_monopoles", "mwf_dispatch", "mwf_retrieve",
    "mwf_calc_force_all", "mwf_get_monopoles", "mwf_device_pointers", "mwf_sync", "mwf_get_counters",
    "mwf_last_dispatch_ms", "mwf_strerror", "mwf_last_cuda_error",
    "mwf_set_velocities", "mwf_get_velocities", "mwf_kick_drift", "mwf_kick", "mwf_step_reuse",
    "mwf_reserve_data_lists", "mwf_dispatch_data", "mwf_set_spj_order", "mwf_get_quadrupoles",
    "mwf_set_sph", "mwf_get_sph", "mwf_dispatch_density", "mwf_dispatch_hydro", "mwf_calc_sph_all",
    "mwf_build", "mwf_build_neighbours", "mwf_get_build_sizes", "mwf_get_permutation", "mwf_get_tree", "mwf_get_groups", "mwf_get_lists", "mwf_get_list_buffer",
    "mwf_set_particles_next", "mwf_swap_store", "mwf_get_tag_split",
    "mwf_monopoles_static", "mwf_static_last_error", "mwf_get_run1_len",
)


class Params(ctypes.Structure):
    _fields_ = [("eps", ctypes.c_float), ("G", ctypes.c_float), ("max_ptcl", ctypes.c_int64), ("max_cell", ctypes.c_int64),
                ("max_group", ctypes.c_int64), ("max_entry", ctypes.c_int64), ("n_tag", ctypes.c_int32), ("device", ctypes.c_int32)]


class MwfError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__("mwf error %d: %s" % (code, text))
        self.code = code


_lib = None


def load_library(path: str | None = None) -> ctypes.CDLL:
    """dlopen csrc/libmwf.so (built in-tree by `build.build_mwf`) and declare the signatures."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    if path is None:
        path = os.environ.get("MWF_LIBRARY") or os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc", "libmwf.so")
        if not os.path.exists(path):
            path = _build.build_mwf()
    lib = ctypes.CDLL(path)
    vp, i64, i32, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_int
    P = ctypes.POINTER
    sig = {
        "mwf_arena_bytes": [P(Params), P(i64)],
        "mwf_create": [P(vp), P(Params), vp, i64],
        "mwf_destroy": [vp],
        "mwf_set_tag_stream": [vp, i32, vp],
        "mwf_set_particles": [vp, vp, i64, i64, ci, vp],
        "mwf_get_particles": [vp, vp, i64, i64, ci],
        "mwf_set_particles_next": [vp, vp, i64, i64, ci, vp],
        "mwf_swap_store": [vp, vp],
        "mwf_get_tag_split": [vp, P(i64)],
        "mwf_set_tree": [vp, vp, i64, vp],
        "mwf_set_lists": [vp, i64, vp, vp, vp, vp, vp, vp, ci, vp],
        "mwf_begin_step": [vp, ci],
        "mwf_refresh_monopoles": [vp, vp],
        "mwf_dispatch": [vp, i32, i64, i64],
        "mwf_retrieve": [vp, i32, vp, ci],
        "mwf_calc_force_all": [vp, vp, ci, vp, ci],
        "mwf_get_monopoles": [vp, vp, ci],
        "mwf_device_pointers": [vp, P(vp), P(vp)],
        "mwf_sync": [vp],
        "mwf_get_counters": [vp, P(i64), P(i64), P(i64)],
        "mwf_last_dispatch_ms": [vp, i32, P(ctypes.c_float)],
        "mwf_set_velocities": [vp, vp, i64, i64, ci, vp],
        "mwf_get_velocities": [vp, vp, i64, i64, ci],
        "mwf_kick_drift": [vp, ctypes.c_float, vp],
        "mwf_kick": [vp, ctypes.c_float, vp],
        "mwf_step_reuse": [vp, ctypes.c_float],
        "mwf_set_spj_order": [vp, ci],
        "mwf_get_quadrupoles": [vp, vp, ci],
        "mwf_reserve_data_lists": [vp, i64],
        "mwf_dispatch_data": [vp, i32, i64, i64, vp, vp, ci],
        "mwf_set_sph": [vp, vp, i64, i64, ci, vp],
        "mwf_get_sph": [vp, vp, i64, i64, ci],
        "mwf_dispatch_density": [vp, i32, i64, i64, ctypes.c_float],
        "mwf_dispatch_hydro": [vp, i32, i64, i64],
        "mwf_calc_sph_all": [vp, vp, ci, vp, ci, vp, ci, ctypes.c_float],
        "mwf_build": [vp, i64, i32, i32, ctypes.c_double, ci, vp],
        "mwf_build_neighbours": [vp, i64, i32, i32, ctypes.c_double, ci, vp],
        "mwf_get_build_sizes": [vp, P(i64), P(i64), P(i64), P(i64), P(i32)],
        "mwf_get_permutation": [vp, vp, ci],
        "mwf_get_tree": [vp, vp, vp],
        "mwf_get_groups": [vp, vp, vp],
        "mwf_get_lists": [vp, vp, vp, vp, vp],
        "mwf_get_list_buffer": [vp, vp, vp, P(i64), P(i64), ci],
        "mwf_monopoles_static": [vp, i64, vp, i64, vp, vp],
        "mwf_get_run1_len": [vp, vp, ci],
    }
    for name, args in sig.items():
        fn = getattr(lib, name)
        fn.argtypes = args
        fn.restype = ci
    lib.mwf_strerror.argtypes = [ci]
    lib.mwf_strerror.restype = ctypes.c_char_p
    lib.mwf_last_cuda_error.argtypes = [vp]
    lib.mwf_last_cuda_error.restype = ctypes.c_char_p
    lib.mwf_static_last_error.argtypes = []
    lib.mwf_static_last_error.restype = ctypes.c_char_p
    _lib = lib
    return lib


def _host_ptr(a: np.ndarray, dtype, what: str):
    if not isinstance(a, np.ndarray) or a.dtype != dtype or not a.flags.c_contiguous:
        raise TypeError("%s must be a C-contiguous numpy array of %s" % (what, np.dtype(dtype)))
    return ctypes.c_void_p(a.ctypes.data)


def _ptr(x, dtype, what: str):
    """(pointer, on_device) of a numpy array, a torch CPU tensor (e.g. pinned) or a torch CUDA tensor."""
    import torch
    if isinstance(x, np.ndarray):
        return _host_ptr(x, dtype, what), 0
    if isinstance(x, torch.Tensor):
        if not x.is_contiguous() or x.dtype != torch.float32:
            raise TypeError("%s must be a contiguous float32 tensor" % what)
        return ctypes.c_void_p(x.data_ptr()), 1 if x.is_cuda else 0
    raise TypeError("%s: unsupported buffer type %r" % (what, type(x)))


def _stream_handle(stream) -> ctypes.c_void_p:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return ctypes.c_void_p(int(stream.cuda_stream))


STATIC_MAX_CELL = 131072      # MWF_STATIC_MAX_CELL of include/mwf.h


def monopoles_static(cells, ptcl, spj, stream=None) -> None:
    """mwf_monopoles_static: the monopole record of every tree cell, for callers that may not allocate device memory.

    Meant for code that lives inside someone else's memory budget -- a plugin under a host application's pool, a step
    on a latency-bound path where cudaMalloc would stall the device, a job on a nearly full GPU -- and so cannot create
    a MultiWalkForce (whose arena has to be allocated by somebody).  Nothing is allocated here either: the three
    arguments are torch CUDA tensors the caller already owns (cells int32 (n_cell, 4), ptcl float32 (n_ptcl, 4), spj
    float32 (n_cell, 4), all contiguous, on the current device) and only their pointers are passed on.  The library's
    working memory is a fixed array in its image, good for at most STATIC_MAX_CELL cells; a larger tree raises MwfError
    (code ENOMEM) with the limit in its text.  Asynchronous on `stream` (default: torch's current stream).  Calls share
    that array: do not let two of them run on the same GPU at the same time.  The first call on a device also looks up
    the array's address; make it before starting a stream capture."""
    import torch
    lib = load_library()
    for t, dt, what in ((cells, torch.int32, "cells"), (ptcl, torch.float32, "ptcl"), (spj, torch.float32, "spj")):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == dt and t.dim() == 2 and t.shape[1] == 4):
            raise TypeError("%s must be a contiguous CUDA tensor of %s with shape (n, 4)" % (what, dt))
    if spj.shape[0] != cells.shape[0]:
        raise ValueError("spj needs one record per cell")
    rc = lib.mwf_monopoles_static(ctypes.c_void_p(cells.data_ptr()), cells.shape[0], ctypes.c_void_p(ptcl.data_ptr()), ptcl.shape[0],
                                  ctypes.c_void_p(spj.data_ptr()), _stream_handle(stream))
    if rc != 0:
        raise MwfError(rc, lib.mwf_static_last_error().decode() or lib.mwf_strerror(rc).decode())


class MultiWalkForce:
    """One mwf_ctx.  Device memory is one torch uint8 arena; tags run on torch streams."""

    def __init__(self, eps: float, G: float = 1.0, *, max_ptcl: int, max_cell: int, max_group: int, max_entry: int,
                 n_tag: int = 8, device: int = 0, tag_priorities: bool = True):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("MultiWalkForce needs a CUDA device (sm_100a); there is no CPU path")
        self._lib = load_library()
        self._torch = torch
        self.device = torch.device("cuda", device)
        self.params = Params(float(eps), float(G), int(max_ptcl), int(max_cell), int(max_group), int(max_entry), int(n_tag), int(device))
        nbytes = ctypes.c_int64(0)
        self._ck(self._lib.mwf_arena_bytes(ctypes.byref(self.params), ctypes.byref(nbytes)), ctx=False)
        self.arena_bytes = nbytes.value
        with torch.cuda.device(self.device):
            self._arena = torch.empty(self.arena_bytes + 256, dtype=torch.uint8, device=self.device)
            base = (self._arena.data_ptr() + 255) // 256 * 256
            self._h = ctypes.c_void_p(None)
            self._ck(self._lib.mwf_create(ctypes.byref(self._h), ctypes.byref(self.params), ctypes.c_void_p(base), self.arena_bytes), ctx=False)
            # priorities fall with the tag (the library does the same for its own streams): tags dispatched together
            # finish roughly in tag order, so a tag's retrieve overlaps the kernels of the tags behind it
            # (tag_priorities=False: equal priorities, for callers that cycle through the tags many times per step --
            # the batched multiwalk pipeline -- where the oldest batch, not the lowest tag, should finish first)
            least, greatest = torch.cuda.Stream.priority_range()
            levels = least - greatest + 1
            self.streams = [torch.cuda.Stream(device=self.device, priority=(greatest + t * levels // n_tag) if tag_priorities else least)
                            for t in range(n_tag)]
        for t, s in enumerate(self.streams):
            self._ck(self._lib.mwf_set_tag_stream(self._h, t, ctypes.c_void_p(int(s.cuda_stream))))
        self.n_tag = n_tag

    @classmethod
    def for_workload(cls, w, eps: float | None = None, G: float = 1.0, n_tag: int = 8, device: int = 0, tag_priorities: bool = True):
        if eps is None:
            eps = w.cfg.eps if w.cfg.eps > 0 else 1.0   # short-range workloads have no softening; the ctx still wants one
        return cls(eps, G, max_ptcl=w.n, max_cell=w.n_cell, max_group=w.n_group,
                   max_entry=max(1, w.n_entry), n_tag=n_tag, device=device, tag_priorities=tag_priorities)

    # -- error handling
    def _ck(self, rc: int, ctx: bool = True):
        if rc != 0:
            text = self._lib.mwf_strerror(rc).decode()
            if rc == ECUDA and ctx and self._h:
                text += " (" + self._lib.mwf_last_cuda_error(self._h).decode() + ")"
            raise MwfError(rc, text)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.mwf_destroy(self._h)
            self._h = None
            self._arena = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C entry points, same names
    def set_particles(self, src, first: int = 0, n: int | None = None, stream=None):
        p, on_dev = _ptr(src, np.float32, "src")
        if n is None:
            n = int(src.shape[0])
        self._ck(self._lib.mwf_set_particles(self._h, p, int(first), int(n), on_dev, _stream_handle(stream)))

    def set_particles_next(self, src, first: int = 0, n: int | None = None, stream=None):
        """Particles [first, first + n) of the NEXT step into the shadow store (pipelined host loop)."""
        p, on_dev = _ptr(src, np.float32, "src")
        if n is None:
            n = int(src.shape[0])
        self._ck(self._lib.mwf_set_particles_next(self._h, p, int(first), int(n), on_dev, _stream_handle(stream)))

    def swap_store(self, stream=None):
        self._ck(self._lib.mwf_swap_store(self._h, _stream_handle(stream)))

    def get_tag_split(self) -> np.ndarray:
        out = np.zeros(self.n_tag + 1, np.int64)
        self._ck(self._lib.mwf_get_tag_split(self._h, out.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))))
        return out

    def get_particles(self, first: int, n: int) -> np.ndarray:
        out = np.empty((n, 4), np.float32)
        self._ck(self._lib.mwf_get_particles(self._h, _host_ptr(out, np.float32, "dst"), int(first), int(n), 0))
        return out

    def set_tree(self, cells: np.ndarray, stream=None):
        self._ck(self._lib.mwf_set_tree(self._h, _host_ptr(cells, np.int32, "cells"), int(cells.shape[0]), _stream_handle(stream)))

    def set_lists(self, grp_first, grp_n, epj_off, epj_id, spj_off, spj_id, mode: int = MAKE_LIST_FOR_REUSE, stream=None):
        self._ck(self._lib.mwf_set_lists(
            self._h, int(grp_first.shape[0]), _host_ptr(grp_first, np.int32, "grp_first"), _host_ptr(grp_n, np.int32, "grp_n"),
            _host_ptr(epj_off, np.int64, "epj_off"), _host_ptr(epj_id, np.int32, "epj_id"),
            _host_ptr(spj_off, np.int64, "spj_off"), _host_ptr(spj_id, np.int32, "spj_id"), int(mode), _stream_handle(stream)))

    def begin_step(self, mode: int):
        self._ck(self._lib.mwf_begin_step(self._h, int(mode)))

    def refresh_monopoles(self, stream=None):
        self._ck(self._lib.mwf_refresh_monopoles(self._h, _stream_handle(stream)))

    def dispatch(self, tag: int, g_begin: int, g_end: int):
        self._ck(self._lib.mwf_dispatch(self._h, int(tag), int(g_begin), int(g_end)))

    def set_spj_order(self, order: int):
        self._ck(self._lib.mwf_set_spj_order(self._h, int(order)))

    def get_quadrupoles(self, n_cell: int) -> np.ndarray:
        out = np.empty((n_cell, 8), np.float32)
        self._ck(self._lib.mwf_get_quadrupoles(self._h, _host_ptr(out, np.float32, "dst"), 0))
        return out

    def reserve_data_lists(self, max_entry_per_tag: int):
        self._ck(self._lib.mwf_reserve_data_lists(self._h, int(max_entry_per_tag)))

    def dispatch_data(self, tag: int, g_begin: int, g_end: int, jdata, joff: np.ndarray):
        """Method G1: jdata = [n,4] float32 j records (numpy, pinned torch CPU tensor or CUDA tensor), joff = int64 offsets."""
        p, on_dev = _ptr(jdata, np.float32, "jdata")
        self._ck(self._lib.mwf_dispatch_data(self._h, int(tag), int(g_begin), int(g_end), p, _host_ptr(joff, np.int64, "joff"), on_dev))

    def retrieve(self, tag: int, dst):
        if dst is None:
            p, on_dev = ctypes.c_void_p(None), 0
        else:
            p, on_dev = _ptr(dst, np.float32, "dst")
        self._ck(self._lib.mwf_retrieve(self._h, int(tag), p, on_dev))

    def calc_force_all(self, src, dst):
        if src is None:
            sp, s_dev = ctypes.c_void_p(None), 0
        else:
            sp, s_dev = _ptr(src, np.float32, "src")
        dp, d_dev = _ptr(dst, np.float32, "dst")
        self._ck(self._lib.mwf_calc_force_all(self._h, sp, s_dev, dp, d_dev))

    def set_velocities(self, src, first: int = 0, n: int | None = None, stream=None):
        p, on_dev = _ptr(src, np.float32, "src")
        if n is None:
            n = int(src.shape[0])
        self._ck(self._lib.mwf_set_velocities(self._h, p, int(first), int(n), on_dev, _stream_handle(stream)))

    def get_velocities(self, first: int, n: int) -> np.ndarray:
        out = np.empty((n, 4), np.float32)
        self._ck(self._lib.mwf_get_velocities(self._h, _host_ptr(out, np.float32, "dst"), int(first), int(n), 0))
        return out

    def kick_drift(self, dt: float, stream=None):
        self._ck(self._lib.mwf_kick_drift(self._h, float(dt), _stream_handle(stream)))

    def kick(self, dt: float, stream=None):
        self._ck(self._lib.mwf_kick(self._h, float(dt), _stream_handle(stream)))

    def step_reuse(self, dt: float):
        self._ck(self._lib.mwf_step_reuse(self._h, float(dt)))

    def set_sph(self, src, first: int = 0, n: int | None = None, stream=None):
        """Short-range workload: [n,4] float32 records (h, u, rho, P/rho^2)."""
        p, on_dev = _ptr(src, np.float32, "src")
        if n is None:
            n = int(src.shape[0])
        self._ck(self._lib.mwf_set_sph(self._h, p, int(first), int(n), on_dev, _stream_handle(stream)))

    def get_sph(self, first: int, n: int) -> np.ndarray:
        out = np.empty((n, 4), np.float32)
        self._ck(self._lib.mwf_get_sph(self._h, _host_ptr(out, np.float32, "dst"), int(first), int(n), 0))
        return out

    def dispatch_density(self, tag: int, g_begin: int, g_end: int, gamma: float):
        self._ck(self._lib.mwf_dispatch_density(self._h, int(tag), int(g_begin), int(g_end), float(gamma)))

    def dispatch_hydro(self, tag: int, g_begin: int, g_end: int):
        self._ck(self._lib.mwf_dispatch_hydro(self._h, int(tag), int(g_begin), int(g_end)))

    def build(self, n: int, n_leaf: int, n_grp: int, theta: float, mode: int = MAKE_LIST_FOR_REUSE, stream=None):
        self._ck(self._lib.mwf_build(self._h, int(n), int(n_leaf), int(n_grp), float(theta), int(mode), _stream_handle(stream)))

    def calc_sph_all(self, src, rec, dst, gamma: float):
        """One whole short-range evaluation: rec (h, u in; rho, P/rho^2 out) and dst (ax, ay, az, 0) are [N,4] float32."""
        if src is None:
            sp, s_dev = ctypes.c_void_p(None), 0
        else:
            sp, s_dev = _ptr(src, np.float32, "src")
        rp, r_dev = _ptr(rec, np.float32, "rec")
        dp, d_dev = _ptr(dst, np.float32, "dst")
        self._ck(self._lib.mwf_calc_sph_all(self._h, sp, s_dev, rp, r_dev, dp, d_dev, float(gamma)))

    def build_neighbours(self, n: int, n_leaf: int, n_grp: int, skin: float, mode: int = MAKE_LIST_FOR_REUSE, stream=None):
        self._ck(self._lib.mwf_build_neighbours(self._h, int(n), int(n_leaf), int(n_grp), float(skin), int(mode), _stream_handle(stream)))

    def get_build_sizes(self):
        a, b, c, d = (ctypes.c_int64(0) for _ in range(4))
        e = ctypes.c_int32(0)
        self._ck(self._lib.mwf_get_build_sizes(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c), ctypes.byref(d), ctypes.byref(e)))
        return dict(n_cell=a.value, n_group=b.value, n_epj=c.value, n_spj=d.value, n_level=e.value)

    def get_permutation(self, n: int) -> np.ndarray:
        out = np.empty(n, np.int32)
        self._ck(self._lib.mwf_get_permutation(self._h, _host_ptr(out, np.int32, "perm"), 0))
        return out

    def get_tree(self, n_cell: int, with_geom: bool = True):
        cells = np.empty((n_cell, 4), np.int32)
        geom = np.empty((n_cell, 4), np.float64) if with_geom else None
        self._ck(self._lib.mwf_get_tree(self._h, _host_ptr(cells, np.int32, "cells"),
                                        _host_ptr(geom, np.float64, "geom") if with_geom else ctypes.c_void_p(None)))
        return cells, geom

    def get_groups(self, n_group: int):
        gf, gn = np.empty(n_group, np.int32), np.empty(n_group, np.int32)
        self._ck(self._lib.mwf_get_groups(self._h, _host_ptr(gf, np.int32, "grp_first"), _host_ptr(gn, np.int32, "grp_n")))
        return gf, gn

    def get_lists(self, n_group: int, n_epj: int, n_spj: int):
        eo, so = np.empty(n_group + 1, np.int64), np.empty(n_group + 1, np.int64)
        ei, si = np.empty(max(1, n_epj), np.int32), np.empty(max(1, n_spj), np.int32)
        self._ck(self._lib.mwf_get_lists(self._h, _host_ptr(eo, np.int64, "epj_off"), _host_ptr(ei, np.int32, "epj_id"),
                                         _host_ptr(so, np.int64, "spj_off"), _host_ptr(si, np.int32, "spj_id")))
        return eo, ei[:n_epj], so, si[:n_spj]

    def get_list_buffer(self, on_device: bool = False):
        """(list_off, list) as the force kernel reads them: numpy arrays, or torch CUDA tensors when on_device."""
        g, n = ctypes.c_int64(0), ctypes.c_int64(0)
        self._ck(self._lib.mwf_get_list_buffer(self._h, None, None, ctypes.byref(g), ctypes.byref(n), 0))
        if on_device:
            t = self._torch
            off = t.empty(g.value + 1, dtype=t.int64, device=self.device)
            lst = t.empty(max(1, n.value), dtype=t.int32, device=self.device)
            self._ck(self._lib.mwf_get_list_buffer(self._h, ctypes.c_void_p(off.data_ptr()), ctypes.c_void_p(lst.data_ptr()), None, None, 1))
            return off, lst[:n.value]
        off, lst = np.empty(g.value + 1, np.int64), np.empty(max(1, n.value), np.int32)
        self._ck(self._lib.mwf_get_list_buffer(self._h, _host_ptr(off, np.int64, "list_off"), _host_ptr(lst, np.int32, "list"), None, None, 0))
        return off, lst[:n.value]

    def get_run1_len(self) -> np.ndarray:
        """Per group: EPJ + far SPJ entries (run 1 of its merged list); the near SPJ entries are the rest of the list."""
        g = ctypes.c_int64(0)
        self._ck(self._lib.mwf_get_list_buffer(self._h, None, None, ctypes.byref(g), None, 0))
        out = np.empty(g.value, np.int32)
        self._ck(self._lib.mwf_get_run1_len(self._h, _host_ptr(out, np.int32, "run1_len"), 0))
        return out

    def get_monopoles(self, n_cell: int) -> np.ndarray:
        out = np.empty((n_cell, 4), np.float32)
        self._ck(self._lib.mwf_get_monopoles(self._h, _host_ptr(out, np.float32, "dst"), 0))
        return out

    def sync(self):
        self._ck(self._lib.mwf_sync(self._h))

    def get_counters(self):
        a, b, c = ctypes.c_int64(0), ctypes.c_int64(0), ctypes.c_int64(0)
        self._ck(self._lib.mwf_get_counters(self._h, ctypes.byref(a), ctypes.byref(b), ctypes.byref(c)))
        return dict(kernel_launches=a.value, interactions=b.value, padded_entries=c.value)

    def last_dispatch_ms(self, tag: int) -> float:
        ms = ctypes.c_float(0)
        self._ck(self._lib.mwf_last_dispatch_ms(self._h, int(tag), ctypes.byref(ms)))
        return float(ms.value)

    # -- marshalling helpers (no arithmetic)
    def upload_workload(self, w, mode: int = MAKE_LIST_FOR_REUSE, stream=None):
        """Construction step: particles, tree and lists of a `workload.Workload`."""
        self.begin_step(mode)
        self.set_particles(w.posm, 0, w.n, stream)
        self.set_tree(w.cells, stream)
        self.set_lists(w.grp_first, w.grp_n, w.epj_off, w.epj_id, w.spj_off, w.spj_id, mode, stream)
        if getattr(w, "sph", None) is not None:
            self.set_sph(w.sph, 0, w.n, stream)

    def pinned(self, n: int):
        """Pinned host float32 [n,4] buffer (for truly asynchronous uploads / retrieves)."""
        return self._torch.empty((n, 4), dtype=self._torch.float32, pin_memory=True)
