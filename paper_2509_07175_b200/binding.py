"""Thin ctypes binding of libvd.so (include/vd.h): argument marshalling only.

Every step of the hot path runs inside the CUDA library; this module converts numpy / torch
arguments to pointers and copies results back on request.  There is no CPU fallback: if
libvd.so is missing, cannot be loaded, or finds no CUDA device, the calls raise.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import numpy as np

from . import build as _build

VD_TRI_2D, VD_TRI_SURFACE, VD_TET_3D, VD_BOX_2D, VD_BOX_3D = 0, 1, 2, 3, 4
STATUS = {0: "VD_OK", 1: "VD_E_ARG", 2: "VD_E_DIM", 3: "VD_E_STATE", 4: "VD_E_INPUT", 5: "VD_E_CUDA",
          6: "VD_E_NOMEM", 7: "VD_E_CAPACITY", 8: "VD_E_NOCONVERGE"}
EXPORTS = ["vd_create", "vd_create_weighted", "vd_partial_moments", "vd_finish_centroids", "vd_update_sites", "vd_lloyd", "vd_set_domain", "vd_compute", "vd_destroy", "vd_set_stream",
           "vd_set_allocator", "vd_set_options", "vd_get_counters", "vd_get_stage_ms", "vd_get_phase_ms", "vd_get_phase_counters", "vd_cells_to_host",
           "vd_nearest", "vd_nearest_static", "vd_get_adjacency", "vd_dfma_peak", "vd_last_error", "vd_version"]

_LIB_PATH = _build.lib_path()
_lib = None


class VdError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


class vd_cells(ctypes.Structure):
    _fields_ = [("n", ctypes.c_int64), ("dim", ctypes.c_int32), ("nfl", ctypes.c_int32),
                ("n_nonempty", ctypes.c_int64), ("n_pieces", ctypes.c_int64), ("n_verts", ctypes.c_int64),
                ("n_nbrs", ctypes.c_int64),
                ("measure", ctypes.c_void_p), ("centroid", ctypes.c_void_p), ("nbr_off", ctypes.c_void_p),
                ("nbr", ctypes.c_void_p), ("piece_off", ctypes.c_void_p), ("piece_simplex", ctypes.c_void_p),
                ("piece_measure", ctypes.c_void_p), ("vert_off", ctypes.c_void_p), ("vert_xyz", ctypes.c_void_p),
                ("vert_flags", ctypes.c_void_p)]


class vd_options(ctypes.Structure):
    _fields_ = [("grid_density", ctypes.c_double), ("ball_cells", ctypes.c_int32), ("real_edges", ctypes.c_int32),
                ("persistent", ctypes.c_int32), ("pair_capacity", ctypes.c_int64), ("vert_capacity", ctypes.c_int64),
                ("near_clips", ctypes.c_int32), ("simplex_begin", ctypes.c_int32), ("simplex_end", ctypes.c_int32),
                ("tail_pairs", ctypes.c_int32), ("first_clip", ctypes.c_int32),
                ("seed_corners", ctypes.c_int32), ("small_wave", ctypes.c_int32), ("step_out", ctypes.c_int32),
                ("dissolve", ctypes.c_int32), ("fp32_filter", ctypes.c_int32), ("count_alg", ctypes.c_int32),
                ("reuse_nbrs", ctypes.c_int32), ("rounds", ctypes.c_int32), ("reserved", ctypes.c_int32 * 2)]


class vd_counters(ctypes.Structure):
    _fields_ = [(k, ctypes.c_int64) for k in ("pairs", "pieces", "queries", "dist_evals", "search_iters", "clips",
                                               "waves", "overflow_pairs", "reruns", "launches", "row_evals", "search_evals", "pre_clips",
                                               "clip_corners", "new_corners", "fan_simplices", "alg_evals", "syncs", "step_probes", "f32_survivors")] + [("reserved", ctypes.c_int64 * 1)]


def load():
    """Load libvd.so (raises if it is missing: build it with __graft_entry__.build())."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise RuntimeError(f"{_LIB_PATH} not found: the CUDA library is not built (python -m paper_2509_07175_b200.build)")
    lib = ctypes.CDLL(_LIB_PATH)
    vp, i64, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
    lib.vd_create.argtypes = [vp, i64, ci, ctypes.POINTER(vp)]
    lib.vd_create_weighted.argtypes = [vp, vp, i64, ci, ctypes.c_double, ctypes.POINTER(vp)]
    lib.vd_partial_moments.argtypes = [vp, vp]
    lib.vd_finish_centroids.argtypes = [vp, vp]
    lib.vd_update_sites.argtypes = [vp, vp]
    lib.vd_lloyd.argtypes = [vp, ci, ctypes.POINTER(vd_cells), vp]
    lib.vd_set_domain.argtypes = [vp, vp, i64, vp, i64, ci]
    lib.vd_compute.argtypes = [vp, ctypes.POINTER(vd_cells)]
    lib.vd_destroy.argtypes = [vp]
    lib.vd_destroy.restype = None
    lib.vd_set_stream.argtypes = [vp, vp]
    lib.vd_set_allocator.argtypes = [vp, vp, vp, vp]
    lib.vd_set_options.argtypes = [vp, ctypes.POINTER(vd_options)]
    lib.vd_get_counters.argtypes = [vp, ctypes.POINTER(vd_counters)]
    lib.vd_get_stage_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_double)]
    lib.vd_get_phase_ms.argtypes = [vp, ctypes.POINTER(ctypes.c_double)]
    lib.vd_get_phase_counters.argtypes = [vp, ci, ctypes.POINTER(vd_counters)]
    lib.vd_cells_to_host.argtypes = [vp] + [vp] * 10
    lib.vd_nearest.argtypes = [vp, vp, i64, vp]
    lib.vd_nearest_static.argtypes = [vp, vp, i64, vp]
    lib.vd_get_adjacency.argtypes = [vp, vp]
    lib.vd_dfma_peak.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    lib.vd_last_error.argtypes = [vp]
    lib.vd_last_error.restype = ctypes.c_char_p
    lib.vd_version.restype = ctypes.c_char_p
    for name in EXPORTS:
        if getattr(lib, name).restype is ctypes.c_int and name not in ("vd_destroy",):
            getattr(lib, name).restype = ctypes.c_int
    _lib = lib
    return lib


def _ptr(x, dtype):
    """(pointer, keepalive) of a numpy array (host) or a torch tensor (host or CUDA)."""
    if isinstance(x, np.ndarray):
        a = np.ascontiguousarray(x, dtype=dtype)
        return a.ctypes.data, a
    if hasattr(x, "data_ptr"):  # torch tensor
        import torch
        want = {np.float64: torch.float64, np.int32: torch.int32}[dtype]
        t = x.contiguous()
        if t.dtype != want:
            t = t.to(want)
        return t.data_ptr(), t
    a = np.ascontiguousarray(np.asarray(x), dtype=dtype)
    return a.ctypes.data, a


_pinned = {}


def _staging(name, shape, dtype, pinned):
    """Host array for a result; pinned=True: a view of a cached page-locked buffer (grown on demand, reused by
    later calls: the arrays of the previous pinned result are overwritten), so that the copy runs at PCIe speed."""
    if not pinned:
        return np.empty(shape, dtype)
    import torch
    count = int(np.prod(shape))
    nbytes = max(1, count * np.dtype(dtype).itemsize)
    buf = _pinned.get(name)
    if buf is None or buf.numel() < nbytes:
        buf = torch.empty(int(nbytes * 1.25) + 4096, dtype=torch.uint8, pin_memory=True)
        _pinned[name] = buf
    return buf.numpy()[:count * np.dtype(dtype).itemsize].view(dtype).reshape(shape)


@dataclass
class HostCells:
    """Result of vd_compute copied to the host (same CSR arrays as include/vd.h's vd_cells)."""
    n: int
    dim: int
    nfl: int
    n_nonempty: int
    measure: np.ndarray
    centroid: np.ndarray
    nbr_off: np.ndarray
    nbr: np.ndarray
    piece_off: np.ndarray
    piece_simplex: np.ndarray
    piece_measure: np.ndarray
    vert_off: np.ndarray
    vert_xyz: np.ndarray
    vert_flags: np.ndarray

    def neighbours(self, i):
        return self.nbr[self.nbr_off[i]:self.nbr_off[i + 1]]

    def pieces(self, i):
        return range(int(self.piece_off[i]), int(self.piece_off[i + 1]))

    def piece_verts(self, p):
        a, b = int(self.vert_off[p]), int(self.vert_off[p + 1])
        return self.vert_xyz[a:b], self.vert_flags[a:b]


class Context:
    """vd_ctx wrapper: vd_create / vd_set_domain / vd_compute / vd_destroy."""

    def __init__(self, sites, dim=None, weights=None, eta=None):
        """weights given: vd_create_weighted (power diagram); eta None = the smallest admissible (max w)."""
        self._lib = load()
        self._h = ctypes.c_void_p()
        shape = tuple(sites.shape)
        self.n, self.dim = int(shape[0]), int(shape[1] if dim is None else dim)
        p, keep = _ptr(sites, np.float64)
        if weights is None:
            self._check(self._lib.vd_create(p, self.n, self.dim, ctypes.byref(self._h)), create=True)
        else:
            pw, keepw = _ptr(weights, np.float64)
            self._check(self._lib.vd_create_weighted(p, pw, self.n, self.dim, float("nan") if eta is None else float(eta),
                                                     ctypes.byref(self._h)), create=True)
        self._callbacks = None
        self.cells = vd_cells()
        self.kind = None
        self.m = 0
        self.nc = 0

    def _check(self, rc, create=False):
        if rc != 0:
            msg = "" if create else (self._lib.vd_last_error(self._h) or b"").decode()
            if create and rc == 5:
                msg = "no CUDA device (this library has no CPU fallback)"
            raise VdError(rc, msg)

    def set_stream(self, cuda_stream: int):
        self._check(self._lib.vd_set_stream(self._h, ctypes.c_void_p(cuda_stream)))

    def set_allocator(self, alloc, release):
        """vd_set_allocator with Python callables alloc(nbytes, stream) -> device pointer (int), release(ptr)."""
        A = ctypes.CFUNCTYPE(ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p, ctypes.c_void_p)
        R = ctypes.CFUNCTYPE(None, ctypes.c_void_p, ctypes.c_void_p)
        a = A(lambda nbytes, user, stream: alloc(int(nbytes), int(stream or 0)))
        r = R(lambda ptr, user: release(int(ptr or 0)))
        self._callbacks = (a, r)   # keep the thunks alive as long as the context
        self._check(self._lib.vd_set_allocator(self._h, ctypes.cast(a, ctypes.c_void_p), ctypes.cast(r, ctypes.c_void_p), None))

    def partial_moments(self, out_ptr: int):
        """vd_partial_moments into a caller-owned device buffer [n][1 + dim] (e.g. a torch tensor's data_ptr())."""
        self._check(self._lib.vd_partial_moments(self._h, ctypes.c_void_p(out_ptr)))

    def finish_centroids(self, sums_ptr: int):
        self._check(self._lib.vd_finish_centroids(self._h, ctypes.c_void_p(sums_ptr)))

    def set_options(self, **kw):
        o = vd_options()
        o.real_edges = 1
        o.persistent = 1
        for k, v in kw.items():
            setattr(o, k, v)
        self._check(self._lib.vd_set_options(self._h, ctypes.byref(o)))

    def update_sites(self, sites):
        p, keep = _ptr(sites, np.float64)
        self._check(self._lib.vd_update_sites(self._h, p))

    def set_domain(self, verts, simplices, kind):
        """verts [nv][dim], simplices [m][3|4]; for VD_BOX_2D / VD_BOX_3D verts = (lo, hi) and simplices is None."""
        pv, k1 = _ptr(verts, np.float64)
        if int(kind) in (VD_BOX_2D, VD_BOX_3D):
            ps, self.m, self.nc = None, 1, 4 if int(kind) == VD_BOX_2D else 8
        else:
            ps, k2 = _ptr(simplices, np.int32)
            self.m, self.nc = int(simplices.shape[0]), int(simplices.shape[1])
        self.kind = int(kind)
        self._check(self._lib.vd_set_domain(self._h, pv, int(verts.shape[0]), ps, self.m, int(kind)))

    def compute(self) -> vd_cells:
        self._check(self._lib.vd_compute(self._h, ctypes.byref(self.cells)))
        return self.cells

    def device_tensors(self):
        """(measure [n], centroid [n][dim]) as torch tensors that VIEW the context's device buffers (no copy; valid
        until the next compute): what the ranks hand to the all-reduce of the sharded path (ranks.combine_partial_cells)."""
        import torch

        class _View:
            def __init__(self, ptr, shape):
                self.__cuda_array_interface__ = {"shape": shape, "typestr": "<f8", "data": (int(ptr), False), "version": 2}

        r = self.cells
        n, dim = int(r.n), int(r.dim)
        dev = torch.device("cuda", torch.cuda.current_device())
        return (torch.as_tensor(_View(r.measure, (n,)), device=dev), torch.as_tensor(_View(r.centroid, (n, dim)), device=dev))

    def lloyd(self, iterations: int) -> np.ndarray:
        """vd_lloyd: returns the final sites [n][dim]; self.cells describes them."""
        out = np.empty((self.n, self.dim), np.float64)
        self._check(self._lib.vd_lloyd(self._h, int(iterations), ctypes.byref(self.cells), out.ctypes.data))
        return out

    def counters(self) -> dict:
        c = vd_counters()
        self._check(self._lib.vd_get_counters(self._h, ctypes.byref(c)))
        return {k: int(getattr(c, k)) for k, _ in vd_counters._fields_ if k != "reserved"}

    def phase_counters(self) -> dict:
        """vd_get_phase_counters: {kernel: counters} for init / verify / fix / finish / tail / other."""
        out = {}
        for k, name in enumerate(("init", "verify", "fix", "finish", "tail", "other")):
            c = vd_counters()
            self._check(self._lib.vd_get_phase_counters(self._h, k, ctypes.byref(c)))
            out[name] = {f: int(getattr(c, f)) for f, _ in vd_counters._fields_ if f != "reserved"}
        return out

    def stage_ms(self):
        a = (ctypes.c_double * 5)()
        self._check(self._lib.vd_get_stage_ms(self._h, a))
        return dict(zip(("index", "seed", "clip", "assemble", "total"), [float(x) for x in a]))

    def phase_ms(self):
        a = (ctypes.c_double * 5)()
        self._check(self._lib.vd_get_phase_ms(self._h, a))
        return dict(zip(("init", "verify", "fix", "finish", "tail"), [float(x) for x in a]))

    def to_host(self, full=True, pinned=False) -> HostCells:
        """vd_cells_to_host into fresh numpy arrays, or (pinned=True) into cached page-locked staging buffers."""
        r = self.cells
        n, dim, nfl = int(r.n), int(r.dim), int(r.nfl)
        npc, nvt, nnb = int(r.n_pieces), int(r.n_verts), int(r.n_nbrs)
        E = lambda name, shape, dt: _staging(name, shape, dt, pinned)
        out = HostCells(
            n=n, dim=dim, nfl=nfl, n_nonempty=int(r.n_nonempty),
            measure=E("measure", (n,), np.float64), centroid=E("centroid", (n, dim), np.float64),
            nbr_off=E("nbr_off", (n + 1,), np.int64), nbr=E("nbr", (nnb,), np.int32),
            piece_off=E("piece_off", (n + 1,), np.int64), piece_simplex=E("piece_simplex", (npc,), np.int32),
            piece_measure=E("piece_measure", (npc,), np.float64), vert_off=E("vert_off", (npc + 1,), np.int64),
            vert_xyz=E("vert_xyz", (nvt, dim), np.float64) if full else np.empty((0, dim), np.float64),
            vert_flags=E("vert_flags", (nvt, nfl), np.int32) if full else np.empty((0, nfl), np.int32))
        d = lambda a: a.ctypes.data if a.size else None
        self._check(self._lib.vd_cells_to_host(
            self._h, d(out.measure), d(out.centroid), d(out.nbr_off), d(out.nbr), d(out.piece_off),
            d(out.piece_simplex), d(out.piece_measure), d(out.vert_off),
            d(out.vert_xyz) if full else None, d(out.vert_flags) if full else None))
        return out

    def nearest(self, queries) -> np.ndarray:
        q = np.ascontiguousarray(queries, dtype=np.float64)
        out = np.empty(q.shape[0], np.int32)
        self._check(self._lib.vd_nearest(self._h, q.ctypes.data, q.shape[0], out.ctypes.data))
        return out

    def nearest_static(self, queries, out=None):
        """vd_nearest_static: no device allocation (at most 65536 queries; the index must exist).  queries / out: numpy
        arrays or torch tensors (host or CUDA); out (int32 [nq]) is created as a numpy array when not given."""
        pq, keep = _ptr(queries, np.float64)
        nq = int(queries.shape[0])
        if out is None:
            out = np.empty(nq, np.int32)
        po = out.data_ptr() if hasattr(out, "data_ptr") else out.ctypes.data
        self._check(self._lib.vd_nearest_static(self._h, pq, nq, po))
        return out

    def adjacency(self) -> np.ndarray:
        out = np.empty((self.m, self.nc), np.int32)
        self._check(self._lib.vd_get_adjacency(self._h, out.ctypes.data))
        return out

    def destroy(self):
        if self._h:
            self._lib.vd_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.destroy()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def fp64_peak(stream=None) -> tuple[float, float]:
    """vd_dfma_peak: (TFLOP/s, ms) of the dependent-FMA-chain kernel on the current device."""
    t, ms = ctypes.c_double(0.0), ctypes.c_double(0.0)
    st = load().vd_dfma_peak(ctypes.c_void_p(stream or 0), ctypes.byref(t), ctypes.byref(ms))
    if st != 0:
        raise VdError(st, "vd_dfma_peak")
    return float(t.value), float(ms.value)


def compute(sites, verts, simplices, kind, **options) -> HostCells:
    """One-shot: vd_create -> vd_set_domain -> vd_compute -> copy to host -> vd_destroy."""
    with Context(sites) as ctx:
        if options:
            ctx.set_options(**options)
        ctx.set_domain(verts, simplices, kind)
        ctx.compute()
        return ctx.to_host()
