"""ctypes loader for the CPU oracle (oracle/vd_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It never imports the CUDA package and the CUDA package never imports it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "vd_oracle.cpp")
_LIB = os.path.join(_HERE, "libvd_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with g++ -O2 (no intrinsics, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O2", "-std=c++14", "-fPIC", "-shared", "-pthread", "-ffp-contract=off",
               _SRC, "-o", _LIB]
        subprocess.check_call(cmd)
    return _LIB


class _Result(ctypes.Structure):
    _fields_ = [
        ("ns", ctypes.c_int64), ("dim", ctypes.c_int), ("nfl", ctypes.c_int),
        ("n_pieces", ctypes.c_int64), ("n_verts", ctypes.c_int64), ("n_nbrs", ctypes.c_int64),
        ("measure", ctypes.POINTER(ctypes.c_double)),
        ("centroid", ctypes.POINTER(ctypes.c_double)),
        ("nbr_off", ctypes.POINTER(ctypes.c_int64)),
        ("nbr", ctypes.POINTER(ctypes.c_int32)),
        ("piece_off", ctypes.POINTER(ctypes.c_int64)),
        ("piece_simplex", ctypes.POINTER(ctypes.c_int32)),
        ("piece_measure", ctypes.POINTER(ctypes.c_double)),
        ("vert_off", ctypes.POINTER(ctypes.c_int64)),
        ("vert_xyz", ctypes.POINTER(ctypes.c_double)),
        ("vert_flags", ctypes.POINTER(ctypes.c_int32)),
        ("simplex_adj", ctypes.POINTER(ctypes.c_int32)),
        ("threads_used", ctypes.c_int),
    ]


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
        _lib.vdo_compute_x.restype = ctypes.c_int
        _lib.vdo_compute_x.argtypes = [
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_void_p, ctypes.c_int64,
            ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_void_p, ctypes.c_int64,
            ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.POINTER(_Result))]
        _lib.vdo_free.restype = None
        _lib.vdo_free.argtypes = [ctypes.POINTER(_Result)]
    return _lib


@dataclass
class Cells:
    """Same CSR shape as include/vd.h's vd_cells, on the host, for `ids` (site ids, in order)."""
    ids: np.ndarray
    dim: int
    nfl: int
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
    simplex_adj: np.ndarray
    threads_used: int

    def neighbours(self, s):
        return self.nbr[self.nbr_off[s]:self.nbr_off[s + 1]]

    def pieces(self, s):
        return range(int(self.piece_off[s]), int(self.piece_off[s + 1]))

    def piece_verts(self, p):
        a, b = int(self.vert_off[p]), int(self.vert_off[p + 1])
        return self.vert_xyz[a:b], self.vert_flags[a:b]


def _arr(ptr, count, dtype, shape=None):
    if count == 0:
        out = np.zeros(0, dtype=dtype)
    else:
        out = np.ctypeslib.as_array(ptr, shape=(count,)).astype(dtype, copy=True)
    return out.reshape(shape) if shape is not None else out


def compute(sites, verts, simplices, kind, subset=None, tier="A", threads=0, weights=None, dissolve=False) -> Cells:
    """Clipped / restricted Voronoi cells by the definition (Eq. 1).

    tier 'A' = literal (all j != i); 'B' = two-phase (box facets, then simplices); see the
    header of vd_oracle.cpp.  subset = site ids to compute (default all).  weights [n]: the power diagram
    (section VII-C) instead of the Voronoi diagram.  dissolve (tets, convex domain): cells that do not reach
    the domain boundary come as ONE piece with simplex id m -- the whole Voronoi cell.
    """
    lib = _load()
    sites = np.ascontiguousarray(sites, dtype=np.float64)
    verts = np.ascontiguousarray(verts, dtype=np.float64)
    n, dim = sites.shape
    nv = verts.shape[0]
    if int(kind) in (3, 4):   # simple domain: verts = (lo, hi), one piece
        simplices = np.zeros((1, 0), dtype=np.int32)
    simplices = np.ascontiguousarray(simplices, dtype=np.int32)
    m, nc = simplices.shape
    if subset is not None:
        subset = np.ascontiguousarray(subset, dtype=np.int64)
        sp, ns = subset.ctypes.data, subset.shape[0]
        ids = subset.copy()
    else:
        sp, ns = None, 0
        ids = np.arange(n, dtype=np.int64)
    res = ctypes.POINTER(_Result)()
    if weights is not None:
        weights = np.ascontiguousarray(weights, dtype=np.float64)
        assert weights.shape == (n,)
    rc = lib.vdo_compute_x(sites.ctypes.data, weights.ctypes.data if weights is not None else None, n, dim, verts.ctypes.data, nv, simplices.ctypes.data if simplices.size else None, m,
                         int(kind), sp, ns, 1 if tier == "B" else 0, int(threads), 1 if dissolve else 0, ctypes.byref(res))
    if rc != 0:
        raise RuntimeError(f"vdo_compute failed with status {rc}")
    r = res.contents
    k = int(r.ns)
    npc, nvt, nnb = int(r.n_pieces), int(r.n_verts), int(r.n_nbrs)
    out = Cells(
        ids=ids, dim=int(r.dim), nfl=int(r.nfl),
        measure=_arr(r.measure, k, np.float64),
        centroid=_arr(r.centroid, k * dim, np.float64, (k, dim)),
        nbr_off=_arr(r.nbr_off, k + 1, np.int64),
        nbr=_arr(r.nbr, nnb, np.int32),
        piece_off=_arr(r.piece_off, k + 1, np.int64),
        piece_simplex=_arr(r.piece_simplex, npc, np.int32),
        piece_measure=_arr(r.piece_measure, npc, np.float64),
        vert_off=_arr(r.vert_off, npc + 1, np.int64),
        vert_xyz=_arr(r.vert_xyz, nvt * dim, np.float64, (nvt, dim)),
        vert_flags=_arr(r.vert_flags, nvt * int(r.nfl), np.int32, (nvt, int(r.nfl))),
        simplex_adj=_arr(r.simplex_adj, m * nc, np.int32, (m, nc)),
        threads_used=int(r.threads_used),
    )
    lib.vdo_free(res)
    return out
