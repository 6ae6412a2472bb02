"""Power diagrams by lifting (paper section VII-C).

The power cell of a weighted site (v_i, w_i) is {x : |x - v_i|^2 - w_i <= |x - v_j|^2 - w_j for all j}.  The paper
computes it as a restricted Voronoi diagram one dimension up: lift every site to p_i = (v_i, sqrt(eta - w_i)) with
eta >= max w (it advises the smallest eta) and restrict the Voronoi diagram of the lifted
sites to the domain embedded at height 0 -- there |x - p_i|^2 = |x - v_i|^2 + eta - w_i, so the restricted cells
are the power cells.  For 2D weighted sites that is a VD_TRI_SURFACE problem, which the library already solves:
these helpers only marshal the inputs (no kernel here; every step of the path still runs in libvd.so).
"""
from __future__ import annotations

import numpy as np


def lift_sites(sites2d: np.ndarray, weights: np.ndarray, eta: float | None = None) -> np.ndarray:
    """[n][2] sites and [n] weights -> [n][3] lifted sites p_i = (v_i, sqrt(eta - w_i)); eta defaults to max w."""
    s = np.ascontiguousarray(sites2d, np.float64)
    w = np.ascontiguousarray(weights, np.float64)
    if s.ndim != 2 or s.shape[1] != 2 or w.shape != (s.shape[0],):
        raise ValueError("lift_sites: sites [n][2] and weights [n] expected")
    if eta is None:
        eta = float(w.max())
    if eta < w.max():
        raise ValueError("lift_sites: eta must be >= max weight (P:L471)")
    return np.concatenate([s, np.sqrt(eta - w)[:, None]], axis=1)


def embed_domain(verts2d: np.ndarray) -> np.ndarray:
    """[nv][2] mesh vertices -> [nv][3] at height 0 (the flat surface the lifted diagram is restricted to)."""
    v = np.ascontiguousarray(verts2d, np.float64)
    return np.concatenate([v, np.zeros((v.shape[0], 1))], axis=1)


def power_cells(sites2d, weights, verts2d, triangles, eta=None, **options):
    """Power diagram of weighted 2D sites clipped to a triangulated 2D domain: one vd_create / vd_set_domain
    (VD_TRI_SURFACE) / vd_compute on the lifted sites.  Returns binding.HostCells (areas, centroids with z = 0,
    neighbour lists, pieces per triangle)."""
    from . import binding
    return binding.compute(lift_sites(sites2d, weights, eta), embed_domain(verts2d), np.ascontiguousarray(triangles, np.int32),
                           1, **options)
