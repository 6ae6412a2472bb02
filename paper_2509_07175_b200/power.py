"""Power diagrams (paper section VII-C): marshalling only.

The power cell of a weighted site (v_i, w_i) is {x : |x - v_i|^2 - w_i <= |x - v_j|^2 - w_j for all j}.  The paper
computes it as a restricted Voronoi diagram one dimension up: every site is lifted to p_i = (v_i, sqrt(eta - w_i)),
eta >= max w (it advises the smallest eta), and the Voronoi diagram of the lifted sites is restricted
to the domain at height 0.  The lifting happens inside the library (vd_create_weighted, kernels k_weight_max / k_lift);
this helper only hands the arrays over.
"""
from __future__ import annotations

import numpy as np


def power_cells(sites, weights, verts, simplices, kind=0, eta=None, **options):
    """Power diagram of weighted sites clipped to a domain: vd_create_weighted / vd_set_domain / vd_compute.
    kind: VD_TRI_2D (2-D sites) or VD_TET_3D / VD_BOX_3D (3-D sites).  Returns binding.HostCells."""
    from . import binding
    with binding.Context(np.ascontiguousarray(sites, np.float64), weights=np.ascontiguousarray(weights, np.float64), eta=eta) as ctx:
        if options:
            ctx.set_options(**options)
        ctx.set_domain(verts, simplices, kind)
        ctx.compute()
        return ctx.to_host()
