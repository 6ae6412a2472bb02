"""Element-by-element comparison of the CUDA result with the oracle.

Both sides deliver the same CSR shape with pieces ordered by simplex id and the corners of a piece
ordered by their ascending flag tuple, so equal structure means equal arrays.
Tolerances (BASELINE.json north_star): neighbour sets, piece simplices, corner counts and corner
flags bit-exact; |Δmeasure| <= 1e-9 * measure; |Δcentroid| <= 1e-9 * max(|centroid|, diam);
|Δvertex| <= 1e-9 * diam.  `simplex_measure` ([m] array, or a scalar) switches on the rounding floor for sliver
cells: a cell whose measure is 1e-9 of a simplex is a difference of nearly equal corner coordinates, so
its measure carries an absolute error of about eps * |T_a| on either side; the floor is 64 * eps * the largest simplex
the cell touches -- nothing looser.
"""
from __future__ import annotations

import numpy as np

REL = 1e-9


def _match_ties(gx, ox, fl):
    """Corners with identical flag tuples (two faces of T_a on the domain boundary both carry ~m) have no
    defined relative order: match them by position inside each tie group (greedy nearest)."""
    worst = 0.0
    k = len(fl)
    c = 0
    while c < k:
        e = c + 1
        while e < k and np.array_equal(fl[e], fl[c]):
            e += 1
        free = list(range(c, e))
        for a in range(c, e):
            d = [float(np.abs(gx[a] - ox[b]).max()) for b in free]
            j = int(np.argmin(d))
            worst = max(worst, d[j])
            free.pop(j)
        c = e
    return worst


EPS = 2.220446049250313e-16


def compare(gpu, ora, diam, ids=None, tiny_measure=1e-12, abs_measure=0.0, simplex_measure=None):
    """gpu: binding.HostCells over all n sites; ora: oracle.Cells over `ora.ids`.
    Returns a dict of mismatch lists (empty lists = parity)."""
    ids = np.asarray(ora.ids if ids is None else ids, dtype=np.int64)
    bad = {"nbr": [], "pieces": [], "verts": [], "flags": [], "measure": [], "centroid": [], "xyz": [], "excused": []}
    max_xyz = 0.0
    max_meas = 0.0
    for s, i in enumerate(ids):
        gn = gpu.nbr[gpu.nbr_off[i]:gpu.nbr_off[i + 1]]
        on = ora.nbr[ora.nbr_off[s]:ora.nbr_off[s + 1]]
        gp0, gp1 = int(gpu.piece_off[i]), int(gpu.piece_off[i + 1])
        op0, op1 = int(ora.piece_off[s]), int(ora.piece_off[s + 1])
        gs, os_ = gpu.piece_simplex[gp0:gp1], ora.piece_simplex[op0:op1]
        structural = not np.array_equal(gn, on) or not np.array_equal(gs, os_)
        if not structural:
            gv = gpu.vert_off[gp0:gp1 + 1] - gpu.vert_off[gp0]
            ov = ora.vert_off[op0:op1 + 1] - ora.vert_off[op0]
            if not np.array_equal(gv, ov):
                structural = True
        if structural:
            # excusable only if the disputed pieces are near-degenerate (measure < 1e-12 of the cell's)
            gm = dict(zip(gs.tolist(), gpu.piece_measure[gp0:gp1].tolist()))
            om = dict(zip(os_.tolist(), ora.piece_measure[op0:op1].tolist()))
            disputed = [max(gm.get(a, 0.0), om.get(a, 0.0)) for a in set(gm) ^ set(om)]
            cellm = max(float(ora.measure[s]), 1e-300)
            if disputed and max(disputed) < tiny_measure * cellm:
                bad["excused"].append((int(i), max(disputed) / cellm))
            elif not np.array_equal(gn, on):
                bad["nbr"].append((int(i), gn.tolist(), on.tolist()))
            elif not np.array_equal(gs, os_):
                bad["pieces"].append((int(i), gs.tolist(), os_.tolist()))
            else:
                bad["verts"].append(int(i))
            continue
        a0, a1 = int(gpu.vert_off[gp0]), int(gpu.vert_off[gp1])
        b0, b1 = int(ora.vert_off[op0]), int(ora.vert_off[op1])
        if not np.array_equal(gpu.vert_flags[a0:a1], ora.vert_flags[b0:b1]):
            bad["flags"].append(int(i))
            continue
        if a1 > a0:
            dx = float(np.abs(gpu.vert_xyz[a0:a1] - ora.vert_xyz[b0:b1]).max())
            if dx > REL * diam:
                dx = _match_ties(gpu.vert_xyz[a0:a1], ora.vert_xyz[b0:b1], ora.vert_flags[b0:b1])
            max_xyz = max(max_xyz, dx)
            if dx > REL * diam:
                bad["xyz"].append((int(i), dx))
        m_o, m_g = float(ora.measure[s]), float(gpu.measure[i])
        if m_o > 0:
            max_meas = max(max_meas, abs(m_g - m_o) / m_o)
        floor = abs_measure
        if simplex_measure is not None and op1 > op0:
            sm = np.asarray(simplex_measure, dtype=np.float64)
            floor += 64.0 * EPS * float(sm[os_].max() if sm.ndim else sm)
        if abs(m_g - m_o) > REL * m_o + floor:
            bad["measure"].append((int(i), m_g, m_o))
        dc = float(np.linalg.norm(gpu.centroid[i] - ora.centroid[s]))
        if dc > REL * max(float(np.linalg.norm(ora.centroid[s])), diam):
            bad["centroid"].append((int(i), dc))
    bad["_max_xyz"] = max_xyz
    bad["_max_rel_measure"] = max_meas
    return bad


def assert_parity(gpu, ora, diam, ids=None, allow_excused=0, abs_measure=0.0, simplex_measure=None):
    bad = compare(gpu, ora, diam, ids, abs_measure=abs_measure, simplex_measure=simplex_measure)
    problems = {k: v for k, v in bad.items() if not k.startswith("_") and k != "excused" and v}
    assert not problems, {k: v[:5] for k, v in problems.items()}
    assert len(bad["excused"]) <= allow_excused, bad["excused"][:5]
    return bad


def simplex_measures(w):
    """|T_a| of every simplex of a meshed workload (plain determinant / cross-product formulas); |box| for box kinds."""
    if w.simplices is None:
        return np.float64(w.measure)
    p = w.verts[w.simplices]
    if w.kind == 0:
        e1, e2 = p[:, 1] - p[:, 0], p[:, 2] - p[:, 0]
        return np.abs(e1[:, 0] * e2[:, 1] - e1[:, 1] * e2[:, 0]) * 0.5
    if w.kind == 1:
        return np.linalg.norm(np.cross(p[:, 1] - p[:, 0], p[:, 2] - p[:, 0]), axis=1) * 0.5
    return np.abs(np.linalg.det(p[:, 1:] - p[:, :1])) / 6.0


def global_checks(gpu, w):
    """Invariants that hold at any size (used at full scale where the oracle only samples)."""
    out = {}
    out["sum_measure_rel"] = abs(float(gpu.measure.sum()) - w.measure) / w.measure
    per_simplex = np.bincount(gpu.piece_simplex, weights=gpu.piece_measure, minlength=w.m)
    p = w.verts[w.simplices]
    if w.kind == 0:
        e1, e2 = p[:, 1] - p[:, 0], p[:, 2] - p[:, 0]
        sm = np.abs(e1[:, 0] * e2[:, 1] - e1[:, 1] * e2[:, 0]) * 0.5
    elif w.kind == 1:
        sm = np.linalg.norm(np.cross(p[:, 1] - p[:, 0], p[:, 2] - p[:, 0]), axis=1) * 0.5
    else:
        sm = np.abs(np.linalg.det(p[:, 1:] - p[:, :1])) / 6.0
    out["per_simplex_rel"] = float(np.abs(per_simplex - sm).max() / sm.max())
    # neighbour symmetry through sorted (i, j) key lists
    owner = np.repeat(np.arange(gpu.n, dtype=np.int64), np.diff(gpu.nbr_off))
    fwd = owner * gpu.n + gpu.nbr.astype(np.int64)
    rev = gpu.nbr.astype(np.int64) * gpu.n + owner
    out["nbr_symmetric"] = bool(np.array_equal(np.sort(fwd), np.sort(rev)))
    return out
