"""Pins of the CPU oracle against what the paper's definition and the mathematics fix.

The paper prints no worked numeric example, so the pins are: hand-worked closed forms
(tests/golden/unit_square_cases.json), regular grids, global invariants (sum of measures,
first-moment identity, per-simplex conservation, neighbour symmetry), brute-force
equidistance / no-nearer-site of every output corner (Eq. 1), Qhull
(scipy.spatial) Voronoi volumes / Delaunay neighbours / circumcentres for interior cells,
and tier A == tier B.  None of these re-types the oracle's own formulas.
"""
import json
import os

import numpy as np
import pytest

from oracle import oracle
from paper_2509_07175_b200 import inputs

HERE = os.path.dirname(os.path.abspath(__file__))


def _mesh_centroid(w):
    p = w.verts[w.simplices]
    c = p.mean(axis=1)
    if w.kind == inputs.KIND_TRI_2D:
        e1, e2 = p[:, 1] - p[:, 0], p[:, 2] - p[:, 0]
        a = np.abs(e1[:, 0] * e2[:, 1] - e1[:, 1] * e2[:, 0]) * 0.5
    elif w.kind == inputs.KIND_TRI_SURFACE:
        a = np.linalg.norm(np.cross(p[:, 1] - p[:, 0], p[:, 2] - p[:, 0]), axis=1) * 0.5
    else:
        a = np.abs(np.linalg.det(p[:, 1:] - p[:, :1])) / 6.0
    return a, (a[:, None] * c).sum(0)


def _check_invariants(w, c, corner_sample=4000, seed=0):
    """Invariants that hold for any correct answer, none using the oracle's code."""
    n = w.n
    simplex_measure, first_moment = _mesh_centroid(w)
    # (1) cells partition the domain
    assert abs(c.measure.sum() - w.measure) <= 1e-11 * w.measure
    # (2) first moments add up to the domain's
    mom = (c.measure[:, None] * c.centroid).sum(0)
    assert np.abs(mom - first_moment).max() <= 1e-11 * max(1.0, np.abs(first_moment).max())
    # (3) pieces partition every simplex
    per_simplex = np.bincount(c.piece_simplex, weights=c.piece_measure, minlength=w.m)
    assert np.abs(per_simplex - simplex_measure).max() <= 1e-11 * simplex_measure.max()
    # (4) neighbour symmetry
    pairs = set()
    for i in range(n):
        for j in c.neighbours(i):
            pairs.add((i, int(j)))
    for (i, j) in pairs:
        assert (j, i) in pairs, f"neighbour relation not symmetric: {i}->{j}"
    # (5) every corner is equidistant from its cell's site and from the sites in its label, and
    #     no site is nearer (brute force over all n) -- Eq. 1
    rng = np.random.default_rng(seed)
    owner = np.repeat(np.repeat(np.arange(n), np.diff(c.piece_off)), np.diff(c.vert_off))
    nvt = c.vert_xyz.shape[0]
    pick = rng.choice(nvt, size=min(corner_sample, nvt), replace=False)
    scale = w.diameter
    for v in pick:
        x = c.vert_xyz[v]
        d = np.linalg.norm(w.sites - x, axis=1)
        di = d[owner[v]]
        assert di <= d.min() + 1e-10 * scale
        for fl in c.vert_flags[v]:
            if fl >= 0:
                assert abs(d[fl] - di) <= 1e-10 * scale
    # (6) 3D pieces are simple polytopes: V = 2F - 4 with F = number of distinct labels
    if w.kind == inputs.KIND_TET_3D:
        for p in range(len(c.piece_simplex)):
            xyz, fl = c.piece_verts(p)
            if (fl == ~w.m).any():
                continue  # two boundary faces of one tet share the label ~m: F is not countable from labels
            F = len(np.unique(fl))
            assert xyz.shape[0] == 2 * F - 4
    # (7) negative flags name the face T_a really shares with that simplex / the domain boundary
    assert _check_negative_flags(w, c) > 0


def _check_negative_flags(w, c):
    """Negative flags (Fig. 2a; 0-based restatement U3): a corner flagged ~b, b < m, lies on the face / edge
    that T_a really SHARES with T_b (the two simplices have exactly d vertices in common, and the corner lies in
    their affine hull); a corner flagged ~m lies on a face of T_a that no other simplex owns, i.e. on the domain
    boundary.  The mesh topology used here is recomputed from `simplices` with numpy (sorted face rows, np.unique),
    not taken from the oracle.  Returns how many (corner, flag) incidences were checked."""
    simp = np.asarray(w.simplices)
    m, nc = simp.shape
    d = nc - 1                                   # vertices of a face (tets: 3) or an edge (triangles: 2)
    tol = 1e-12 * w.diameter
    V = w.verts
    # owners of every face: face k of simplex a = its vertices without local corner k
    faces = np.stack([np.sort(np.delete(simp, k, axis=1), axis=1) for k in range(nc)], axis=1)   # [m, nc, d]
    _, inv, counts = np.unique(faces.reshape(-1, d), axis=0, return_inverse=True, return_counts=True)
    owners = counts[inv].reshape(m, nc)          # 1 = boundary face, 2 = interior face
    assert owners.max() <= 2

    def dist_to_hull(x, P):
        """distance from points x [k, dim] to the affine hull of P [k, d, dim] (a plane through 3 points in R^3, a
        line through 2 points in R^2 or R^3)"""
        e = P[:, 1:] - P[:, :1]
        r = x - P[:, 0]
        if d == 3:
            n = np.cross(e[:, 0], e[:, 1])
            return np.abs((r * n).sum(1)) / np.linalg.norm(n, axis=1)
        t = (r * e[:, 0]).sum(1) / (e[:, 0] ** 2).sum(1)
        return np.linalg.norm(r - t[:, None] * e[:, 0], axis=1)

    a_of_corner = np.repeat(c.piece_simplex, np.diff(c.vert_off))
    checked = 0
    for col in range(c.vert_flags.shape[1]):
        fl = c.vert_flags[:, col]
        neg = np.nonzero(fl < 0)[0]
        b = ~fl[neg]
        a = a_of_corner[neg]
        x = c.vert_xyz[neg]
        inner = b < m
        # ---- ~b, b < m: the face is shared, and the corner lies on it
        ai, bi, xi = a[inner], b[inner], x[inner]
        common = (simp[ai][:, :, None] == simp[bi][:, None, :]).any(2)          # [k, nc] vertex of a also in b
        assert (common.sum(1) == d).all(), "flag ~b names a simplex that does not share a face with T_a"
        P = V[simp[ai]][common].reshape(len(ai), d, V.shape[1])
        assert dist_to_hull(xi, P).max(initial=0.0) <= tol, "corner flagged ~b is not on the face T_a shares with T_b"
        checked += len(ai)
        # ---- ~m: on a boundary face of T_a
        ab, xb = a[~inner], x[~inner]
        assert (b[~inner] == m).all()
        best = np.full(len(ab), np.inf)
        for k in range(nc):
            on_bd = owners[ab, k] == 1
            if on_bd.any():
                P = V[np.delete(simp[ab[on_bd]], k, axis=1)]
                best[on_bd] = np.minimum(best[on_bd], dist_to_hull(xb[on_bd], P))
        assert best.max(initial=0.0) <= tol, "corner flagged ~m is not on the domain boundary"
        checked += len(ab)
    # ---- converse: a corner that lies on face k of T_a carries that face's flag (~other owner, or ~m)
    order = np.argsort(inv, kind="stable")
    flat_owner = np.repeat(np.arange(m), nc)[order]
    other = np.full(m * nc, m, dtype=np.int64)
    first = np.nonzero(np.diff(np.concatenate([[-1], inv[order]])) != 0)[0]
    for s, cnt in zip(first, counts):
        if cnt == 2:
            other[order[s]], other[order[s + 1]] = flat_owner[s + 1], flat_owner[s]
    other = other.reshape(m, nc)
    for k in range(nc):
        P = V[np.delete(simp[a_of_corner], k, axis=1)]
        on = dist_to_hull(c.vert_xyz, P) <= tol
        want = ~other[a_of_corner[on], k]
        assert (c.vert_flags[on] == want[:, None]).any(1).all(), "corner on a face of T_a lacks that face's flag"
        checked += int(on.sum())
    return checked


# ---------------------------------------------------------------------- golden hand cases
def test_golden_unit_square_cases():
    with open(os.path.join(HERE, "golden", "unit_square_cases.json")) as f:
        cases = json.load(f)["cases"]
    v, t = inputs.unit_square_mesh()
    for case in cases:
        s = np.array(case["sites"], dtype=np.float64)
        c = oracle.compute(s, v, t, inputs.KIND_TRI_2D)
        assert np.allclose(c.measure, case["area"], rtol=0, atol=1e-12)
        for i, cen in enumerate(case["centroid"]):
            if cen is not None:
                assert np.allclose(c.centroid[i], cen, rtol=0, atol=1e-12)
        for i, nb in enumerate(case["nbr"]):
            assert c.neighbours(i).tolist() == nb
        if case["pieces"] is not None:
            for i, pcs in enumerate(case["pieces"]):
                got = [[int(c.piece_simplex[p]), int(c.vert_off[p + 1] - c.vert_off[p])] for p in c.pieces(i)]
                assert got == pcs


def test_three_site_voronoi_vertex_and_flags():
    # sites (0.5,0.2),(0.2,0.8),(0.8,0.8): the Voronoi vertex is (0.5, 0.575) by hand.
    v, t = inputs.unit_square_mesh()
    s = np.array([[0.5, 0.2], [0.2, 0.8], [0.8, 0.8]])
    c = oracle.compute(s, v, t, inputs.KIND_TRI_2D)
    hits = 0
    for vtx, fl in zip(c.vert_xyz, c.vert_flags):
        if fl[0] >= 0 and fl[1] >= 0:
            assert np.allclose(vtx, [0.5, 0.575], atol=1e-14)
            hits += 1
    assert hits == 3  # one per cell
    # boundary flags: ~flag == m (=2) on the square's sides, ~flag == other triangle on the diagonal
    assert set(np.unique(c.vert_flags[c.vert_flags < 0]).tolist()) <= {~0, ~1, ~2}
    assert c.simplex_adj.tolist() == [[2, 1, 2], [2, 2, 0]]


def test_two_sites_in_cube():
    # bisector x = 1/2: two half cubes, centroids (1/4,1/2,1/2), (3/4,1/2,1/2)
    v, t = inputs.cube_kuhn_mesh(1)
    s = np.array([[0.25, 0.5, 0.5], [0.75, 0.5, 0.5]])
    c = oracle.compute(s, v, t, inputs.KIND_TET_3D)
    assert np.allclose(c.measure, [0.5, 0.5], atol=1e-15)
    assert np.allclose(c.centroid, s, atol=1e-15)
    assert c.neighbours(0).tolist() == [1] and c.neighbours(1).tolist() == [0]


@pytest.mark.parametrize("dim,k", [(2, 4), (3, 3)])
def test_regular_grid_equal_cells(dim, k):
    # degenerate (cocircular / cospherical) input: only measure and centroid are unique
    s = inputs.grid_sites(k, dim)
    if dim == 2:
        v, t = inputs.unit_square_mesh()
        kind = inputs.KIND_TRI_2D
    else:
        v, t = inputs.cube_kuhn_mesh(2)
        kind = inputs.KIND_TET_3D
    c = oracle.compute(s, v, t, kind)
    assert np.allclose(c.measure, 1.0 / k ** dim, rtol=0, atol=1e-14)
    assert np.allclose(c.centroid, s, rtol=0, atol=1e-13)
    # face-adjacent sites must be neighbours
    for i in range(len(s)):
        d = np.abs(s - s[i]).sum(1)
        face_adj = set(np.nonzero(np.isclose(d, 1.0 / k))[0].tolist())
        assert face_adj <= set(c.neighbours(i).tolist())


# ---------------------------------------------------------------------- invariants, full C1 + replicas
def test_c1_full_invariants():
    w = inputs.config(1)
    c = oracle.compute(w.sites, w.verts, w.simplices, w.kind)
    _check_invariants(w, c)
    assert (c.measure > 0).all()


@pytest.mark.parametrize("idx", [2, 3, 4, 5])
def test_replica_invariants(idx):
    w = inputs.config(idx, "small")
    c = oracle.compute(w.sites, w.verts, w.simplices, w.kind)
    _check_invariants(w, c, corner_sample=1500)


@pytest.mark.parametrize("idx", [1, 2, 3, 5])
def test_tier_b_equals_tier_a(idx):
    w = inputs.config(idx, "small")
    rng = np.random.default_rng(10 + idx)
    sub = np.sort(rng.choice(w.n, size=min(w.n, 300), replace=False))
    a = oracle.compute(w.sites, w.verts, w.simplices, w.kind, subset=sub, tier="A")
    b = oracle.compute(w.sites, w.verts, w.simplices, w.kind, subset=sub, tier="B")
    assert np.array_equal(a.piece_off, b.piece_off)
    assert np.array_equal(a.piece_simplex, b.piece_simplex)
    assert np.array_equal(a.vert_off, b.vert_off)
    assert np.array_equal(a.vert_flags, b.vert_flags)
    assert np.array_equal(a.nbr_off, b.nbr_off) and np.array_equal(a.nbr, b.nbr)
    assert np.abs(a.vert_xyz - b.vert_xyz).max() <= 1e-12 * w.diameter
    assert np.allclose(a.measure, b.measure, rtol=1e-11, atol=0)


# ---------------------------------------------------------------------- library special case (Qhull)
def test_qhull_interior_cells_3d():
    """Cells that do not touch the cube boundary are ordinary Voronoi cells: volume = hull of the
    Qhull Voronoi region, neighbours = Delaunay neighbours, 3-site corners = circumcentres."""
    from scipy.spatial import ConvexHull, Delaunay, Voronoi
    w = inputs.config(2, "small")
    c = oracle.compute(w.sites, w.verts, w.simplices, w.kind)
    vor = Voronoi(w.sites)
    tri = Delaunay(w.sites)
    indptr, indices = tri.vertex_neighbor_vertices
    m = w.m
    checked = 0
    for i in range(w.n):
        fl = np.concatenate([c.piece_verts(p)[1].ravel() for p in c.pieces(i)])
        if (fl == ~m).any():
            continue  # touches the domain boundary
        region = vor.regions[vor.point_region[i]]
        assert -1 not in region
        vol = ConvexHull(vor.vertices[region]).volume
        assert abs(vol - c.measure[i]) <= 1e-9 * vol
        assert sorted(indices[indptr[i]:indptr[i + 1]].tolist()) == c.neighbours(i).tolist()
        # corners labelled by three sites are Voronoi vertices (circumcentres of Delaunay tets)
        vv = vor.vertices[region]
        for p in c.pieces(i):
            xyz, f3 = c.piece_verts(p)
            for x, f in zip(xyz, f3):
                if (f >= 0).all():
                    assert np.linalg.norm(vv - x, axis=1).min() <= 1e-9
        checked += 1
    assert checked > 200


def test_qhull_interior_cells_2d():
    from scipy.spatial import Delaunay, Voronoi
    w = inputs.config(1)
    c = oracle.compute(w.sites, w.verts, w.simplices, w.kind)
    vor = Voronoi(w.sites)
    tri = Delaunay(w.sites)
    indptr, indices = tri.vertex_neighbor_vertices
    checked = 0
    for i in range(w.n):
        fl = np.concatenate([c.piece_verts(p)[1].ravel() for p in c.pieces(i)])
        if (fl == ~w.m).any():
            continue
        region = vor.regions[vor.point_region[i]]
        assert -1 not in region
        P = vor.vertices[region]
        cx = P[:, 0] * np.roll(P[:, 1], -1) - np.roll(P[:, 0], -1) * P[:, 1]
        assert abs(abs(cx.sum()) * 0.5 - c.measure[i]) <= 1e-10 * c.measure[i]
        assert sorted(indices[indptr[i]:indptr[i + 1]].tolist()) == c.neighbours(i).tolist()
        checked += 1
    assert checked > 1500


def test_surface_pieces_lie_in_their_triangle():
    w = inputs.config(4, "small")
    c = oracle.compute(w.sites, w.verts, w.simplices, w.kind)
    for p in range(len(c.piece_simplex)):
        tri = w.verts[w.simplices[c.piece_simplex[p]]]
        nrm = np.cross(tri[1] - tri[0], tri[2] - tri[0])
        nrm /= np.linalg.norm(nrm)
        xyz, _ = c.piece_verts(p)
        assert np.abs((xyz - tri[0]) @ nrm).max() <= 1e-13
    # cells with an empty restricted cell follow the empty-cell convention
    empty = c.measure == 0
    assert empty.any()
    assert np.array_equal(c.centroid[empty], w.sites[empty])


# ---------------------------------------------------------------------- simple domains (box kinds)
@pytest.mark.parametrize("dim", [2, 3])
def test_box_cells_are_the_dissolved_mesh_cells(dim):
    """The box kinds must give, per site, exactly the union of the pieces the meshed kinds give on a
    mesh of the same box (Eq. 1 does not depend on how the domain is cut up): same measure, centroid
    and neighbour sets; every corner with a box-face flag lies on the box boundary."""
    n = 300
    wb = inputs.box(dim, n, seed=21)
    if dim == 2:
        v, t = inputs.square_grid_mesh(3)
        kind = inputs.KIND_TRI_2D
    else:
        v, t = inputs.cube_kuhn_mesh(2)
        kind = inputs.KIND_TET_3D
    cm = oracle.compute(wb.sites, v, t, kind)
    cb = oracle.compute(wb.sites, wb.verts, None, wb.kind)
    assert abs(cb.measure.sum() - 1.0) <= 1e-12
    assert np.allclose(cb.measure, cm.measure, rtol=1e-11, atol=0)
    assert np.abs(cb.centroid - cm.centroid).max() <= 1e-12
    assert np.array_equal(cb.nbr_off, cm.nbr_off) and np.array_equal(cb.nbr, cm.nbr)
    assert np.array_equal(cb.piece_off, np.arange(n + 1)) and (cb.piece_simplex == 0).all()
    on_face = (cb.vert_flags == ~1).any(axis=1)
    x = cb.vert_xyz[on_face]
    assert (np.minimum(np.abs(x), np.abs(x - 1.0)).min(axis=1) <= 1e-14).all()
    assert on_face.any() and (~on_face).any()


def test_box_cells_qhull_and_tiers():
    """Interior cells of a shifted, non-cubic box against Qhull; tier A == tier B; sites outside the box."""
    from scipy.spatial import ConvexHull, Voronoi
    lo, hi = np.array([0.1, -0.2, 0.3]), np.array([1.3, 0.9, 1.1])
    rng = np.random.default_rng(4)
    sites = lo + (hi - lo) * (rng.random((400, 3)) * 1.2 - 0.1)
    box = np.stack([lo, hi])
    a = oracle.compute(sites, box, None, inputs.KIND_BOX_3D)
    b = oracle.compute(sites, box, None, inputs.KIND_BOX_3D, tier="B")
    assert abs(a.measure.sum() - np.prod(hi - lo)) <= 1e-12
    assert np.array_equal(a.vert_flags, b.vert_flags) and np.array_equal(a.nbr, b.nbr)
    assert np.allclose(a.measure, b.measure, rtol=1e-11, atol=0)
    vor = Voronoi(sites)
    checked = 0
    for i in range(len(sites)):
        if a.measure[i] == 0:
            continue
        _, fl = a.piece_verts(int(a.piece_off[i]))
        if (fl < 0).any():
            continue
        region = vor.regions[vor.point_region[i]]
        assert -1 not in region
        vol = ConvexHull(vor.vertices[region]).volume
        assert abs(vol - a.measure[i]) <= 1e-9 * vol
        checked += 1
    assert checked > 40


# ---------------------------------------------------------------------- dissolved output (Alg. 5)
@pytest.mark.parametrize("domain", ["cube", "octahedron"])
def test_dissolved_cells_are_the_union_of_their_pieces(domain):
    """The oracle's dissolved kind against its per-piece kind and against Qhull: a cell that does not reach the boundary of
    the convex domain comes as one piece (simplex id m) that is the union of its per-simplex pieces -- same measure,
    centroid and neighbour set --, an ordinary Voronoi cell (Qhull volume, V = 2F - 4, site labels only); every other
    cell keeps exactly its pieces."""
    from scipy.spatial import ConvexHull, Voronoi
    rng = np.random.default_rng(61)
    if domain == "cube":
        v, t = inputs.cube_kuhn_mesh(3)
        s = rng.random((600, 3)) * 1.1 - 0.05             # a few sites outside the cube
    else:
        v, t = inputs.octahedron_mesh()
        s = rng.random((1500, 3)) * 2.0 - 1.0             # many sites outside the octahedron, inside its bounding box
    m = len(t)
    plain = oracle.compute(s, v, t, inputs.KIND_TET_3D)
    for tier in ("A", "B"):
        dis = oracle.compute(s, v, t, inputs.KIND_TET_3D, dissolve=True, tier=tier)
        assert np.allclose(dis.measure, plain.measure, rtol=1e-11, atol=1e-15)
        assert np.abs(dis.centroid - plain.centroid).max() <= 1e-11
        assert np.array_equal(dis.nbr_off, plain.nbr_off) and np.array_equal(dis.nbr, plain.nbr)
    vor = Voronoi(s)
    whole = 0
    for i in range(len(s)):
        pp = list(plain.pieces(i))
        touches = any((plain.piece_verts(p)[1] == ~m).any() for p in pp)
        dp = list(dis.pieces(i))
        if not pp:
            assert not dp
        elif touches:
            assert [int(dis.piece_simplex[p]) for p in dp] == [int(plain.piece_simplex[p]) for p in pp]
            for a, b in zip(dp, pp):
                assert np.array_equal(dis.piece_verts(a)[1], plain.piece_verts(b)[1])
                assert np.abs(dis.piece_verts(a)[0] - plain.piece_verts(b)[0]).max() <= 1e-12    # (tier B against tier A: rounding)
        else:
            assert len(dp) == 1 and dis.piece_simplex[dp[0]] == m
            xyz, fl = dis.piece_verts(dp[0])
            assert (fl >= 0).all() and xyz.shape[0] == 2 * len(np.unique(fl)) - 4
            region = vor.regions[vor.point_region[i]]
            assert -1 not in region
            vol = ConvexHull(vor.vertices[region]).volume
            assert abs(vol - dis.measure[i]) <= 1e-9 * vol
            whole += 1
    assert whole > 30 and whole < (plain.measure > 0).sum()


# ---------------------------------------------------------------------- non-convex, disconnected domains
def _carved_cases():
    with open(os.path.join(HERE, "golden", "carved_square_cases.json")) as f:
        d = json.load(f)
    v, t = inputs.carved_domain(d["domain"]["kind"], d["domain"]["k"])
    return v, t, d["cases"]


def test_golden_carved_square_cases():
    """Hand-worked cells on the U-shaped square with a detached island: a cell in several connected components, and Voronoi
    neighbours whose common edge misses the domain are not restricted neighbours."""
    v, t, cases = _carved_cases()
    assert abs(inputs.mesh_measure(v, t, inputs.KIND_TRI_2D) - 0.62) < 1e-14
    for case in cases:
        s = np.array(case["sites"], dtype=np.float64)
        c = oracle.compute(s, v, t, inputs.KIND_TRI_2D)
        assert np.allclose(c.measure, case["area"], rtol=0, atol=1e-12)
        for i, cen in enumerate(case["centroid"]):
            if cen is not None:
                assert np.allclose(c.centroid[i], cen, rtol=0, atol=1e-12)
        for i, nb in enumerate(case["nbr"]):
            assert c.neighbours(i).tolist() == nb


@pytest.mark.parametrize("kind,n", [(inputs.KIND_TRI_2D, 600), (inputs.KIND_TRI_SURFACE, 800), (inputs.KIND_TET_3D, 700)])
def test_carved_domain_invariants_and_tiers(kind, n):
    w = inputs.carved(kind, n)
    c = oracle.compute(w.sites, w.verts, w.simplices, w.kind)
    _check_invariants(w, c, corner_sample=1500)
    if kind != inputs.KIND_TRI_SURFACE:
        b = oracle.compute(w.sites, w.verts, w.simplices, w.kind, tier="B")
        assert np.array_equal(c.piece_off, b.piece_off) and np.array_equal(c.piece_simplex, b.piece_simplex)
        assert np.array_equal(c.vert_flags, b.vert_flags) and np.array_equal(c.nbr, b.nbr)
        assert np.allclose(c.measure, b.measure, rtol=1e-11, atol=0)
