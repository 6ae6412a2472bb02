"""Power diagrams.  The oracle's weighted kinds clip with the power cell's own half-spaces; they are
pinned against (a) that definition written out here in numpy (2D), (b) the paper's construction -- the oracle's
restricted Voronoi diagram of the LIFTED sites on the flat surface --, (c) equal weights = the Voronoi diagram, and
(d) in 3D, brute force: every output corner has equal power distance to its cell's site and the sites of its flags,
and no site has a smaller one.  The CUDA path (vd_create_weighted: the lifting runs in its kernels) is compared with
the oracle on the same weighted inputs."""
import numpy as np
import pytest

from oracle import oracle
from paper_2509_07175_b200 import inputs


def _weighted(n, seed, spread):
    rng = np.random.default_rng(seed)
    return rng.random((n, 2)), spread * rng.random(n)


def _lift(s, w):          # written out here on purpose: the pin must not lean on the package
    return np.concatenate([s, np.sqrt(w.max() - w)[:, None]], axis=1)


def _clip_halfplane(poly, nrm, d):
    """Sutherland-Hodgman: keep n.x <= d."""
    out = []
    k = len(poly)
    for a in range(k):
        p, q = poly[a], poly[(a + 1) % k]
        sp, sq = nrm @ p - d, nrm @ q - d
        if sp <= 0:
            out.append(p)
        if (sp < 0 < sq) or (sq < 0 < sp):
            out.append(p + (q - p) * (sp / (sp - sq)))
    return out


def _power_cell_area(i, s, w):
    """Definition: {x in the unit square : |x - v_i|^2 - w_i <= |x - v_j|^2 - w_j for all j}."""
    poly = [np.array(p, float) for p in ((0, 0), (1, 0), (1, 1), (0, 1))]
    nbrs = []
    for j in range(len(s)):
        if j == i:
            continue
        nrm = 2.0 * (s[j] - s[i])
        d = s[j] @ s[j] - s[i] @ s[i] - w[j] + w[i]
        before = len(poly)
        new = _clip_halfplane(poly, nrm, d)
        if len(new) < 3:
            return 0.0
        poly = new
    x = np.array([p[0] for p in poly]); y = np.array([p[1] for p in poly])
    return 0.5 * abs(np.dot(x, np.roll(y, -1)) - np.dot(y, np.roll(x, -1)))


def test_oracle_surface_kind_on_lifted_sites_is_the_power_diagram():
    s, w = _weighted(300, 11, 0.004)          # weights comparable to the squared site spacing: some cells vanish
    verts, tris = inputs.unit_square_mesh()
    v3 = np.concatenate([verts, np.zeros((len(verts), 1))], axis=1)
    o = oracle.compute(_lift(s, w), v3, tris, inputs.KIND_TRI_SURFACE, tier="A")
    ref = np.array([_power_cell_area(i, s, w) for i in range(len(s))])
    assert np.abs(o.measure - ref).max() <= 1e-12
    assert (ref == 0).sum() > 0 and ((o.measure > 0) == (ref > 0)).all()      # hidden sites have empty cells
    assert abs(o.measure.sum() - 1.0) <= 1e-12
    # equal weights: the ordinary Voronoi diagram
    o0 = oracle.compute(_lift(s, np.full(len(s), 0.3)), v3, tris, inputs.KIND_TRI_SURFACE, tier="A")
    o2 = oracle.compute(s, verts, tris, inputs.KIND_TRI_2D, tier="A")
    assert np.abs(o0.measure - o2.measure).max() <= 1e-13
    assert np.array_equal(o0.nbr_off, o2.nbr_off) and np.array_equal(o0.nbr, o2.nbr)


def test_oracle_weighted_kind_2d():
    """The weighted 2D kind against the numpy definition and against the paper's lifted construction."""
    s, w = _weighted(300, 11, 0.004)
    verts, tris = inputs.square_grid_mesh(3)
    ow = oracle.compute(s, verts, tris, inputs.KIND_TRI_2D, weights=w)
    ref = np.array([_power_cell_area(i, s, w) for i in range(len(s))])
    assert np.abs(ow.measure - ref).max() <= 1e-12 and (ref == 0).sum() > 0
    v3 = np.concatenate([verts, np.zeros((len(verts), 1))], axis=1)
    ol = oracle.compute(_lift(s, w), v3, tris, inputs.KIND_TRI_SURFACE, tier="A")
    for f in ("nbr_off", "nbr", "piece_off", "piece_simplex", "vert_off", "vert_flags"):
        assert np.array_equal(getattr(ow, f), getattr(ol, f)), f
    assert np.abs(ow.vert_xyz - ol.vert_xyz[:, :2]).max() <= 1e-12 and np.abs(ol.vert_xyz[:, 2]).max() == 0.0
    assert np.abs(ow.measure - ol.measure).max() <= 1e-13
    # tier B (facets in the bounding box first) gives the same cells
    ob = oracle.compute(s, verts, tris, inputs.KIND_TRI_2D, weights=w, tier="B")
    assert np.array_equal(ob.vert_flags, ow.vert_flags) and np.abs(ob.measure - ow.measure).max() <= 1e-13


def _weighted3(n, seed, scale=1.0):
    rng = np.random.default_rng(seed)
    s = rng.random((n, 3))
    return s, scale * rng.uniform(-1.0, 1.0, n) / n ** (2.0 / 3.0)     # comparable to the squared site spacing


def test_oracle_weighted_kind_3d():
    s, w = _weighted3(400, 21, 0.6)
    verts, tets = inputs.cube_kuhn_mesh(2)
    o = oracle.compute(s, verts, tets, inputs.KIND_TET_3D, weights=w)
    assert abs(o.measure.sum() - 1.0) <= 1e-12
    assert (o.measure == 0).sum() > 0                                  # some sites are hidden
    # every corner: equal power distance to its own site and to the sites of its flags, none smaller (brute force)
    owner = np.repeat(np.repeat(np.arange(len(s)), np.diff(o.piece_off)), np.diff(o.vert_off))
    rng = np.random.default_rng(0)
    for v in rng.choice(len(o.vert_xyz), 3000, replace=False):
        pd = ((s - o.vert_xyz[v]) ** 2).sum(1) - w
        assert pd[owner[v]] <= pd.min() + 1e-12
        for fl in o.vert_flags[v]:
            if fl >= 0:
                assert abs(pd[fl] - pd[owner[v]]) <= 1e-12
    # neighbour symmetry, and a constant added to every weight changes nothing
    pairs = {(i, int(j)) for i in range(len(s)) for j in o.neighbours(i)}
    assert all((j, i) in pairs for i, j in pairs)
    o2 = oracle.compute(s, verts, tets, inputs.KIND_TET_3D, weights=w + 0.37)
    assert np.array_equal(o.vert_flags, o2.vert_flags) and np.abs(o.measure - o2.measure).max() <= 1e-13
    # equal weights: the Voronoi diagram, in the box kind too
    o0 = oracle.compute(s, verts, tets, inputs.KIND_TET_3D, weights=np.full(len(s), 0.2))
    o1 = oracle.compute(s, verts, tets, inputs.KIND_TET_3D)
    assert np.array_equal(o0.vert_flags, o1.vert_flags) and np.abs(o0.measure - o1.measure).max() <= 1e-13
    box = np.array([[0.0, 0, 0], [1.0, 1, 1]])
    ob = oracle.compute(s, box, None, inputs.KIND_BOX_3D, weights=w)
    assert np.abs(ob.measure - o.measure).max() <= 1e-12 and np.array_equal(ob.nbr, o.nbr)


@pytest.mark.gpu
@pytest.mark.parametrize("n,spread,k", [(2000, 0.0005, 8), (500, 0.01, 4)])
def test_power_diagram_parity_on_the_gpu(n, spread, k):
    import parity
    from paper_2509_07175_b200 import binding, power
    s, w = _weighted(n, 5, spread)
    verts, tris = inputs.square_grid_mesh(k)
    g = power.power_cells(s, w, verts, tris)
    assert g.dim == 2 and g.vert_xyz.shape[1] == 2
    o = oracle.compute(s, verts, tris, inputs.KIND_TRI_2D, weights=w)
    parity.assert_parity(g, o, np.sqrt(2.0))
    assert abs(g.measure.sum() - 1.0) <= 1e-11
    assert (g.measure == 0).sum() == (o.measure == 0).sum() > 0 or spread < 0.001
    g2 = power.power_cells(s, w, verts, tris, eta=float(w.max()) + 0.05)     # any admissible eta gives the same cells
    parity.assert_parity(g2, o, np.sqrt(2.0))
    with pytest.raises(binding.VdError) as e:                                # eta below the largest weight
        power.power_cells(s, w, verts, tris, eta=float(w.max()) - 1e-3)
    assert e.value.status == 4


@pytest.mark.gpu
@pytest.mark.parametrize("kind,opts", [("tet", {}), ("tet", dict(small_wave=-1)), ("box", {}), ("box", dict(small_wave=-1, near_clips=-1))])
def test_power_diagram_3d_parity_on_the_gpu(kind, opts):
    """3-D weighted sites (lifted to R^4 inside the library: the fourth coordinate enters as an additive term) on a tet
    mesh and on the box kind, against the oracle's power cells; some sites are hidden (empty cells), some do not lie in
    their own cell."""
    import parity
    from paper_2509_07175_b200 import binding, power
    s, w = _weighted3(3000, 33, 0.8)
    if kind == "tet":
        verts, simp, k = *inputs.cube_kuhn_mesh(3), inputs.KIND_TET_3D
        o = oracle.compute(s, verts, simp, k, weights=w, tier="B")
    else:
        verts, simp, k = np.array([[0.0, 0, 0], [1.0, 1, 1]]), None, inputs.KIND_BOX_3D
        o = oracle.compute(s, verts, None, k, weights=w, tier="B")
    g = power.power_cells(s, w, verts, simp, kind=k, **opts)
    parity.assert_parity(g, o, np.sqrt(3.0))
    assert abs(g.measure.sum() - 1.0) <= 1e-11
    assert (g.measure == 0).sum() == (o.measure == 0).sum() > 0
    own = np.array([np.argmin(((s - s[i]) ** 2).sum(1) - w) for i in range(0, len(s), 7)])
    assert (own != np.arange(0, len(s), 7)).any()           # the case exists: a site outside its own power cell
    g2 = power.power_cells(s, w, verts, simp, kind=k, eta=float(w.max()) + 0.01, **opts)
    parity.assert_parity(g2, o, np.sqrt(3.0))
