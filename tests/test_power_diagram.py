"""Power diagrams by lifting: the oracle's surface kind on lifted sites is pinned against the power
cell's own definition (half-plane clipping with power bisectors, written out here in numpy), and the CUDA path is
compared with the oracle on the same lifted inputs."""
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


def test_lift_helper():
    from paper_2509_07175_b200 import power
    s, w = _weighted(50, 3, 0.1)
    p = power.lift_sites(s, w)
    assert p.shape == (50, 3) and np.allclose(p, _lift(s, w)) and p[:, 2].min() == 0.0       # eta = max w
    q = power.lift_sites(s, w, eta=1.0)
    # |x - p_i|^2 - |x - p_j|^2 at height 0 equals the power-distance difference, whatever eta
    x = np.array([0.3, 0.7, 0.0])
    for lifted in (p, q):
        dd = ((x - lifted) ** 2).sum(1)
        pw = ((x[:2] - s) ** 2).sum(1) - w
        assert np.allclose(dd - dd[0], pw - pw[0], atol=1e-12)
    with pytest.raises(ValueError):
        power.lift_sites(s, w, eta=float(w.max()) - 1e-3)


@pytest.mark.gpu
@pytest.mark.parametrize("n,spread,k", [(2000, 0.0005, 8), (500, 0.01, 4)])
def test_power_diagram_parity_on_the_gpu(n, spread, k):
    import parity
    from paper_2509_07175_b200 import power
    s, w = _weighted(n, 5, spread)
    verts, tris = inputs.square_grid_mesh(k)
    g = power.power_cells(s, w, verts, tris)
    o = oracle.compute(power.lift_sites(s, w), power.embed_domain(verts), tris, inputs.KIND_TRI_SURFACE, tier="A")
    parity.assert_parity(g, o, np.sqrt(2.0))
    assert abs(g.measure.sum() - 1.0) <= 1e-11
    assert (g.measure == 0).sum() == (o.measure == 0).sum()
