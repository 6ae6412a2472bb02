"""Full-size BASELINE.json configs on the GPU, in the launch configuration bench.py times: global
invariants over all cells plus element-by-element parity on sampled sites the oracle computes one by
one (seeded-random half, extremes of the GPU report half -- choosing WHICH sites to check from the GPU
output is harmless, the check itself is independent)."""
import numpy as np
import pytest

from oracle import oracle
from paper_2509_07175_b200 import binding, inputs

import parity

pytestmark = pytest.mark.gpu


def _sample(g, n, k, seed):
    """K sites: half seeded-random, half the extremes of the GPU report.  Where most cells are empty
    (C4: 70 %, C5: 99.93 %) three quarters of the random half are drawn from the non-empty cells and the rest over all
    sites, which checks emptiness."""
    rng = np.random.default_rng(seed)
    pos = np.where(g.measure > 0)[0]
    half = min(n, k // 2)
    if len(pos) < 0.9 * n:
        rnd = np.concatenate([rng.choice(pos, size=min(len(pos), (3 * half) // 4), replace=False),
                              rng.choice(n, size=half - (3 * half) // 4, replace=False)])
    else:
        rnd = rng.choice(n, size=half, replace=False)
    npieces = np.diff(g.piece_off)
    nnbr = np.diff(g.nbr_off)
    q = k // 8
    ext = np.concatenate([np.argsort(-g.measure)[:q], np.argsort(-npieces)[:q], np.argsort(-nnbr)[:q],
                          pos[np.argsort(g.measure[pos])[:q]]])
    return np.unique(np.concatenate([rnd, ext])).astype(np.int64)


@pytest.mark.parametrize("idx,k", [(2, 512), (4, 512), (5, 512), (3, 512)])
def test_full_config_invariants_and_sampled_parity(idx, k):
    w = inputs.config(idx)
    with binding.Context(w.sites) as ctx:
        ctx.set_domain(w.verts, w.simplices, w.kind)
        ctx.compute()
        g = ctx.to_host()
        cnt = ctx.counters()
    chk = parity.global_checks(g, w)
    assert chk["sum_measure_rel"] <= 1e-11, chk
    assert chk["per_simplex_rel"] <= 1e-10, chk
    assert chk["nbr_symmetric"], chk
    assert cnt["pieces"] == len(g.piece_simplex)
    ids = _sample(g, w.n, k, 1000 + idx)
    tier = "A" if w.kind == inputs.KIND_TRI_SURFACE else "B"
    o = oracle.compute(w.sites, w.verts, w.simplices, w.kind, subset=ids, tier=tier)
    bad = parity.assert_parity(g, o, w.diameter, simplex_measure=parity.simplex_measures(w))
    print(f"C{idx}: {len(ids)} sampled cells ({int((o.measure == 0).sum())} empty), max rel measure error "
          f"{bad['_max_rel_measure']:.3e}, max corner error {bad['_max_xyz']:.3e}")


@pytest.mark.parametrize("dim,n,k", [(3, 1000000, 256), (2, 2000000, 256)])
def test_box_domain_at_scale(dim, n, k):
    """Whole-cell mode at the paper's scale of sites in a cube / square: cells partition
    the box, neighbour relation symmetric, sampled cells equal the oracle's."""
    w = inputs.box(dim, n, seed=9)
    with binding.Context(w.sites) as ctx:
        ctx.set_domain(w.verts, None, w.kind)
        ctx.compute()
        g = ctx.to_host()
        cnt = ctx.counters()
    assert abs(g.measure.sum() - 1.0) <= 1e-11
    assert np.abs((g.measure[:, None] * g.centroid).sum(0) - 0.5).max() <= 1e-11
    assert cnt["pieces"] == n and (np.diff(g.piece_off) == 1).all()
    src = np.repeat(np.arange(n, dtype=np.int64), np.diff(g.nbr_off))
    fwd = np.sort(src * n + g.nbr)
    rev = np.sort(g.nbr.astype(np.int64) * n + src)
    assert np.array_equal(fwd, rev)
    ids = _sample(g, n, k, 77 + dim)
    o = oracle.compute(w.sites, w.verts, None, w.kind, subset=ids, tier="B")
    parity.assert_parity(g, o, w.diameter, ids=ids, simplex_measure=parity.simplex_measures(w))


def test_c2_dissolve_mode_all_cells():
    """Alg. 5's site division at full size (C2: 100,000 sites, 48,000 tets): every cell's measure, centroid and neighbour set
    equal the per-piece run's (itself oracle-checked above), 512 sampled cells equal the oracle's dissolved kind element by
    element, and the counters say what the mode saves."""
    w = inputs.config(2)
    with binding.Context(w.sites) as ctx:
        ctx.set_options(count_alg=1)                 # per-query statistics on (off by default)
        ctx.set_domain(w.verts, w.simplices, w.kind)
        ctx.compute()
        plain, c0 = ctx.to_host(), ctx.counters()
        ctx.set_options(dissolve=1, count_alg=1)
        ctx.compute()
        g, c1 = ctx.to_host(), ctx.counters()
        ctx.set_options(dissolve=1)                  # the default kernels: same cells, no per-query statistics
        ctx.compute()
        g2, c2 = ctx.to_host(), ctx.counters()
    assert np.array_equal(g2.vert_flags, g.vert_flags) and np.allclose(g2.measure, g.measure, rtol=1e-11, atol=0)
    assert c2["queries"] < 0.01 * c1["queries"] and c2["pairs"] == c1["pairs"]     # (what is left: the seeds' queries of the mesh vertices)
    assert np.array_equal(g.nbr_off, plain.nbr_off) and np.array_equal(g.nbr, plain.nbr)
    assert np.allclose(g.measure, plain.measure, rtol=1e-9, atol=0)
    assert np.abs(g.centroid - plain.centroid).max() <= 1e-9 * w.diameter
    whole = (g.piece_simplex == w.m)
    assert 0.8 * w.n < whole.sum() < 0.95 * w.n and (np.diff(g.piece_off)[g.piece_simplex[g.piece_off[:-1]] == w.m] == 1).all()
    assert c1["pairs"] < 0.25 * c0["pairs"] and c1["queries"] < 0.6 * c0["queries"]
    print(f"C2 dissolve: {int(whole.sum())} whole cells, pairs {c0['pairs']} -> {c1['pairs']}, queries per cell "
          f"{c0['queries'] / w.n:.1f} -> {c1['queries'] / w.n:.1f} (paper, serial Alg. 2 on 1 M cells in a cube: 20.5, P:L375)")
    ids = _sample(g, w.n, 512, 4242)
    o = oracle.compute(w.sites, w.verts, w.simplices, w.kind, subset=ids, tier="B", dissolve=True)
    parity.assert_parity(g, o, w.diameter, simplex_measure=parity.simplex_measures(w).max())
