"""Seeded synthetic inputs: domains (simplicial meshes) and site sets.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA library, so it
holds none of the method's arithmetic: no nearest-site search, no clipping, no
bisectors -- only mesh construction and random draws (numpy ``default_rng(seed)``,
PCG64).  The recipes restate BASELINE.json ``configs[0..4]``;
they stand in for the paper's workloads (white noise PAPER.md L409, voids / uneven
density L399, sites far from the domain L481, surface meshes L290), whose own meshes
and site sets are not available.

Domain kinds follow ``include/vd.h``: 0 = 2D triangles, 1 = surface triangles (in
R^3), 2 = 3D tetrahedra, 3 / 4 = axis-aligned rectangle / box given by (lo, hi)
(the "simple domains" of PAPER.md L241-243: no mesh, one piece per cell).
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass

import numpy as np

KIND_TRI_2D = 0
KIND_TRI_SURFACE = 1
KIND_TET_3D = 2
KIND_BOX_2D = 3
KIND_BOX_3D = 4


@dataclass
class Workload:
    name: str
    kind: int
    dim: int
    sites: np.ndarray      # [n, dim] float64
    verts: np.ndarray      # [nv, dim] float64
    simplices: np.ndarray  # [m, 3 or 4] int32; None for the box kinds
    measure: float         # |M| (area / surface area / volume), from the mesh recipe
    diameter: float        # diameter of the domain's bounding box

    @property
    def n(self) -> int:
        return int(self.sites.shape[0])

    @property
    def m(self) -> int:
        return 1 if self.simplices is None else int(self.simplices.shape[0])


# --------------------------------------------------------------------------- domains
def unit_square_mesh():
    """Unit square split along (0,0)-(1,1): triangles (0,1,2), (0,2,3)."""
    verts = np.array([[0.0, 0.0], [1.0, 0.0], [1.0, 1.0], [0.0, 1.0]], dtype=np.float64)
    tris = np.array([[0, 1, 2], [0, 2, 3]], dtype=np.int32)
    return verts, tris


def square_grid_mesh(k: int):
    """Unit square as a k x k grid of quads, each split into 2 triangles."""
    g = np.arange(k + 1, dtype=np.float64) / k
    X, Y = np.meshgrid(g, g, indexing="ij")
    verts = np.stack([X.ravel(), Y.ravel()], axis=1)
    vid = lambda ix, iy: ix * (k + 1) + iy
    tris = []
    for ix in range(k):
        for iy in range(k):
            a, b, c, d = vid(ix, iy), vid(ix + 1, iy), vid(ix + 1, iy + 1), vid(ix, iy + 1)
            tris.append((a, b, c))
            tris.append((a, c, d))
    return verts, np.array(tris, dtype=np.int32)


def cube_kuhn_mesh(k: int):
    """Unit cube as k^3 sub-cubes x 6 Kuhn tetrahedra (conforming across cubes).

    Vertex id = (ix*(k+1)+iy)*(k+1)+iz; for each permutation pi of the axes the tet
    has corners o, o+e_pi1, o+e_pi1+e_pi2, o+(1,1,1).  Orientation alternates with
    the parity of pi (the library and the oracle both accept any orientation).
    """
    k1 = k + 1
    g = np.arange(k1, dtype=np.float64) / k
    X, Y, Z = np.meshgrid(g, g, g, indexing="ij")
    verts = np.stack([X.ravel(), Y.ravel(), Z.ravel()], axis=1)
    ix, iy, iz = np.meshgrid(np.arange(k), np.arange(k), np.arange(k), indexing="ij")
    base = np.stack([ix.ravel(), iy.ravel(), iz.ravel()], axis=1)  # [k^3, 3]
    tets = []
    for perm in itertools.permutations(range(3)):
        c = [base.copy()]
        cur = base.copy()
        for ax in perm:
            cur = cur.copy()
            cur[:, ax] += 1
            c.append(cur)
        ids = [(p[:, 0] * k1 + p[:, 1]) * k1 + p[:, 2] for p in c]
        tets.append(np.stack(ids, axis=1))
    # interleave so that the 6 tets of a sub-cube are adjacent in memory
    tets = np.stack(tets, axis=1).reshape(-1, 4).astype(np.int32)
    return verts, tets


def torus_mesh(nu: int, nv: int, R: float = 1.0, r: float = 0.35):
    """Torus P(u,v) tessellated nu x nv quads -> 2*nu*nv triangles."""
    iu, iv = np.meshgrid(np.arange(nu), np.arange(nv), indexing="ij")
    u = 2.0 * np.pi * iu.ravel() / nu
    v = 2.0 * np.pi * iv.ravel() / nv
    verts = np.stack([(R + r * np.cos(v)) * np.cos(u),
                      (R + r * np.cos(v)) * np.sin(u),
                      r * np.sin(v)], axis=1)
    vid = lambda a, b: (a % nu) * nv + (b % nv)
    a = vid(iu, iv).ravel()
    b = vid(iu + 1, iv).ravel()
    c = vid(iu + 1, iv + 1).ravel()
    d = vid(iu, iv + 1).ravel()
    tris = np.stack([np.stack([a, b, c], axis=1), np.stack([a, c, d], axis=1)], axis=1)
    return verts.astype(np.float64), tris.reshape(-1, 3).astype(np.int32)


def octahedron_mesh():
    """Regular octahedron |x| + |y| + |z| <= 1 as 8 tetrahedra around the origin: a convex domain that is not a box
    (8 boundary triangles in 8 distinct planes)."""
    verts = np.array([[0, 0, 0], [1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]], dtype=np.float64)
    tets = [(0, 1 + (sx < 0), 3 + (sy < 0), 5 + (sz < 0)) for sx in (1, -1) for sy in (1, -1) for sz in (1, -1)]
    return verts, np.array(tets, dtype=np.int32)


def carve(verts: np.ndarray, simplices: np.ndarray, keep: np.ndarray):
    """The sub-mesh of the simplices flagged in `keep`, its vertices renumbered without gaps."""
    simp = simplices[keep]
    used = np.unique(simp)
    remap = np.full(len(verts), -1, dtype=np.int64)
    remap[used] = np.arange(len(used))
    return np.ascontiguousarray(verts[used]), remap[simp].astype(np.int32)


def carved_domain(kind: int, k: int = 10, jitter: float = 0.0, seed: int = 5):
    """A non-convex, disconnected domain (Alg. 4 makes no convexity assumption): the unit square / cube /
    torus minus a notch (the rest is U-shaped, or an open band with two boundary loops) and minus a strip that detaches
    an island.  `jitter` > 0 moves every vertex by up to jitter x grid spacing (uneven simplices, all still positively
    sized for jitter < 0.2); on the square and the cube the outer boundary vertices move too, so the measure is the
    mesh's own (`mesh_measure`), not a closed form."""
    rng = np.random.default_rng(seed)
    if kind == KIND_TRI_SURFACE:
        verts, simp = torus_mesh(4 * k, 2 * k)
        c = verts[simp].mean(axis=1)
        u = np.arctan2(c[:, 1], c[:, 0])                       # angle around the axis, (-pi, pi]
        keep = ~((u > 0.4) & (u < 1.3)) & ~((u > 2.2) & (u < 2.5)) & ~((u > -2.0) & (u < -1.8) & (c[:, 2] > 0))
        h = 2.0 * np.pi / (4 * k)
    else:
        verts, simp = square_grid_mesh(k) if kind == KIND_TRI_2D else cube_kuhn_mesh(k)
        c = verts[simp].mean(axis=1)
        notch = (c[:, 0] > 0.3) & (c[:, 0] < 0.7) & (c[:, 1] > 0.3)
        strip = (c[:, 0] > 0.8) & (c[:, 0] < 0.9)
        keep = ~notch & ~strip
        h = 1.0 / k
    if jitter > 0.0:
        verts = verts + (rng.random(verts.shape) * 2.0 - 1.0) * (jitter * h)
    return carve(verts, simp, keep)


def mesh_measure(verts: np.ndarray, simplices: np.ndarray, kind: int) -> float:
    """|M| from the mesh itself (plain determinant / cross-product formulas)."""
    p = verts[simplices]
    if kind == KIND_TRI_2D:
        e1, e2 = p[:, 1] - p[:, 0], p[:, 2] - p[:, 0]
        return float(np.abs(e1[:, 0] * e2[:, 1] - e1[:, 1] * e2[:, 0]).sum() * 0.5)
    if kind == KIND_TRI_SURFACE:
        return float(np.linalg.norm(np.cross(p[:, 1] - p[:, 0], p[:, 2] - p[:, 0]), axis=1).sum() * 0.5)
    e = p[:, 1:] - p[:, :1]
    return float(np.abs(np.linalg.det(e)).sum() / 6.0)


def _wl(name, kind, sites, verts, simplices):
    verts = np.ascontiguousarray(verts, dtype=np.float64)
    sites = np.ascontiguousarray(sites, dtype=np.float64)
    simplices = np.ascontiguousarray(simplices, dtype=np.int32)
    diam = float(np.linalg.norm(verts.max(0) - verts.min(0)))
    return Workload(name, kind, sites.shape[1], sites, verts, simplices,
                    mesh_measure(verts, simplices, kind), diam)


# --------------------------------------------------------------------------- site sets
def sites_uniform(rng, n, dim):
    return rng.random((n, dim))


def sites_clustered(rng, n, n_clusters=32, sig_lo=0.005, sig_hi=0.1):
    """Mixture of anisotropic Gaussians, samples rejected outside the unit cube."""
    mu = 0.1 + 0.8 * rng.random((n_clusters, 3))
    sig = np.exp(rng.uniform(np.log(sig_lo), np.log(sig_hi), (n_clusters, 3)))
    out, have = [], 0
    batch = max(n, 1024)
    while have < n:
        k = rng.integers(0, n_clusters, batch)
        x = mu[k] + sig[k] * rng.standard_normal((batch, 3))
        keep = np.all((x >= 0.0) & (x <= 1.0), axis=1)
        out.append(x[keep])
        have += int(keep.sum())
    return np.concatenate(out, axis=0)[:n]


def sites_torus_shell(rng, n, R=1.0, r=0.35, t_max=0.05):
    """Area-uniform on the torus, displaced along the normal by U(-t_max, t_max)."""
    us, vs = [], []
    have = 0
    batch = max(2 * n, 1024)
    while have < n:
        u = 2.0 * np.pi * rng.random(batch)
        v = 2.0 * np.pi * rng.random(batch)
        acc = rng.random(batch) < (R + r * np.cos(v)) / (R + r)
        us.append(u[acc])
        vs.append(v[acc])
        have += int(acc.sum())
    u = np.concatenate(us)[:n]
    v = np.concatenate(vs)[:n]
    t = rng.uniform(-t_max, t_max, n)
    nrm = np.stack([np.cos(v) * np.cos(u), np.cos(v) * np.sin(u), np.sin(v)], axis=1)
    p = np.stack([(R + r * np.cos(v)) * np.cos(u), (R + r * np.cos(v)) * np.sin(u), r * np.sin(v)], axis=1)
    return p + t[:, None] * nrm


def sites_far_slab(rng, n, z0=1.5):
    x = rng.random(n)
    y = rng.random(n)
    z = z0 + rng.random(n)
    return np.stack([x, y, z], axis=1)


# --------------------------------------------------------------------------- configs
def config(idx: int, scale: str = "full") -> Workload:
    """BASELINE.json configs[idx-1] (idx = 1..5).  scale='full' or 'small' (the
    scaled-down replicas used for the literal O(n^2) oracle)."""
    small = scale == "small"
    if idx == 1:
        rng = np.random.default_rng(0)
        v, t = unit_square_mesh()
        return _wl("C1" + ("s" if small else ""), KIND_TRI_2D, sites_uniform(rng, 200 if small else 2000, 2), v, t)
    if idx == 2:
        rng = np.random.default_rng(1)
        v, t = cube_kuhn_mesh(4 if small else 20)
        return _wl("C2" + ("s" if small else ""), KIND_TET_3D, sites_uniform(rng, 2000 if small else 100000, 3), v, t)
    if idx == 3:
        rng = np.random.default_rng(2)
        v, t = cube_kuhn_mesh(6 if small else 48)
        return _wl("C3" + ("s" if small else ""), KIND_TET_3D, sites_clustered(rng, 5000 if small else 1000000), v, t)
    if idx == 4:
        rng = np.random.default_rng(3)
        v, t = torus_mesh(32, 16) if small else torus_mesh(512, 256)
        return _wl("C4" + ("s" if small else ""), KIND_TRI_SURFACE, sites_torus_shell(rng, 1000 if small else 200000), v, t)
    if idx == 5:
        rng = np.random.default_rng(4)
        v, t = cube_kuhn_mesh(4 if small else 32)
        return _wl("C5" + ("s" if small else ""), KIND_TET_3D, sites_far_slab(rng, 20000 if small else 2000000), v, t)
    raise ValueError("config index must be 1..5")


def custom(kind: int, sites, verts, simplices, name="custom") -> Workload:
    return _wl(name, kind, np.asarray(sites, dtype=np.float64), verts, simplices)


def carved(kind: int, n: int, jitter: float = 0.15, seed: int = 31, k: int = 10) -> Workload:
    """`carved_domain` with sites over its bounding box, the removed parts included (cells that lose pieces to the
    notch, cells that own nothing, cells split between an arm and the island); surface kind: a shell around the torus as
    in C4."""
    v, t = carved_domain(kind, k, jitter)
    rng = np.random.default_rng(seed)
    if kind == KIND_TRI_SURFACE:
        sites = sites_torus_shell(rng, n)
    else:
        lo, hi = v.min(0) - 0.03, v.max(0) + 0.03
        sites = lo + rng.random((n, v.shape[1])) * (hi - lo)
    return custom(kind, sites, v, t, f"carved{kind}")


def box(dim: int, n: int, seed: int = 7, lo=None, hi=None, name=None) -> Workload:
    """n white-noise sites in an axis-aligned box, the box itself as the (simple) domain: the paper's
    "Voronoi diagram of sites in a cube" setting (Fig. 1 caption L5, Table VI)."""
    lo = np.zeros(dim) if lo is None else np.asarray(lo, dtype=np.float64)
    hi = np.ones(dim) if hi is None else np.asarray(hi, dtype=np.float64)
    rng = np.random.default_rng(seed)
    sites = lo + (hi - lo) * rng.random((n, dim))
    return Workload(name or f"box{dim}d_{n}", KIND_BOX_2D if dim == 2 else KIND_BOX_3D, dim, sites,
                    np.stack([lo, hi]), None, float(np.prod(hi - lo)), float(np.linalg.norm(hi - lo)))


def grid_sites(k: int, dim: int) -> np.ndarray:
    """Regular k^dim grid of sites at ((a+1/2)/k, ...): the degenerate hand case."""
    g = (np.arange(k, dtype=np.float64) + 0.5) / k
    mesh = np.meshgrid(*([g] * dim), indexing="ij")
    return np.stack([x.ravel() for x in mesh], axis=1)
