// vd_oracle.cpp -- CPU ORACLE for clipped / restricted Voronoi cells.  TEST INFRASTRUCTURE ONLY.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// build, load or call this file.  It shares no code, header, table or helper with the CUDA path
// (paper_2509_07175_b200/csrc) and neither includes the other.
//
// What it computes is the plain DEFINITION, not the paper's method (the method reaches exactly
// the defined result, "guarantees exact results", L441):
//
//   Omega_i = { x : |x - v_i| <= |x - v_j|  for all j != i }                 (Eq. 1)
//   Omega_i|M = Omega_i  intersect  M,   M = { T_a }
//   P_{a,i}  = T_a  intersect  (intersection over j != i of H_ij)            (pieces)
//   H_ij     = { x : (v_j - v_i).(x - v_i) <= 1/2 |v_j - v_i|^2 }            (the half-space of Eq. 1)
//
// There is no grid, no nearest-site query, no point-in-cell test, no bisector search and no
// flag-driven propagation here.  Each simplex is clipped by the half-spaces one after another
// (Sutherland-Hodgman on a polygon; per-face Sutherland-Hodgman plus a cap face on a polyhedron),
// carrying one label per edge / face (the flag of an edge/face is the adjacent
// simplex or the neighbouring cell):
//     label >= 0      : site id j   (the edge/face lies on the bisector B_ij)
// Kinds 3 / 4 are the paper's "simple domains" (section V-B): an axis-aligned rectangle / box given
// by its two opposite corners, treated as ONE convex piece (simplex id 0, m = 1, every face labelled ~m).
//     label <  0      : ~label = id of the simplex adjacent across that edge/face,
//                       ~label == m means a face on the domain boundary
// (0-based restatement of the paper's +j / -b convention; reading U3 in DESIGN.md).
//
// Tier A ("literal"):  every (a, i) is clipped by ALL j != i, in index order, stopping only when
//                      the piece has become empty (an empty intersection stays empty).
// Tier B ("two-phase", exact by convexity):  phase 1 clips an axis-aligned box containing M by all
//                      n-1 half-spaces -> the facet sites F_i of Omega_i in that box;  phase 2 clips
//                      each T_a by H_ij, j in F_i only.  A convex polytope is the intersection of
//                      its facet half-spaces and T_a lies in the box, so the result is the same set.
//                      tests/ check tier B == tier A on the small replicas before it is used.
//
// Per cell:  measure = sum_a |P_{a,i}|,  centroid = sum_a |P|.c(P) / measure,
// neighbours = { j : some piece has an edge/face labelled j },  pieces with their corners, each
// corner carrying the labels of the edges/faces that meet there (2 for triangles, 3 for tets),
// corners of a piece sorted lexicographically by their ascending label tuple.
//
// Arithmetic: fp64 (the paper's GPU runs were fp32; BASELINE.json fixes fp64).
//
// Pins (tests/test_oracle_pins.py): hand-worked closed forms in the unit square, regular grids,
// sum of measures = |M|, first-moment identity, per-simplex conservation, neighbour symmetry,
// corner equidistance + no nearer site by brute force, scipy/Qhull Voronoi volumes and Delaunay
// neighbours for interior cells, tier A == tier B; negative flags: every corner flagged ~b lies on the face T_a
// really shares with T_b, every corner flagged ~m on a face no other simplex owns, and conversely every corner on a
// face of T_a carries that face's flag (mesh topology recomputed in numpy) -- so no function here is "parity unpinned".

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <thread>
#include <utility>
#include <vector>

namespace {

typedef double real;

struct V3 {
  real x, y, z;
};
static inline V3 operator+(const V3& a, const V3& b) { return {a.x + b.x, a.y + b.y, a.z + b.z}; }
static inline V3 operator-(const V3& a, const V3& b) { return {a.x - b.x, a.y - b.y, a.z - b.z}; }
static inline V3 operator*(real s, const V3& a) { return {s * a.x, s * a.y, s * a.z}; }
static inline real dot(const V3& a, const V3& b) { return a.x * b.x + a.y * b.y + a.z * b.z; }
static inline V3 cross(const V3& a, const V3& b) {
  return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}

enum { KIND_TRI_2D = 0, KIND_TRI_SURFACE = 1, KIND_TET_3D = 2, KIND_BOX_2D = 3, KIND_BOX_3D = 4 };
static const int LABEL_PAD = INT32_MIN;        // padding when a corner has fewer labels than expected
static const int LABEL_BOX = INT32_MIN + 1;    // faces of the phase-1 box (tier B), never output

// ------------------------------------------------------------------------------------------------
// Half-space H_ij written as  s(x) = (v_j - v_i).(x - v_i) - 1/2 |v_j - v_i|^2  <= 0   (Eq. 1)
struct HalfSpace {
  V3 n;      // v_j - v_i
  V3 o;      // v_i
  real h;    // 1/2 |n|^2
  int label; // j
  real eval(const V3& x) const { return dot(n, x - o) - h; }
};

static HalfSpace bisector(const V3& vi, const V3& vj, int j) {
  HalfSpace H;
  H.n = vj - vi;
  H.o = vi;
  H.h = 0.5 * dot(H.n, H.n);
  H.label = j;
  return H;
}

// Power diagram (section VII-C; Aurenhammer's power cell): the half-space of
//   |x - v_i|^2 - w_i <= |x - v_j|^2 - w_j   <=>   (v_j - v_i).(x - v_i) <= 1/2 |v_j - v_i|^2 + 1/2 (w_i - w_j).
// (With p = (v, sqrt(eta - w)) in R^(d+1) and x at height 0, |x - p_i|^2 = |x - v_i|^2 + eta - w_i: the paper's lifted
// restricted Voronoi diagram is this set, whatever eta.)
static HalfSpace power_bisector(const V3& vi, real wi, const V3& vj, real wj, int j) {
  HalfSpace H = bisector(vi, vj, j);
  H.h = H.h + 0.5 * (wi - wj);
  return H;
}

// ------------------------------------------------------------------------------------------------
// Convex polygon (2D domain or a planar polygon in R^3): ordered corners + one label per edge.
// Edge k runs from corner k to corner k+1 (cyclic).
struct Polygon {
  std::vector<V3> P;
  std::vector<int> L;
  bool empty() const { return P.empty(); }
};

// Sutherland-Hodgman by one half-space.  A convex polygon meets the boundary line in at most
// one exit and one entry crossing; the new edge between them takes the half-space's label.
static void clip_polygon(Polygon& G, const HalfSpace& H) {
  const size_t k = G.P.size();
  if (k == 0) return;
  std::vector<real> s(k);
  bool anyOut = false, anyIn = false;
  for (size_t c = 0; c < k; ++c) {
    s[c] = H.eval(G.P[c]);
    if (s[c] > 0) anyOut = true; else anyIn = true;
  }
  if (!anyOut) return;
  if (!anyIn) { G.P.clear(); G.L.clear(); return; }
  std::vector<V3> outP;
  std::vector<int> outL;
  for (size_t c = 0; c < k; ++c) {
    const size_t d = (c + 1) % k;
    const bool inA = s[c] <= 0, inB = s[d] <= 0;
    if (inA && inB) {
      outP.push_back(G.P[c]); outL.push_back(G.L[c]);
    } else if (inA && !inB) {
      outP.push_back(G.P[c]); outL.push_back(G.L[c]);
      const real t = s[c] / (s[c] - s[d]);
      outP.push_back(G.P[c] + t * (G.P[d] - G.P[c]));   // exit point: the cut edge starts here
      outL.push_back(H.label);
    } else if (!inA && inB) {
      const real t = s[d] / (s[d] - s[c]);
      outP.push_back(G.P[d] + t * (G.P[c] - G.P[d]));   // entry point: rest of edge c keeps its label
      outL.push_back(G.L[c]);
    }
  }
  G.P.swap(outP);
  G.L.swap(outL);
  if (G.P.size() < 3) { G.P.clear(); G.L.clear(); }
}

// ------------------------------------------------------------------------------------------------
// Convex polyhedron: vertex array + faces as vertex-index loops (counter-clockwise seen from
// outside) + one label per face.
struct Polyhedron {
  std::vector<V3> V;
  std::vector<std::vector<int> > F;
  std::vector<int> L;
  bool empty() const { return F.empty(); }
  void clear() { V.clear(); F.clear(); L.clear(); }
};

// Clip by one half-space: Sutherland-Hodgman on every face; the crossing points (one per cut
// polyhedron edge, shared by its two faces through the edge's vertex-id pair) are chained into
// the cap face, which takes the half-space's label.
static void clip_polyhedron(Polyhedron& G, const HalfSpace& H) {
  const size_t nv = G.V.size();
  if (G.F.empty()) return;
  std::vector<real> s(nv);
  bool anyOut = false, anyIn = false;
  for (size_t v = 0; v < nv; ++v) {
    s[v] = H.eval(G.V[v]);
    if (s[v] > 0) anyOut = true; else anyIn = true;
  }
  if (!anyOut) return;
  if (!anyIn) { G.clear(); return; }

  std::map<std::pair<int, int>, int> cut;  // (inside vertex, outside vertex) -> new vertex id
  auto cutVertex = [&](int u, int v) -> int {  // u inside, v outside
    std::pair<int, int> key(u, v);
    std::map<std::pair<int, int>, int>::iterator it = cut.find(key);
    if (it != cut.end()) return it->second;
    const real t = s[u] / (s[u] - s[v]);
    G.V.push_back(G.V[u] + t * (G.V[v] - G.V[u]));
    const int id = (int)G.V.size() - 1;
    cut[key] = id;
    return id;
  };

  std::vector<std::vector<int> > newF;
  std::vector<int> newL;
  std::map<int, int> capNext;  // entry vertex -> exit vertex of the same face (cap edge, reversed)
  for (size_t f = 0; f < G.F.size(); ++f) {
    const std::vector<int>& loop = G.F[f];
    const size_t k = loop.size();
    std::vector<int> out;
    int X = -1, E = -1;
    for (size_t c = 0; c < k; ++c) {
      const int a = loop[c], b = loop[(c + 1) % k];
      const bool inA = s[a] <= 0, inB = s[b] <= 0;
      if (inA) out.push_back(a);
      if (inA && !inB) { X = cutVertex(a, b); out.push_back(X); }
      else if (!inA && inB) { E = cutVertex(b, a); out.push_back(E); }
    }
    if (out.size() >= 3) { newF.push_back(out); newL.push_back(G.L[f]); }
    if (X >= 0 && E >= 0) capNext[E] = X;   // the face has edge X->E; the cap has E->X
  }
  if (capNext.size() >= 3) {
    std::vector<int> cap;
    const int start = capNext.begin()->first;
    int cur = start;
    for (size_t guard = 0; guard <= capNext.size(); ++guard) {
      cap.push_back(cur);
      std::map<int, int>::iterator it = capNext.find(cur);
      if (it == capNext.end()) break;
      cur = it->second;
      if (cur == start) break;
    }
    if (cap.size() >= 3) { newF.push_back(cap); newL.push_back(H.label); }
  }
  // drop unreferenced vertices
  std::vector<int> remap(G.V.size(), -1);
  std::vector<V3> newV;
  for (size_t f = 0; f < newF.size(); ++f)
    for (size_t c = 0; c < newF[f].size(); ++c) {
      int& v = newF[f][c];
      if (remap[v] < 0) { remap[v] = (int)newV.size(); newV.push_back(G.V[v]); }
      v = remap[v];
    }
  G.V.swap(newV);
  G.F.swap(newF);
  G.L.swap(newL);
  if (G.F.size() < 4) G.clear();
}

// ------------------------------------------------------------------------------------------------
// Measures and first moments (the paper times "centroids computation", L443,
// without giving a formula: these are the textbook fan decompositions).
static void polygon_measure(const Polygon& G, int kind, real& meas, V3& moment) {
  // fan from corner 0; vector area summed, then its norm (2D: the z component).
  V3 A = {0, 0, 0};
  const size_t k = G.P.size();
  for (size_t c = 1; c + 1 < k; ++c) A = A + cross(G.P[c] - G.P[0], G.P[c + 1] - G.P[0]);
  const real nA = std::sqrt(dot(A, A));
  meas = 0.5 * nA;
  moment = {0, 0, 0};
  if (nA <= 0) { meas = 0; return; }
  const V3 nh = (1.0 / nA) * A;
  for (size_t c = 1; c + 1 < k; ++c) {
    const real a = 0.5 * dot(cross(G.P[c] - G.P[0], G.P[c + 1] - G.P[0]), nh);
    moment = moment + (a / 3.0) * (G.P[0] + G.P[c] + G.P[c + 1]);
  }
  (void)kind;
}

static void polyhedron_measure(const Polyhedron& G, real& meas, V3& moment) {
  // signed tetrahedra (ref, f0, fk, fk+1) over every face fan; ref = the piece's first corner.
  meas = 0;
  moment = {0, 0, 0};
  if (G.F.empty()) return;
  const V3 ref = G.V[G.F[0][0]];
  for (size_t f = 0; f < G.F.size(); ++f) {
    const std::vector<int>& loop = G.F[f];
    const V3 a = G.V[loop[0]] - ref;
    for (size_t c = 1; c + 1 < loop.size(); ++c) {
      const V3 b = G.V[loop[c]] - ref, d = G.V[loop[c + 1]] - ref;
      const real vol = dot(a, cross(b, d)) / 6.0;
      meas += vol;
      // centroid of the tet = ref + (a + b + d)/4
      moment = moment + vol * (ref + 0.25 * (a + b + d));
    }
  }
}

// ------------------------------------------------------------------------------------------------
struct Domain {
  int kind, dim, nc;   // nc = corners per simplex
  int64_t nv, m;
  std::vector<V3> verts;
  std::vector<int32_t> simp;   // m * nc
  std::vector<int32_t> adj;    // m * nc : simplex across the face opposite local corner k, or m
};

static V3 load_point(const double* p, int dim) {
  V3 r = {p[0], p[1], dim == 3 ? p[2] : 0.0};
  return r;
}

// Adjacency: two simplices are adjacent across a face iff they share its d vertices (PAPER.md L85,
// Fig. 2a "edge/face flags of a domain simplex").  Returns nonzero on a non-manifold face.
static int build_adjacency(Domain& D) {
  const int nc = D.nc;
  typedef std::vector<int32_t> Key;
  std::map<Key, std::vector<std::pair<int32_t, int> > > faces;
  for (int64_t a = 0; a < D.m; ++a)
    for (int k = 0; k < nc; ++k) {
      Key key;
      for (int c = 0; c < nc; ++c)
        if (c != k) key.push_back(D.simp[a * nc + c]);
      std::sort(key.begin(), key.end());
      faces[key].push_back(std::make_pair((int32_t)a, k));
    }
  D.adj.assign(D.m * nc, (int32_t)D.m);
  for (std::map<Key, std::vector<std::pair<int32_t, int> > >::iterator it = faces.begin(); it != faces.end(); ++it) {
    std::vector<std::pair<int32_t, int> >& v = it->second;
    if (v.size() > 2) return 1;
    if (v.size() == 2) {
      D.adj[(int64_t)v[0].first * nc + v[0].second] = v[1].first;
      D.adj[(int64_t)v[1].first * nc + v[1].second] = v[0].first;
    }
  }
  return 0;
}

// The simplex as a labelled polygon: edge opposite local corner k is labelled ~adj[a][k].
static Polygon simplex_polygon(const Domain& D, int64_t a) {
  Polygon G;
  const int32_t* s = &D.simp[a * 3];
  const int32_t* ad = &D.adj[a * 3];
  // loop 0,1,2: edge 0->1 is opposite corner 2, 1->2 opposite 0, 2->0 opposite 1
  G.P = {D.verts[s[0]], D.verts[s[1]], D.verts[s[2]]};
  G.L = {~ad[2], ~ad[0], ~ad[1]};
  return G;
}

// The simplex as a labelled polyhedron: face opposite local corner k is labelled ~adj[a][k];
// loops are counter-clockwise seen from outside for a positively oriented tet, reversed otherwise.
static Polyhedron simplex_polyhedron(const Domain& D, int64_t a) {
  Polyhedron G;
  const int32_t* s = &D.simp[a * 4];
  const int32_t* ad = &D.adj[a * 4];
  G.V = {D.verts[s[0]], D.verts[s[1]], D.verts[s[2]], D.verts[s[3]]};
  static const int loops[4][3] = {{1, 2, 3}, {0, 3, 2}, {0, 1, 3}, {0, 2, 1}};
  const real det = dot(G.V[1] - G.V[0], cross(G.V[2] - G.V[0], G.V[3] - G.V[0]));
  for (int k = 0; k < 4; ++k) {
    std::vector<int> loop(loops[k], loops[k] + 3);
    if (det < 0) std::reverse(loop.begin(), loop.end());
    G.F.push_back(loop);
    G.L.push_back(~ad[k]);
  }
  return G;
}

static Polyhedron box_polyhedron(const V3& lo, const V3& hi, int label = LABEL_BOX) {
  Polyhedron G;
  for (int c = 0; c < 8; ++c)
    G.V.push_back({(c & 1) ? hi.x : lo.x, (c & 2) ? hi.y : lo.y, (c & 4) ? hi.z : lo.z});
  static const int loops[6][4] = {{0, 4, 6, 2}, {1, 3, 7, 5}, {0, 1, 5, 4}, {2, 6, 7, 3}, {0, 2, 3, 1}, {4, 5, 7, 6}};
  for (int f = 0; f < 6; ++f) {
    G.F.push_back(std::vector<int>(loops[f], loops[f] + 4));
    G.L.push_back(label);
  }
  return G;
}

// ------------------------------------------------------------------------------------------------
struct PieceOut {
  int32_t simplex;
  real meas;
  V3 moment;
  std::vector<V3> corners;
  std::vector<int32_t> flags;  // nfl per corner, ascending
  std::vector<int32_t> faceSites;  // labels >= 0 of the piece's edges / faces
};

struct CellOut {
  real meas;
  V3 centroid;
  std::vector<int32_t> nbr;
  std::vector<PieceOut> pieces;
};

static void sort_corners(PieceOut& po, int nfl) {
  const size_t k = po.corners.size();
  std::vector<size_t> idx(k);
  for (size_t c = 0; c < k; ++c) idx[c] = c;
  const std::vector<int32_t>& fl = po.flags;
  std::stable_sort(idx.begin(), idx.end(), [&](size_t a, size_t b) {
    for (int t = 0; t < nfl; ++t)
      if (fl[a * nfl + t] != fl[b * nfl + t]) return fl[a * nfl + t] < fl[b * nfl + t];
    return false;
  });
  std::vector<V3> c2(k);
  std::vector<int32_t> f2(k * nfl);
  for (size_t c = 0; c < k; ++c) {
    c2[c] = po.corners[idx[c]];
    for (int t = 0; t < nfl; ++t) f2[c * nfl + t] = fl[idx[c] * nfl + t];
  }
  po.corners.swap(c2);
  po.flags.swap(f2);
}

static bool finish_polygon(const Polygon& G, int kind, int32_t a, PieceOut& po) {
  if (G.P.size() < 3) return false;
  polygon_measure(G, kind, po.meas, po.moment);
  if (!(po.meas > 0)) return false;
  po.simplex = a;
  const size_t k = G.P.size();
  for (size_t c = 0; c < k; ++c) {
    po.corners.push_back(G.P[c]);
    int32_t l0 = G.L[(c + k - 1) % k], l1 = G.L[c];   // the two edges meeting at corner c
    if (l0 > l1) std::swap(l0, l1);
    po.flags.push_back(l0);
    po.flags.push_back(l1);
    if (G.L[c] >= 0) po.faceSites.push_back(G.L[c]);
  }
  sort_corners(po, 2);
  return true;
}

static bool finish_polyhedron(const Polyhedron& G, int32_t a, PieceOut& po) {
  if (G.F.size() < 4) return false;
  polyhedron_measure(G, po.meas, po.moment);
  if (!(po.meas > 0)) return false;
  po.simplex = a;
  const size_t nv = G.V.size();
  std::vector<std::vector<int32_t> > lab(nv);
  for (size_t f = 0; f < G.F.size(); ++f) {
    for (size_t c = 0; c < G.F[f].size(); ++c) lab[G.F[f][c]].push_back(G.L[f]);
    if (G.L[f] >= 0) po.faceSites.push_back(G.L[f]);
  }
  for (size_t v = 0; v < nv; ++v) {
    std::sort(lab[v].begin(), lab[v].end());
    po.corners.push_back(G.V[v]);
    for (int t = 0; t < 3; ++t) po.flags.push_back(t < (int)lab[v].size() ? lab[v][t] : LABEL_PAD);
  }
  sort_corners(po, 3);
  return true;
}

struct Problem {
  Domain D;
  int64_t n;
  std::vector<V3> sites;
  std::vector<real> w;   // weights (power diagram); empty = the ordinary Voronoi diagram
  // "dissolved" output for convex volumetric domains ("an interior site's clipped cell equals its Voronoi
  // cell"; reading U1): a cell none of whose pieces has a face on the domain boundary is reported as ONE piece -- the bounding
  // box of M clipped by the same half-spaces, simplex id m, site labels only -- instead of its per-simplex pieces.
  bool dissolve = false;
  V3 lo, hi;             // bounding box of the domain's vertices
  HalfSpace half_space(int64_t i, int64_t j) const {
    return w.empty() ? bisector(sites[i], sites[j], (int)j) : power_bisector(sites[i], w[i], sites[j], w[j], (int)j);
  }
};

// One cell, tier A: T_a clipped by every H_ij, j != i, in index order (the literal definition).
// planes == NULL -> all j != i;  else only the listed sites (tier B phase 2).
static void compute_cell(const Problem& Pb, int64_t i, const std::vector<int32_t>* planes, CellOut& out) {
  const Domain& D = Pb.D;
  const V3 vi = Pb.sites[i];
  out.meas = 0;
  V3 mom = {0, 0, 0};
  std::vector<HalfSpace> HS;
  if (planes) {
    for (size_t k = 0; k < planes->size(); ++k) HS.push_back(Pb.half_space(i, (*planes)[k]));
  }
  for (int64_t a = 0; a < D.m; ++a) {
    PieceOut po;
    bool ok = false;
    if (D.kind == KIND_TET_3D || D.kind == KIND_BOX_3D) {
      // a simple domain (section V-B: "e.g. a cube") is one convex piece; its faces are domain boundary (~m)
      Polyhedron G = D.kind == KIND_BOX_3D ? box_polyhedron(D.verts[0], D.verts[1], ~(int)D.m) : simplex_polyhedron(D, a);
      if (planes) {
        for (size_t k = 0; k < HS.size() && !G.empty(); ++k) clip_polyhedron(G, HS[k]);
      } else {
        for (int64_t j = 0; j < Pb.n && !G.empty(); ++j)
          if (j != i) clip_polyhedron(G, Pb.half_space(i, j));
      }
      ok = !G.empty() && finish_polyhedron(G, (int32_t)a, po);
    } else {
      Polygon G;
      if (D.kind == KIND_BOX_2D) {
        const V3 lo = D.verts[0], hi = D.verts[1];
        G.P = {{lo.x, lo.y, 0}, {hi.x, lo.y, 0}, {hi.x, hi.y, 0}, {lo.x, hi.y, 0}};
        G.L = {~(int)D.m, ~(int)D.m, ~(int)D.m, ~(int)D.m};
      } else {
        G = simplex_polygon(D, a);
      }
      if (planes) {
        for (size_t k = 0; k < HS.size() && !G.empty(); ++k) clip_polygon(G, HS[k]);
      } else {
        for (int64_t j = 0; j < Pb.n && !G.empty(); ++j)
          if (j != i) clip_polygon(G, Pb.half_space(i, j));
      }
      ok = !G.empty() && finish_polygon(G, D.kind, (int32_t)a, po);
    }
    if (!ok) continue;
    out.meas += po.meas;
    mom = mom + po.moment;
    for (size_t k = 0; k < po.faceSites.size(); ++k) out.nbr.push_back(po.faceSites[k]);
    out.pieces.push_back(po);
  }
  if (Pb.dissolve && D.kind == KIND_TET_3D && !out.pieces.empty()) {
    bool onBoundary = false;
    for (size_t p = 0; p < out.pieces.size() && !onBoundary; ++p)
      for (size_t k = 0; k < out.pieces[p].flags.size(); ++k)
        if (out.pieces[p].flags[k] == ~(int32_t)D.m) { onBoundary = true; break; }
    if (!onBoundary) {
      // the cell does not reach the boundary of the convex domain: Omega_i ∩ M = Omega_i, and the box contains it
      Polyhedron G = box_polyhedron(Pb.lo, Pb.hi, ~(int)D.m);
      if (planes) {
        for (size_t k = 0; k < HS.size() && !G.empty(); ++k) clip_polyhedron(G, HS[k]);
      } else {
        for (int64_t j = 0; j < Pb.n && !G.empty(); ++j)
          if (j != i) clip_polyhedron(G, Pb.half_space(i, j));
      }
      PieceOut po;
      if (!G.empty() && finish_polyhedron(G, (int32_t)D.m, po)) {
        out.pieces.clear();
        out.nbr = po.faceSites;
        out.meas = po.meas;
        mom = po.moment;
        out.pieces.push_back(po);
      }
    }
  }
  std::sort(out.nbr.begin(), out.nbr.end());
  out.nbr.erase(std::unique(out.nbr.begin(), out.nbr.end()), out.nbr.end());
  if (out.meas > 0) out.centroid = (1.0 / out.meas) * mom;
  else out.centroid = vi;   // empty cell convention of include/vd.h
}

// Tier B phase 1: facet sites of Omega_i inside an axis-aligned box that contains the domain.
// Works for dim 3 (box polyhedron) and dim 2 (box polygon).
// Returns false when Omega_i does not meet the box at all (then every piece is empty).
static bool facet_sites(const Problem& Pb, int64_t i, const V3& lo, const V3& hi, std::vector<int32_t>& F) {
  const V3 vi = Pb.sites[i];
  F.clear();
  if (Pb.D.dim == 3) {
    Polyhedron G = box_polyhedron(lo, hi);
    for (int64_t j = 0; j < Pb.n && !G.empty(); ++j)
      if (j != i) clip_polyhedron(G, Pb.half_space(i, j));
    if (G.empty()) return false;
    for (size_t f = 0; f < G.L.size(); ++f)
      if (G.L[f] >= 0) F.push_back(G.L[f]);
  } else {
    Polygon G;
    G.P = {{lo.x, lo.y, 0}, {hi.x, lo.y, 0}, {hi.x, hi.y, 0}, {lo.x, hi.y, 0}};
    G.L = {LABEL_BOX, LABEL_BOX, LABEL_BOX, LABEL_BOX};
    for (int64_t j = 0; j < Pb.n && !G.empty(); ++j)
      if (j != i) clip_polygon(G, Pb.half_space(i, j));
    if (G.empty()) return false;
    for (size_t f = 0; f < G.L.size(); ++f)
      if (G.L[f] >= 0) F.push_back(G.L[f]);
  }
  std::sort(F.begin(), F.end());
  return true;
}

}  // namespace

// ================================================================================================
// C entry points (loaded with ctypes by oracle/oracle.py)
extern "C" {

struct vdo_result {
  int64_t ns;       // cells computed
  int dim, nfl;     // nfl = labels per corner (2 triangles, 3 tets)
  int64_t n_pieces, n_verts, n_nbrs;
  double* measure;        // [ns]
  double* centroid;       // [ns*dim]
  int64_t* nbr_off;       // [ns+1]
  int32_t* nbr;           // [n_nbrs]
  int64_t* piece_off;     // [ns+1]
  int32_t* piece_simplex; // [n_pieces]
  double* piece_measure;  // [n_pieces]
  int64_t* vert_off;      // [n_pieces+1]
  double* vert_xyz;       // [n_verts*dim]
  int32_t* vert_flags;    // [n_verts*nfl]
  int32_t* simplex_adj;   // [m*(nc)] adjacency the oracle derived (for tests)
  int threads_used;
};

void vdo_free(vdo_result* r) {
  if (!r) return;
  free(r->measure); free(r->centroid); free(r->nbr_off); free(r->nbr); free(r->piece_off);
  free(r->piece_simplex); free(r->piece_measure); free(r->vert_off); free(r->vert_xyz);
  free(r->vert_flags); free(r->simplex_adj);
  free(r);
}

// sites [n][dim], verts [nv][dim], simplices [m][dim+1 or 3], kind as include/vd.h.
// subset: site ids to compute (NULL -> all n).  tier: 0 = A (literal), 1 = B (two-phase).
// Returns 0 on success; 1 bad argument; 4 bad input (non-manifold face, index out of range).
// weights: NULL = Voronoi diagram; else [n] weights of the power diagram (section VII-C).
// dissolve != 0 (tets): cells that do not reach the domain boundary come as one whole piece (Problem::dissolve).
int vdo_compute_x(const double* sites, const double* weights, int64_t n, int dim, const double* verts, int64_t nv,
                  const int32_t* simplices, int64_t m, int kind, const int64_t* subset, int64_t n_subset,
                  int tier, int nthreads, int dissolve, vdo_result** out) {
  const bool box = kind == KIND_BOX_2D || kind == KIND_BOX_3D;
  if (!sites || !verts || (!simplices && !box) || !out || n < 1 || m < 1 || nv < 1) return 1;
  if (!(((kind == KIND_TRI_2D || kind == KIND_BOX_2D) && dim == 2) || ((kind == KIND_TRI_SURFACE || kind == KIND_TET_3D || kind == KIND_BOX_3D) && dim == 3))) return 1;
  if (box && (nv != 2 || m != 1)) return 1;   // verts = the two opposite corners (lo, hi)
  if (kind == KIND_TRI_SURFACE && tier == 1) return 1;  // a surface has no enclosing-box shortcut here: use tier A
  Problem Pb;
  Pb.n = n;
  Pb.sites.resize(n);
  for (int64_t i = 0; i < n; ++i) Pb.sites[i] = load_point(sites + i * dim, dim);
  if (weights) Pb.w.assign(weights, weights + n);
  Domain& D = Pb.D;
  D.kind = kind; D.dim = dim; D.nc = box ? 0 : ((kind == KIND_TET_3D) ? 4 : 3); D.nv = nv; D.m = m;
  D.verts.resize(nv);
  for (int64_t v = 0; v < nv; ++v) D.verts[v] = load_point(verts + v * dim, dim);
  if (!box) D.simp.assign(simplices, simplices + m * D.nc);
  for (int64_t k = 0; k < m * D.nc; ++k)
    if (D.simp[k] < 0 || D.simp[k] >= nv) return 4;
  if (!box && build_adjacency(D)) return 4;

  const int64_t ns = subset ? n_subset : n;
  std::vector<CellOut> cells(ns);
  V3 lo = D.verts[0], hi = D.verts[0];
  for (int64_t v = 0; v < nv; ++v) {
    lo.x = std::min(lo.x, D.verts[v].x); hi.x = std::max(hi.x, D.verts[v].x);
    lo.y = std::min(lo.y, D.verts[v].y); hi.y = std::max(hi.y, D.verts[v].y);
    lo.z = std::min(lo.z, D.verts[v].z); hi.z = std::max(hi.z, D.verts[v].z);
  }
  Pb.dissolve = dissolve != 0;
  Pb.lo = lo; Pb.hi = hi;
  if (nthreads < 1) nthreads = (int)std::thread::hardware_concurrency();
  if (nthreads < 1) nthreads = 1;
  if ((int64_t)nthreads > ns) nthreads = (int)ns;
  std::atomic<int64_t> next(0);
  auto worker = [&]() {
    for (;;) {
      const int64_t s = next.fetch_add(1);
      if (s >= ns) break;
      const int64_t i = subset ? subset[s] : s;
      if (tier == 1) {
        std::vector<int32_t> F;
        if (facet_sites(Pb, i, lo, hi, F)) {
          compute_cell(Pb, i, &F, cells[s]);
        } else {
          cells[s].meas = 0;
          cells[s].centroid = Pb.sites[i];
        }
      } else {
        compute_cell(Pb, i, NULL, cells[s]);
      }
    }
  };
  std::vector<std::thread> pool;
  for (int t = 1; t < nthreads; ++t) pool.push_back(std::thread(worker));
  worker();
  for (size_t t = 0; t < pool.size(); ++t) pool[t].join();

  vdo_result* R = (vdo_result*)calloc(1, sizeof(vdo_result));
  R->ns = ns; R->dim = dim; R->nfl = (kind == KIND_TET_3D || kind == KIND_BOX_3D) ? 3 : 2; R->threads_used = nthreads;
  for (int64_t s = 0; s < ns; ++s) {
    R->n_pieces += (int64_t)cells[s].pieces.size();
    R->n_nbrs += (int64_t)cells[s].nbr.size();
    for (size_t p = 0; p < cells[s].pieces.size(); ++p) R->n_verts += (int64_t)cells[s].pieces[p].corners.size();
  }
  R->measure = (double*)malloc(sizeof(double) * (ns + 1));
  R->centroid = (double*)malloc(sizeof(double) * (ns * dim + 1));
  R->nbr_off = (int64_t*)malloc(sizeof(int64_t) * (ns + 1));
  R->nbr = (int32_t*)malloc(sizeof(int32_t) * (R->n_nbrs + 1));
  R->piece_off = (int64_t*)malloc(sizeof(int64_t) * (ns + 1));
  R->piece_simplex = (int32_t*)malloc(sizeof(int32_t) * (R->n_pieces + 1));
  R->piece_measure = (double*)malloc(sizeof(double) * (R->n_pieces + 1));
  R->vert_off = (int64_t*)malloc(sizeof(int64_t) * (R->n_pieces + 1));
  R->vert_xyz = (double*)malloc(sizeof(double) * (R->n_verts * dim + 1));
  R->vert_flags = (int32_t*)malloc(sizeof(int32_t) * (R->n_verts * R->nfl + 1));
  R->simplex_adj = (int32_t*)malloc(sizeof(int32_t) * (m * D.nc + 1));
  if (!box) memcpy(R->simplex_adj, D.adj.data(), sizeof(int32_t) * m * D.nc);
  int64_t ip = 0, iv = 0, in = 0;
  for (int64_t s = 0; s < ns; ++s) {
    const CellOut& c = cells[s];
    R->measure[s] = c.meas;
    R->centroid[s * dim + 0] = c.centroid.x;
    R->centroid[s * dim + 1] = c.centroid.y;
    if (dim == 3) R->centroid[s * dim + 2] = c.centroid.z;
    R->nbr_off[s] = in;
    for (size_t k = 0; k < c.nbr.size(); ++k) R->nbr[in++] = c.nbr[k];
    R->piece_off[s] = ip;
    for (size_t p = 0; p < c.pieces.size(); ++p) {
      const PieceOut& po = c.pieces[p];
      R->piece_simplex[ip] = po.simplex;
      R->piece_measure[ip] = po.meas;
      R->vert_off[ip] = iv;
      for (size_t k = 0; k < po.corners.size(); ++k) {
        R->vert_xyz[iv * dim + 0] = po.corners[k].x;
        R->vert_xyz[iv * dim + 1] = po.corners[k].y;
        if (dim == 3) R->vert_xyz[iv * dim + 2] = po.corners[k].z;
        for (int t = 0; t < R->nfl; ++t) R->vert_flags[iv * R->nfl + t] = po.flags[k * R->nfl + t];
        ++iv;
      }
      ++ip;
    }
  }
  R->nbr_off[ns] = in;
  R->piece_off[ns] = ip;
  R->vert_off[ip] = iv;
  *out = R;
  return 0;
}

int vdo_compute_w(const double* sites, const double* weights, int64_t n, int dim, const double* verts, int64_t nv,
                  const int32_t* simplices, int64_t m, int kind, const int64_t* subset, int64_t n_subset,
                  int tier, int nthreads, vdo_result** out) {
  return vdo_compute_x(sites, weights, n, dim, verts, nv, simplices, m, kind, subset, n_subset, tier, nthreads, 0, out);
}

int vdo_compute(const double* sites, int64_t n, int dim, const double* verts, int64_t nv,
                const int32_t* simplices, int64_t m, int kind, const int64_t* subset, int64_t n_subset,
                int tier, int nthreads, vdo_result** out) {
  return vdo_compute_w(sites, NULL, n, dim, verts, nv, simplices, m, kind, subset, n_subset, tier, nthreads, out);
}

}  // extern "C"
