// vd_nearest.cuh -- S2: warp-cooperative nearest-site query over the grid index.
// All 32 lanes of a warp call these functions with the SAME query point; lanes split the candidate
// rows / sites; results are warp-uniform.
#pragma once
#include "vd_common.cuh"

namespace vd {

struct QueryStats {
  int skip;   // SKIP instantiations only (S1b): the site id that does not count as a candidate
};
// How the query routines receive it.  The counting fields this struct once had live in shared memory (WarpStats below); what is left
// is S1b's skip id, which only kernels outside the lean build use -- there the struct travels by value (a dead 4-byte argument)
// instead of by reference (a pointer that every not-inlined routine keeps alive across its own calls).
#if VD_EXT
using StRef = QueryStats&;
#else
using StRef = QueryStats;
#endif

// Work counters that are bumped rarely (per clip, per piece, per measurement-mode query) live in shared memory, one row
// per warp, instead of in registers of kernels that run at their register cap: [0] corners side-tested by clips,
// [1] corners created by clips, [2] fan simplices of finished pieces, [3] step-out probes, [4] D_alg.
constexpr int kExtraCnt = 6;   // [5] candidates that passed the fp32 filter (evaluated in fp64)
static __shared__ unsigned sExtraCnt[kWarpsPerBlock][kExtraCnt + 3];

// The statistics of the queries (nearest-site queries, site distance evaluations, grid rows examined) live in shared memory
// too, one row per warp, bumped by lane 0 with warp-uniform amounts: as fields of a struct passed by reference into the (not
// inlined) query routines they lived in LOCAL memory -- a load and a store per update, through the L1 the site records
// stream through (measured: 3-4 % of a step).  VD_STAT(st.rows += n;) names the row `st`, shadowing the unused parameter.
struct WarpStats { unsigned queries, dist_evals, rows, pad; };
static __shared__ WarpStats sWarpStats[kWarpsPerBlock];
__device__ __forceinline__ WarpStats& warp_stats() { return sWarpStats[(threadIdx.x / kLanes) % kWarpsPerBlock]; }
// They exist in the full kernels only (VD_EXT, vd_options.count_alg): in the default kernels the updates alone -- a
// predicated read-modify-write per query, row pass and candidate round -- were 3-4 % of a step (C2 19.98 -> 19.35 ms).
#if !VD_EXT
#define VD_STAT(x)
#else
#define VD_STAT(x) { if (lane_id() == 0) { WarpStats& st = warp_stats(); x } }
#endif
// Work counters of the clip path (clips, first clips, search iterations, corners tested / created, fan simplices): also the full
// kernels' only -- the by-reference LocalCnt fields live in local memory and each update waits for its own load (measured: ~4 % of
// the stall samples of k_ph_tail on C2).  pairs / pieces stay in every build.
#if !VD_EXT
#define VD_WORK(x)
#else
#define VD_WORK(x) x
#endif

__device__ __forceinline__ void extra_cnt_reset() {
  if (lane_id() < kExtraCnt) sExtraCnt[(threadIdx.x / kLanes) % kWarpsPerBlock][lane_id()] = 0u;
  if (lane_id() == 0) { WarpStats& w = warp_stats(); w.queries = 0u; w.dist_evals = 0u; w.rows = 0u; w.pad = 0u; }
  __syncwarp();
}
__device__ __forceinline__ void extra_cnt_add(int which, unsigned v) {
  if (lane_id() == 0) sExtraCnt[(threadIdx.x / kLanes) % kWarpsPerBlock][which] += v;
}

__device__ __forceinline__ int cell_of(const GridIndex& g, int ax, double q) {
  int c = (int)floor((q - g.lo[ax]) * g.inv_h[ax]);
  return min(max(c, 0), g.G[ax] - 1);
}

// squared distance from q to the slab [lo + c0*h, lo + (c1+1)*h] along one axis (slightly widened:
// conservative against the rounding of the cell assignment)
__device__ __forceinline__ double slab_d2(const GridIndex& g, int ax, double q, int c0, int c1) {
  const double a = g.lo[ax] + (c0 - 1e-9) * g.h[ax];
  const double b = g.lo[ax] + (c1 + 1 + 1e-9) * g.h[ax];
  const double d = (q < a) ? (a - q) : ((q > b) ? (q - b) : 0.0);
  return d * d;
}

// The one packing routine of every candidate scan (nearest query, batched tests, nearest-site lists, one-shot search): lane r
// holds row r of up to 32 grid rows -- `cnt` sites from position `s` of the sorted site array (cnt = 0: none).  Their candidates
// are handed out 32 per round: body(valid, pos, owner) runs once per round with all lanes converged; lane l gets candidate
// t0 + l -- `valid`: it exists, `pos`: its position in the site array, `owner`: the index, among the rows that start in or
// straddle this round (in lane order), of the row it belongs to.  on_row(slot) has run before on the lane that holds row
// number `slot` of the round (for per-row payloads such as the query a row belongs to).  base: 32 ints of shared scratch of
// this warp.  At most `limit` candidates are handed out.  Returns how many.
template <class OnRow, class Body>
__device__ __forceinline__ int for_each_packed(int s, int cnt, int* base, int limit, OnRow&& on_row, Body&& body) {
  const int lane = lane_id();
  const int incl = warp_incl_scan(cnt);
  const int excl = incl - cnt;
  const int total = min(shfl(incl, kLanes - 1), limit);
  for (int t0 = 0; t0 < total; t0 += kLanes) {
    // rows that start inside this round, plus the row that straddles its beginning
    unsigned bit = 0;
    if (cnt > 0) {
      if (excl >= t0 && excl < t0 + kLanes) bit = 1u << (excl - t0);
      else if (excl < t0 && incl > t0) bit = 1u;
    }
    const unsigned starts = __reduce_or_sync(kFull, bit);
    const unsigned owners = __ballot_sync(kFull, bit != 0);
    if (bit) {
      const int slot = __popc(owners & ((1u << lane) - 1u));
      base[slot] = s - excl;
      on_row(slot);
    }
    __syncwarp();
    const int t = t0 + lane;
    const bool valid = t < total;
    const int owner = valid ? __popc(starts & ((2u << lane) - 1u)) - 1 : 0;
    body(valid, valid ? base[owner] + t : 0, owner);
    __syncwarp();
  }
  return total;
}

// Scan every cell of the box [x0..x1]x[y0..y1]x[z0..z1] whose row can hold a site closer than best.
// One lane per row (y,z): box-distance pruning, x-extent tightened to the ball, one contiguous site
// range per row.  The candidates of all rows are then packed 32 at a time over the lanes (prefix sum of
// the row counts; the row that owns candidate t is found from a bit mask of row starts), so a typical
// query of ~30 candidates in 4-9 rows costs one round of distance evaluations instead of one per row.
template <bool SKIP>
static __device__ __noinline__ void scan_cell(const GridIndex& g, int x, int y, int z, double qx, double qy, double qz, double& best,
                                              int& bestId, StRef st);

// TOP = true: g is the site index itself and may hold refined cells (second level); a row that contains
// one is walked cell by cell afterwards: plain cells are scanned as they are, a refined cell through its
// own sub-grid (the same routine with TOP = false on a view of that cell).
template <bool TOP, bool SKIP = false>
static __device__ __noinline__ void scan_box(const GridIndex& g, double qx, double qy, double qz, int x0, int x1, int y0, int y1,
                                      int z0, int z1, double& best, int& bestId, StRef st) {
  __shared__ int sBase[kWarpsPerBlock][kLanes];
  const int lane = lane_id();
  int* base = sBase[(threadIdx.x / kLanes) % kWarpsPerBlock];
  const int ny = y1 - y0 + 1;
  const int nrows = ny * (z1 - z0 + 1);
  VD_STAT(st.rows += (unsigned)nrows;)
  // fp32 filter: the query in float, and the fp32 threshold of the current bound (recomputed when the bound moves)
  const bool f32 = has_f32(g) && !has_weights(g);
  float qxf = 0.f, qyf = 0.f, qzf = 0.f, thr = 0.f;
  double fM = 0.0;
  if (f32) { qxf = (float)qx; qyf = (float)qy; qzf = (float)qz; fM = f32_magnitude(g, qx, qy, qz); thr = f32_threshold(best, fM); }
  for (int r0 = 0; r0 < nrows; r0 += kLanes) {
    const int r = r0 + lane;
    int s = 0, cnt = 0;
    int hxa = 0, hxb = -1;   // x extent of a row that holds refined cells
    if (r < nrows) {
      const int rz = __float2int_rz(__fdividef((float)r + 0.5f, (float)ny));   // r / ny without the integer-division sequence
      const int y = y0 + (r - rz * ny), z = z0 + rz;
      const double rd2 = slab_d2(g, 1, qy, y, y) + slab_d2(g, 2, qz, z, z);
      if (!(rd2 > best)) {
        int xa = x0, xb = x1;
        if (best < 1e300) {
          const double w = sqrt(best - rd2);
          xa = max(x0, (int)floor((qx - w - g.lo[0]) * g.inv_h[0] - 1e-6));
          xb = min(x1, (int)floor((qx + w - g.lo[0]) * g.inv_h[0] + 1e-6));
        }
        if (xa <= xb) {
          const int rowBase = (z * g.G[1] + y) * g.G[0];
          s = __ldg(&g.cellStart[rowBase + xa]);
          cnt = __ldg(&g.cellStart[rowBase + xb + 1]) - s;
          if (TOP && g.heavyPrefix && cnt > kHeavy &&
              __ldg(&g.heavyPrefix[rowBase + xb + 1]) != __ldg(&g.heavyPrefix[rowBase + xa])) {
            cnt = 0; hxa = xa; hxb = xb;
          }
        }
      }
    }
    const int total = for_each_packed(s, cnt, base, 0x7fffffff, [](int) {}, [&](bool valid, int pos, int) {
      double d2 = best;
      int id = 0x7fffffff;
      if (f32) {
        if (valid) {
          const float4 pf = g.sites32[pos];
          const float fx = qxf - pf.x, fy = qyf - pf.y, fz = qzf - pf.z;
          valid = fx * fx + fy * fy + fz * fz <= thr;   // else: farther than the bound, whatever fp64 would say
        }
        const unsigned pass = __ballot_sync(kFull, valid);
        extra_cnt_add(5, (unsigned)__popc(pass));
      }
      if (valid) {
        const double4 p = g.sites[pos];
        const double dx = qx - p.x, dy = qy - p.y, dz = qz - p.z;
        d2 = dx * dx + dy * dy + dz * dz;
        if (has_weights(g)) d2 += __ldg(&g.sitesW[pos]);
        id = (int)(__double_as_longlong(p.w) & 0x7fffffff);
      }
      const bool better = valid && closer(d2, id, best, bestId) && !(SKIP && id == st.skip);
      if (__any_sync(kFull, better)) {
        if (!better) { d2 = best; id = bestId; }
        warp_argmin(d2, id);
        best = d2;
        bestId = id;
        if (f32) thr = f32_threshold(best, fM);
      }
    });
    VD_STAT(st.dist_evals += (unsigned)total;)
    if (TOP) {
      unsigned hm = __ballot_sync(kFull, hxa <= hxb);
      while (hm) {
        const int src = __ffs(hm) - 1;
        hm &= hm - 1;
        const int rr = r0 + src;
        const int y = y0 + rr % ny, z = z0 + rr / ny;
        const int xa = shfl(hxa, src), xb = shfl(hxb, src);
        for (int x = xa; x <= xb; ++x) scan_cell<SKIP>(g, x, y, z, qx, qy, qz, best, bestId, st);
      }
    }
  }
}

// One GridIndex per warp in shared memory: the view of a refined cell's sub-grid that a query (or a batch of queries,
// or a one-shot search) works in.  (As a local variable it lived in local memory: the struct is passed by reference
// to functions that are not inlined.)
static __shared__ GridIndex sView[kWarpsPerBlock];

__device__ __forceinline__ GridIndex& warp_view() { return sView[(threadIdx.x / kLanes) % kWarpsPerBlock]; }

// Is the ball (q, r) strictly inside cell (cx, cy, cz) of g (with a margin against the rounding of cell assignment)?
__device__ __forceinline__ bool ball_in_cell(const GridIndex& g, int cx, int cy, int cz, double qx, double qy, double qz, double r) {
  const int cc[3] = {cx, cy, cz};
  const double q[3] = {qx, qy, qz};
  bool in = r < 1e150;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    if (g.h[a] > 0) {
      const double lo = g.lo[a] + cc[a] * g.h[a], m = 1e-6 * g.h[a];
      in = in && (q[a] - r > lo + m) && (q[a] + r < lo + g.h[a] - m);
    }
  }
  return in;
}

// View of a refined cell's sub-grid as a grid of its own.
__device__ __forceinline__ void sub_view(const GridIndex& g, int x, int y, int z, int so, GridIndex& v) {
  const int K = so >> 26;
  const int cc[3] = {x, y, z};
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const int Ka = g.h[a] > 0 ? K : 1;
    v.lo[a] = g.lo[a] + cc[a] * g.h[a];
    v.h[a] = g.h[a] * (1.0 / Ka);
    v.inv_h[a] = Ka * g.inv_h[a];
    v.hi[a] = v.lo[a] + g.h[a];
    v.G[a] = Ka;
  }
  v.n = 0;
  v.cellStart = g.subStart + (so & 0x3ffffff);
  v.sites = g.sites;
  v.heavyPrefix = nullptr; v.subOff = nullptr; v.subStart = nullptr; v.countAlg = 0; v.delta = nullptr; v.stepMode = 0;
  v.sitesW = g.sitesW; v.siteWid = g.siteWid; v.sites32 = g.sites32; v.f32M = g.f32M;
}

// One cell of the top grid: a plain cell is scanned directly, a refined cell through its sub-grid,
// restricted to the ball (q, sqrt(best)).
template <bool SKIP>
static __device__ __noinline__ void scan_cell(const GridIndex& g, int x, int y, int z, double qx, double qy, double qz, double& best,
                                              int& bestId, StRef st) {
  const int c = (z * g.G[1] + y) * g.G[0] + x;
  if (slab_d2(g, 0, qx, x, x) + slab_d2(g, 1, qy, y, y) + slab_d2(g, 2, qz, z, z) > best) return;
  const int so = __ldg(&g.subOff[c]);
  if (so < 0) {
    scan_box<false, SKIP>(g, qx, qy, qz, x, x, y, y, z, z, best, bestId, st);   // plain cell: a 1 x 1 x 1 box of the top grid
    return;
  }
  GridIndex& v = warp_view();
  __syncwarp();
  if (lane_id() == 0) sub_view(g, x, y, z, so, v);
  __syncwarp();
  int vx0 = 0, vx1 = v.G[0] - 1, vy0 = 0, vy1 = v.G[1] - 1, vz0 = 0, vz1 = v.G[2] - 1;
  if (best < 1e300) {
    const double r = sqrt(best);
    vx0 = cell_of(v, 0, qx - r - 1e-6 * v.h[0]); vx1 = cell_of(v, 0, qx + r + 1e-6 * v.h[0]);
    vy0 = cell_of(v, 1, qy - r - 1e-6 * v.h[1]); vy1 = cell_of(v, 1, qy + r + 1e-6 * v.h[1]);
    vz0 = cell_of(v, 2, qz - r - 1e-6 * v.h[2]); vz1 = cell_of(v, 2, qz + r + 1e-6 * v.h[2]);
  }
  scan_box<false, SKIP>(v, qx, qy, qz, vx0, vx1, vy0, vy1, vz0, vz1, best, bestId, st);
}

// D_alg: the sites stored in the grid cells (sub-cells of refined cells) that meet the ball (q, sqrt(r2)) --
// the least any exact search over this index examines.  One THREAD per query; measurement runs only (vd_options.count_alg).
static __device__ __noinline__ unsigned ball_sites(const GridIndex& g, double qx, double qy, double qz, double r2) {
  if (!(r2 < 1e300)) return (unsigned)g.n;
  const double r = sqrt(r2);
  const int y0 = cell_of(g, 1, qy - r), y1 = cell_of(g, 1, qy + r), z0 = cell_of(g, 2, qz - r), z1 = cell_of(g, 2, qz + r);
  const int x0 = cell_of(g, 0, qx - r), x1 = cell_of(g, 0, qx + r);
  unsigned total = 0;
  for (int z = z0; z <= z1; ++z)
    for (int y = y0; y <= y1; ++y) {
      const double rd2 = slab_d2(g, 1, qy, y, y) + slab_d2(g, 2, qz, z, z);
      if (rd2 > r2) continue;
      const double w = sqrt(r2 - rd2);
      const int xa = max(x0, cell_of(g, 0, qx - w)), xb = min(x1, cell_of(g, 0, qx + w));
      if (xa > xb) continue;
      const int rowBase = (z * g.G[1] + y) * g.G[0];
      if (!g.subOff) { total += (unsigned)(g.cellStart[rowBase + xb + 1] - g.cellStart[rowBase + xa]); continue; }
      for (int x = xa; x <= xb; ++x) {
        const int so = g.subOff[rowBase + x];
        const unsigned cnt = (unsigned)(g.cellStart[rowBase + x + 1] - g.cellStart[rowBase + x]);
        if (so < 0) { total += cnt; continue; }
        GridIndex v;
        sub_view(g, x, y, z, so, v);
        const int sx0 = cell_of(v, 0, qx - r), sx1 = cell_of(v, 0, qx + r), sy0 = cell_of(v, 1, qy - r), sy1 = cell_of(v, 1, qy + r);
        const int sz0 = cell_of(v, 2, qz - r), sz1 = cell_of(v, 2, qz + r);
        if (sx0 == 0 && sy0 == 0 && sz0 == 0 && sx1 == v.G[0] - 1 && sy1 == v.G[1] - 1 && sz1 == v.G[2] - 1) { total += cnt; continue; }
        for (int sz = sz0; sz <= sz1; ++sz)
          for (int sy = sy0; sy <= sy1; ++sy) {
            const double sd2 = slab_d2(v, 1, qy, sy, sy) + slab_d2(v, 2, qz, sz, sz);
            if (sd2 > r2) continue;
            const double sw = sqrt(r2 - sd2);
            const int sa = max(sx0, cell_of(v, 0, qx - sw)), sb = min(sx1, cell_of(v, 0, qx + sw));
            if (sa > sb) continue;
            const int sb0 = (sz * v.G[1] + sy) * v.G[0];
            total += (unsigned)(v.cellStart[sb0 + sb + 1] - v.cellStart[sb0 + sa]);
          }
      }
    }
  return total;
}

// N_q: the site nearest to q among those closer than the incoming (best, bestId); ties to
// the lowest id (reading U5).  Call with best = +inf, bestId = INT_MAX for an unbounded query, or
// with best = |q - v_i|^2, bestId = i for a point-in-cell test (Eq. 2).
// nearer_ok: the caller only needs SOME site clearly nearer than the incoming bound when one exists (a
// corner that is outside Omega_i, an intermediate step of the bisector search): the routine then returns as
// soon as the cells around q have produced one, without proving it the nearest (reading U17).  When no
// site is clearly nearer, the full scan runs and the answer is exact, so acceptance is always exact.
#ifndef VD_MAX_SHELLS
#define VD_MAX_SHELLS 0   // measured on C3: unlimited 382 ms, 4 shells 361, 2: 348, 1: 337, 0 (the home cell only): 324
#endif
template <bool HV, bool SKIP>
static __device__ __noinline__ void nearest_impl(const GridIndex& g, double qx, double qy, double qz, double& best, int& bestId,
                                             StRef st, bool nearer_ok);

template <bool HV, bool SKIP = false>
__device__ __forceinline__ void nearest(const GridIndex& g, double qx, double qy, double qz, double& best, int& bestId,
                                        StRef st, bool nearer_ok = false) {
  nearest_impl<HV, SKIP>(g, qx, qy, qz, best, bestId, st, nearer_ok);
  if (counts_alg(g)) {
    if (lane_id() == 0) sExtraCnt[(threadIdx.x / kLanes) % kWarpsPerBlock][4] += ball_sites(g, qx, qy, qz, best);
    __syncwarp();
  }
}

template <bool HV, bool SKIP>
static __device__ __noinline__ void nearest_impl(const GridIndex& g, double qx, double qy, double qz, double& best, int& bestId,
                                             StRef st, bool nearer_ok) {
  const double bound0 = best;
  VD_STAT(st.queries += 1;)
  const int cx = cell_of(g, 0, qx), cy = cell_of(g, 1, qy), cz = cell_of(g, 2, qz);
  if (HV) {
    // Refined home cell (dense cluster): work in its sub-grid.  If the ball lies inside the home cell,
    // the sub-grid alone decides; a loose bound is first tightened on the 3 x 3 x 3 sub-cells around q.
    const int so = __ldg(&g.subOff[(cz * g.G[1] + cy) * g.G[0] + cx]);
    if (so >= 0) {
      GridIndex& v = warp_view();
      __syncwarp();
      if (lane_id() == 0) sub_view(g, cx, cy, cz, so, v);
      __syncwarp();
#pragma unroll 1   // (code size: the refined-index kernels are instruction-fetch bound)
      for (int pass = 0; pass < 2; ++pass) {
        if (best < 1e300) {
          const double r = sqrt(best);
          bool in = true;
#pragma unroll
          for (int a = 0; a < 3; ++a) {
            const double qa = a == 0 ? qx : (a == 1 ? qy : qz);
            if (g.h[a] > 0) in = in && (qa - r > v.lo[a] + 1e-6 * g.h[a]) && (qa + r < v.hi[a] - 1e-6 * g.h[a]);
            else in = in && (r < 1e300);
          }
          const int vx0 = cell_of(v, 0, qx - r - 1e-6 * v.h[0]), vx1 = cell_of(v, 0, qx + r + 1e-6 * v.h[0]);
          const int vy0 = cell_of(v, 1, qy - r - 1e-6 * v.h[1]), vy1 = cell_of(v, 1, qy + r + 1e-6 * v.h[1]);
          const int vz0 = cell_of(v, 2, qz - r - 1e-6 * v.h[2]), vz1 = cell_of(v, 2, qz + r + 1e-6 * v.h[2]);
          if (in && (vy1 - vy0 + 1) * (vz1 - vz0 + 1) <= kLanes) {
            scan_box<false, SKIP>(v, qx, qy, qz, vx0, vx1, vy0, vy1, vz0, vz1, best, bestId, st);
            return;
          }
        }
        if (pass == 0) {
          const int hx = cell_of(v, 0, qx), hy = cell_of(v, 1, qy), hz = cell_of(v, 2, qz);
          scan_box<false, SKIP>(v, qx, qy, qz, max(hx - 1, 0), min(hx + 1, v.G[0] - 1), max(hy - 1, 0), min(hy + 1, v.G[1] - 1),
                          max(hz - 1, 0), min(hz + 1, v.G[2] - 1), best, bestId, st);
          if (nearer_ok && best < bound0 * (1.0 - 1e-9)) return;
        }
      }
    }
  }
  // how far q lies outside the grid box on each axis
  const double ox = fmax(fmax(g.lo[0] - qx, qx - g.hi[0]), 0.0);
  const double oy = fmax(fmax(g.lo[1] - qy, qy - g.hi[1]), 0.0);
  const double oz = fmax(fmax(g.lo[2] - qz, qz - g.hi[2]), 0.0);
  bool needSeed = !(best < 1e300);  // callers pass best >= 2e300 for "unbounded"
  if (!needSeed) {
    // rows of the ball's bounding box; a loose bound is first tightened around the home cell
    const double r = sqrt(best);
    const double ry = 2.0 * r * g.inv_h[1] + 2.0, rz = 2.0 * r * g.inv_h[2] + 2.0;
    needSeed = ry * rz > 16.0;
  }
  if (needSeed) {
    // expanding shells around the (clamped) home cell until some site is known (sb, si); then the
    // ball's box below decides.  Stops at once when no unscanned cell can beat the bound.
    double sb = 2e300;
    int si = 0x7fffffff;
    bool done = false;
    const int smax = max(g.G[0], max(g.G[1], g.G[2]));
    for (int s = 0; s <= smax; ++s) {
      if (s > 0) {
        // lower bound of the distance to any cell outside the box of radius s-1 (faces that lie
        // beyond the grid hold no cells)
        double lb = 2e300;
        const int k = s - 1;
        const double o2 = ox * ox + oy * oy + oz * oz;
        auto axis_bound = [&](int a) {
          const int ca = a == 0 ? cx : (a == 1 ? cy : cz);
          const double qa = a == 0 ? qx : (a == 1 ? qy : qz), oa = a == 0 ? ox : (a == 1 ? oy : oz);
          const double rest = o2 - oa * oa;   // how far q lies outside the grid box on the other two axes
          if (ca - k > 0) lb = fmin(lb, slab_d2(g, a, qa, 0, ca - k - 1) + rest);
          if (ca + k < g.G[a] - 1) lb = fmin(lb, slab_d2(g, a, qa, ca + k + 1, g.G[a] - 1) + rest);
        };
        // rolled in the refined-index kernels only: they are bound by instruction fetch (75 KB of code), the
        // plain-index kernels by the instructions they execute
        if constexpr (HV) {
#pragma unroll 1
          for (int a = 0; a < 3; ++a) axis_bound(a);
        } else {
          axis_bound(0); axis_bound(1); axis_bound(2);
        }
        if (lb > fmin(best, sb)) { done = true; break; }
        if (sb < 1e300) break;
        // a bounded query that found nothing in the first shells (a corner in a void, most often inside its cell): the box
        // scan of the ball below visits the same cells 32 rows at a time, with rows pruned and x-extents tightened -- the
        // shells would visit them face by face
        if (s > VD_MAX_SHELLS && best < 1e300) break;
      }
      // shell s: rows with max(|dy|,|dz|) == s take the full x extent, inner rows the two end cells
      const int y0 = max(cy - s, 0), y1 = min(cy + s, g.G[1] - 1);
      const int z0 = max(cz - s, 0), z1 = min(cz + s, g.G[2] - 1);
      const int xl = cx - s, xr = cx + s;
      const int xa = max(xl, 0), xb = min(xr, g.G[0] - 1);
      // the shell's faces: z = cz -+ s, then y = cy -+ s between them, then x = cx -+ s inside both (through ONE call
      // site in the refined-index kernels: six inlined call sequences are 3 KB of code)
      const int zi0 = max(cz - s + 1, 0), zi1 = min(cz + s - 1, g.G[2] - 1);
      const int yi0 = max(cy - s + 1, 0), yi1 = min(cy + s - 1, g.G[1] - 1);
      auto face = [&](int f) {
        int bx0 = xa, bx1 = xb, by0 = y0, by1 = y1, bz0 = z0, bz1 = z1;
        bool ok = true;
        if (s > 0) {
          if (f < 2) {
            const int z = f == 0 ? cz - s : cz + s;
            ok = z >= 0 && z < g.G[2];
            bz0 = z; bz1 = z;
          } else if (f < 4) {
            const int y = f == 2 ? cy - s : cy + s;
            ok = y >= 0 && y < g.G[1] && zi0 <= zi1;
            by0 = y; by1 = y; bz0 = zi0; bz1 = zi1;
          } else {
            const int x = f == 4 ? xl : xr;
            ok = x >= 0 && x < g.G[0] && zi0 <= zi1 && yi0 <= yi1;
            bx0 = x; bx1 = x; by0 = yi0; by1 = yi1; bz0 = zi0; bz1 = zi1;
          }
        }
        if (ok) scan_box<HV, SKIP>(g, qx, qy, qz, bx0, bx1, by0, by1, bz0, bz1, sb, si, st);
      };
      if constexpr (HV) {
        const int nf = s == 0 ? 1 : 6;
#pragma unroll 1
        for (int f = 0; f < nf; ++f) face(f);
      } else {
        face(0);
        if (s > 0) { face(1); face(2); face(3); face(4); face(5); }
      }
    }
    if (closer(sb, si, best, bestId)) { best = sb; bestId = si; }
    if (done || !(best < 1e300)) return;
  }
  if (nearer_ok && best < bound0 * (1.0 - 1e-9)) return;
  // the ball (q, sqrt(best)) decides: scan its bounding box of cells, rows pruned as best shrinks
  const double r = sqrt(best);
  const int x0 = cell_of(g, 0, qx - r - 1e-6 * g.h[0]), x1 = cell_of(g, 0, qx + r + 1e-6 * g.h[0]);
  const int y0 = cell_of(g, 1, qy - r - 1e-6 * g.h[1]), y1 = cell_of(g, 1, qy + r + 1e-6 * g.h[1]);
  const int z0 = cell_of(g, 2, qz - r - 1e-6 * g.h[2]), z1 = cell_of(g, 2, qz + r + 1e-6 * g.h[2]);
  scan_box<HV, SKIP>(g, qx, qy, qz, x0, x1, y0, y1, z0, z1, best, bestId, st);
}

}  // namespace vd
