// vd_batch.cuh -- S2, batched: the point-in-cell tests of up to kQB unclassified corners of ONE piece
// answered in one pass of the warp.  The corners created by a clip are independent queries
// of ~30 candidate sites in 4-9 grid rows each; one at a time they leave most lanes idle and repeat the
// uniform bookkeeping.  Together, the rows of all queries share one row pass and their candidates are
// packed 32 per round.  Same bound / tie rule / exactness as nearest() (vd_nearest.cuh); a query whose
// ball spans many rows takes that single-query path.
#pragma once
#include "vd_nearest.cuh"

namespace vd {

constexpr int kQB = 8;          // queries per batch
constexpr int kQBMaxRows = 16;  // rows of a query's ball above which it takes the single-query path

struct QBatch {
  double qx[kQB], qy[kQB], qz[kQB];
  double best[kQB];     // in: bound d^2; out: distance^2 of N_q
  int bestId[kQB];      // in: site of the bound; out: N_q
  int x0[kQB], x1[kQB], y0[kQB], ny[kQB], z0[kQB];
  int rowStart[kQB + 1];
  int item[kQB];        // caller's payload (corner index)
  int base[kLanes];     // per packed row: first site index minus first candidate index
  unsigned char qid[kLanes];
  unsigned char flag[kQB];   // refined index: the query met a refined cell in the row pass
};

// Lanes 0..nq-1 have filled qx,qy,qz,best,bestId of their slot (and the warp has synchronised).  On
// return best/bestId of every slot hold the nearest site among those closer than the incoming bound
// (or, for a loose bound, some clearly nearer site: nearer_ok of nearest(), reading U17).
//
// Refined index (HV): the batched pass needs plain cells.  Two cases keep it: (a) the balls of ALL queries lie inside one
// and the same refined cell (a piece inside a dense cluster: its corners are a few sub-cells apart) -- then the pass runs
// on that cell's sub-grid, viewed as a grid of its own; (b) no row of a query's ball holds a refined cell (found in the
// row pass from the prefix count of refined cells) -- then the top grid is plain for that query.  Every other query
// takes the single-query path.
template <bool HV>
static __device__ __noinline__ void batch_nearest(const GridIndex& gTop, QBatch& B, int nq, QueryStats& st) {
  const int lane = lane_id();
  const GridIndex* gp = &gTop;
  bool checkRefined = false;
  if (HV) {
    checkRefined = true;
    int c = -1;
    bool ok = false;
    int hx = 0, hy = 0, hz = 0;
    if (lane < nq && B.best[lane] < 1e300) {
      const double qx = B.qx[lane], qy = B.qy[lane], qz = B.qz[lane];
      hx = cell_of(gTop, 0, qx); hy = cell_of(gTop, 1, qy); hz = cell_of(gTop, 2, qz);
      c = (hz * gTop.G[1] + hy) * gTop.G[0] + hx;
      ok = __ldg(&gTop.subOff[c]) >= 0 && ball_in_cell(gTop, hx, hy, hz, qx, qy, qz, sqrt(B.best[lane]));
    }
    const int c0 = shfl(c, 0);
    if (__all_sync(kFull, lane >= nq || (ok && c == c0))) {
      GridIndex& v = warp_view();
      __syncwarp();
      if (lane == 0) sub_view(gTop, hx, hy, hz, __ldg(&gTop.subOff[c]), v);
      __syncwarp();
      gp = &v;
      checkRefined = false;
    }
  }
  const GridIndex& g = *gp;
  int myRows = 0;
  bool loose = false;
  if (lane < kQB) B.flag[lane] = 0;
  if (lane < nq) {
    const double b = B.best[lane];
    if (!(b < 1e300)) {
      loose = true;
    } else {
      const double r = sqrt(b);
      const double qx = B.qx[lane], qy = B.qy[lane], qz = B.qz[lane];
      const int x0 = cell_of(g, 0, qx - r - 1e-6 * g.h[0]), x1 = cell_of(g, 0, qx + r + 1e-6 * g.h[0]);
      const int y0 = cell_of(g, 1, qy - r - 1e-6 * g.h[1]), y1 = cell_of(g, 1, qy + r + 1e-6 * g.h[1]);
      const int z0 = cell_of(g, 2, qz - r - 1e-6 * g.h[2]), z1 = cell_of(g, 2, qz + r + 1e-6 * g.h[2]);
      myRows = (y1 - y0 + 1) * (z1 - z0 + 1);
      B.x0[lane] = x0; B.x1[lane] = x1; B.y0[lane] = y0; B.ny[lane] = y1 - y0 + 1; B.z0[lane] = z0;
      if (myRows > kQBMaxRows) { loose = true; myRows = 0; }
    }
  }
  const int incl = warp_incl_scan(myRows);
  if (lane < nq) B.rowStart[lane] = incl - myRows;
  if (lane == nq - 1) B.rowStart[nq] = incl;
  unsigned looseMask = __ballot_sync(kFull, loose);
  st.queries += (unsigned)(nq - __popc(looseMask));
  __syncwarp();
  const int R = B.rowStart[nq];
  st.rows += (unsigned)R;
  for (int r0 = 0; r0 < R; r0 += kLanes) {
    const int rho = r0 + lane;
    int s = 0, cnt = 0, u = 0;
    if (rho < R) {
      while (u + 1 < nq && B.rowStart[u + 1] <= rho) ++u;
      const int r = rho - B.rowStart[u];
      const int ny = B.ny[u];
      const int rz = __float2int_rz(__fdividef((float)r + 0.5f, (float)ny));
      const int y = B.y0[u] + (r - rz * ny), z = B.z0[u] + rz;
      const double rd2 = slab_d2(g, 1, B.qy[u], y, y) + slab_d2(g, 2, B.qz[u], z, z);
      if (!(rd2 > B.best[u])) {
        const int rowBase = (z * g.G[1] + y) * g.G[0];
        s = __ldg(&g.cellStart[rowBase + B.x0[u]]);
        cnt = __ldg(&g.cellStart[rowBase + B.x1[u] + 1]) - s;
        if (HV && checkRefined && cnt > kHeavy &&
            __ldg(&g.heavyPrefix[rowBase + B.x1[u] + 1]) != __ldg(&g.heavyPrefix[rowBase + B.x0[u]])) {
          cnt = 0;           // a refined cell in this row: the query goes to the single-query path
          B.flag[u] = 1;
        }
      }
    }
    const int pin = warp_incl_scan(cnt);
    const int excl = pin - cnt;
    const int total = shfl(pin, kLanes - 1);
    st.dist_evals += (unsigned)total;
    for (int t0 = 0; t0 < total; t0 += kLanes) {
      unsigned bit = 0;
      if (cnt > 0) {
        if (excl >= t0 && excl < t0 + kLanes) bit = 1u << (excl - t0);
        else if (excl < t0 && pin > t0) bit = 1u;
      }
      const unsigned starts = __reduce_or_sync(kFull, bit);
      const unsigned owners = __ballot_sync(kFull, bit != 0);
      if (bit) {
        const int slot = __popc(owners & ((1u << lane) - 1u));
        B.base[slot] = s - excl;
        B.qid[slot] = (unsigned char)u;
      }
      __syncwarp();
      const int t = t0 + lane;
      const bool valid = t < total;
      double d2 = 0.0;
      int id = 0x7fffffff, cu = 0;
      bool better = false;
      if (valid) {
        const int owner = __popc(starts & ((2u << lane) - 1u)) - 1;
        cu = B.qid[owner];
        const double4 p = g.sites[B.base[owner] + t];
        const double dx = B.qx[cu] - p.x, dy = B.qy[cu] - p.y, dz = B.qz[cu] - p.z;
        d2 = dx * dx + dy * dy + dz * dz;
        id = (int)(__double_as_longlong(p.w) & 0x7fffffff);
        better = closer(d2, id, B.best[cu], B.bestId[cu]);
      }
      unsigned m = __ballot_sync(kFull, better);
      while (m) {   // rare: a candidate beats its query's bound; apply one at a time, re-test the rest
        const int src = __ffs(m) - 1;
        const int bu = shfl(cu, src), bi = shfl(id, src);
        const double bd = shfl(d2, src);
        if (lane == 0 && closer(bd, bi, B.best[bu], B.bestId[bu])) { B.best[bu] = bd; B.bestId[bu] = bi; }
        __syncwarp();
        better = better && lane != src && closer(d2, id, B.best[cu], B.bestId[cu]);
        m = __ballot_sync(kFull, better);
      }
      __syncwarp();
    }
  }
  if (HV && checkRefined) {
    __syncwarp();
    const unsigned flagged = __ballot_sync(kFull, lane < nq && B.flag[lane] != 0);
    st.queries -= (unsigned)__popc(flagged & ~looseMask);
    looseMask |= flagged;
  }
  if (gTop.countAlg) {
    // D_alg of the batched queries (the loose ones count inside nearest())
    unsigned v = 0;
    if (lane < nq && !((looseMask >> lane) & 1u)) v = ball_sites(gTop, B.qx[lane], B.qy[lane], B.qz[lane], B.best[lane]);
    v = (unsigned)warp_sum((int)v);
    extra_cnt_add(4, v);
  }
  while (looseMask) {
    const int u = __ffs(looseMask) - 1;
    looseMask &= looseMask - 1;
    double best = B.best[u];
    int bestId = B.bestId[u];
    nearest<HV>(gTop, B.qx[u], B.qy[u], B.qz[u], best, bestId, st, true);
    __syncwarp();
    if (lane == 0) { B.best[u] = best; B.bestId[u] = bestId; }
    __syncwarp();
  }
}

}  // namespace vd
