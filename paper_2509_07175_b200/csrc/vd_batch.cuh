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
// rows of a query's ball above which it takes the single-query path: 32, and 64 on the top grid of a refined index (measured:
// 8 / 16 / 32 / 64 rows: C3 405 / 324 / 311 / 306 ms, C5 16.2 / 16.3 / 16.2 / 18.1 ms, C2 21.1 / 20.2 / 20.2 / 20.2 ms)
#ifndef VD_QB_ROWS
#define VD_QB_ROWS 32
#endif
#ifndef VD_QB_ROWS_REFINED
#define VD_QB_ROWS_REFINED 64
#endif
#ifndef VD_QB_ROWS_PLANAR
#define VD_QB_ROWS_PLANAR 16
#endif
constexpr int kQBMaxRows = VD_QB_ROWS, kQBMaxRowsPlanar = VD_QB_ROWS_PLANAR, kQBMaxRowsRefined = VD_QB_ROWS_REFINED;   // (planar grid, C1: 16 rows 1.05 ms, 32 rows 1.23 ms --
// the batched pass has no early exit, and a bare triangle's corners have loose bounds in a dense grid)

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
  float qf[kQB][4];          // fp32 filter: the query in float, and the fp32 threshold of its current bound
};

// One pass of the batch over ONE grid view g (the top grid, the sub-grid of a refined cell, or a single plain cell seen as a
// 1 x 1 x 1 grid): the queries named in `active` enumerate the rows of g that their balls meet, the candidates of all rows
// are packed 32 per round.  SKIP_REFINED (top grid of a refined index): a row that holds a refined cell is not scanned; the
// query is flagged (B.flag) and that row is visited cell by cell afterwards.  A query whose ball spans more than
// kQBMaxRows rows of g does not take part: it is returned in the mask of loose queries.
template <bool SKIP_REFINED>
static __device__ __noinline__ unsigned batch_pass(const GridIndex& g, QBatch& B, int nq, unsigned active, StRef st) {
  const int lane = lane_id();
  int myRows = 0;
  bool loose = false;
  const bool f32 = has_f32(g) && !has_weights(g);
  if (f32 && lane < nq) {
    const double qx = B.qx[lane], qy = B.qy[lane], qz = B.qz[lane];
    B.qf[lane][0] = (float)qx; B.qf[lane][1] = (float)qy; B.qf[lane][2] = (float)qz;
    B.qf[lane][3] = f32_threshold(B.best[lane], f32_magnitude(g, qx, qy, qz));
  }
  if (lane < nq && ((active >> lane) & 1u)) {
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
      if (myRows > (SKIP_REFINED ? kQBMaxRowsRefined : (g.h[2] > 0 ? kQBMaxRows : kQBMaxRowsPlanar))) { loose = true; myRows = 0; }
    }
  }
  const int incl = warp_incl_scan(myRows);
  if (lane < nq) B.rowStart[lane] = incl - myRows;
  if (lane == nq - 1) B.rowStart[nq] = incl;
  const unsigned looseMask = __ballot_sync(kFull, loose);
  __syncwarp();
  const int R = B.rowStart[nq];
  VD_STAT(st.rows += (unsigned)R;)
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
        if (SKIP_REFINED && cnt > kHeavy &&
            __ldg(&g.heavyPrefix[rowBase + B.x1[u] + 1]) != __ldg(&g.heavyPrefix[rowBase + B.x0[u]])) {
          cnt = 0;           // a refined cell in this row
          B.flag[u] = 1;
        }
      }
    }
    const int total = for_each_packed(s, cnt, B.base, 0x7fffffff, [&](int slot) { B.qid[slot] = (unsigned char)u; },
                                      [&](bool valid, int pos, int owner) {
      double d2 = 0.0;
      int id = 0x7fffffff, cu = 0;
      bool better = false;
      if (valid) cu = B.qid[owner];
      if (f32) {
        if (valid) {
          const float4 pf = g.sites32[pos];
          const float fx = B.qf[cu][0] - pf.x, fy = B.qf[cu][1] - pf.y, fz = B.qf[cu][2] - pf.z;
          valid = fx * fx + fy * fy + fz * fz <= B.qf[cu][3];   // else: farther than its query's bound, whatever fp64 would say
        }
        extra_cnt_add(5, (unsigned)__popc(__ballot_sync(kFull, valid)));
      }
      if (valid) {
        const double4 p = g.sites[pos];
        const double dx = B.qx[cu] - p.x, dy = B.qy[cu] - p.y, dz = B.qz[cu] - p.z;
        d2 = dx * dx + dy * dy + dz * dz;
        if (has_weights(g)) d2 += __ldg(&g.sitesW[pos]);
        id = (int)(__double_as_longlong(p.w) & 0x7fffffff);
        better = closer(d2, id, B.best[cu], B.bestId[cu]);
      }
      unsigned m = __ballot_sync(kFull, better);
      while (m) {   // rare: a candidate beats its query's bound; apply one at a time, re-test the rest
        const int src = __ffs(m) - 1;
        const int bu = shfl(cu, src), bi = shfl(id, src);
        const double bd = shfl(d2, src);
        if (lane == 0 && closer(bd, bi, B.best[bu], B.bestId[bu])) {
          B.best[bu] = bd; B.bestId[bu] = bi;
          if (f32) B.qf[bu][3] = f32_threshold(bd, f32_magnitude(g, B.qx[bu], B.qy[bu], B.qz[bu]));
        }
        __syncwarp();
        better = better && lane != src && closer(d2, id, B.best[cu], B.bestId[cu]);
        m = __ballot_sync(kFull, better);
      }
    });
    VD_STAT(st.dist_evals += (unsigned)total;)
  }
  return looseMask;
}

// Lanes 0..nq-1 have filled qx,qy,qz,best,bestId of their slot (and the warp has synchronised).  On
// return best/bestId of every slot hold the nearest site among those closer than the incoming bound
// (or, for a loose bound, some clearly nearer site: nearer_ok of nearest(), reading U17).
//
// Refined index (HV): the corners of a piece inside a dense cluster sit in refined cells, and their balls usually reach
// into a neighbouring cell -- refined as well, or plain.  Pass A runs on the top grid and scans the rows made of plain
// cells only; pass B then visits, one after the other, the top cells of the rows pass A left out: a refined cell through
// its sub-grid, a plain one as a 1 x 1 x 1 grid, each as a view that the same batched pass runs on, for the queries
// whose ball meets that cell.  Only a query whose ball spans many rows (a corner in the void between clusters) takes the
// single-query path.
//
// FALLBACK = false: the queries that would take the single-query path are NOT answered; their mask is returned (bit u = query
// u) and the routine carries no call of nearest(): the refined-index step kernels exist in a fast form without that code --
// the expanding-shell search is a third of their instructions and half of their executed code, and they are bound by
// instruction fetch -- and a second pass of the same kernels (with the fallback) takes what the fast pass left.
template <bool HV, bool FALLBACK = true>
static __device__ __noinline__ unsigned batch_nearest(const GridIndex& gTop, QBatch& B, int nq, StRef st) {
  const int lane = lane_id();
  if (lane < kQB) B.flag[lane] = 0;
  __syncwarp();
  unsigned looseMask = batch_pass<HV>(gTop, B, nq, (1u << nq) - 1u, st);
  if (HV) {
    __syncwarp();
    const bool mine = lane < nq && B.flag[lane] != 0 && !((looseMask >> lane) & 1u);
    const unsigned flagged = __ballot_sync(kFull, mine);
    if (flagged) {
      // my ball's box in the top grid (pass A left it in B), and the union over the flagged queries
      int tx0 = 0x7fffffff, tx1 = -1, ty0 = 0x7fffffff, ty1 = -1, tz0 = 0x7fffffff, tz1 = -1;
      if (mine) {
        tx0 = B.x0[lane]; tx1 = B.x1[lane]; ty0 = B.y0[lane]; ty1 = ty0 + B.ny[lane] - 1;
        const double r = sqrt(B.best[lane]);
        tz0 = B.z0[lane]; tz1 = cell_of(gTop, 2, B.qz[lane] + r + 1e-6 * gTop.h[2]);
      }
      const int ux0 = __reduce_min_sync(kFull, tx0), ux1 = __reduce_max_sync(kFull, tx1);
      const int uy0 = __reduce_min_sync(kFull, ty0), uy1 = __reduce_max_sync(kFull, ty1);
      const int uz0 = __reduce_min_sync(kFull, tz0), uz1 = __reduce_max_sync(kFull, tz1);
      if ((ux1 - ux0 + 1) * (uy1 - uy0 + 1) * (uz1 - uz0 + 1) > 64) {
        looseMask |= flagged;   // (the flagged queries are far apart: not worth a cell-by-cell visit)
      } else {
        GridIndex& v = warp_view();
        for (int z = uz0; z <= uz1; ++z)
          for (int y = uy0; y <= uy1; ++y) {
            const int rowBase = (z * gTop.G[1] + y) * gTop.G[0];
            // was this row left out for me in pass A?  (it holds a refined cell within my x range)
            bool rowMine = mine && y >= ty0 && y <= ty1 && z >= tz0 && z <= tz1;
            if (rowMine) rowMine = __ldg(&gTop.heavyPrefix[rowBase + tx1 + 1]) != __ldg(&gTop.heavyPrefix[rowBase + tx0]);
            if (!__any_sync(kFull, rowMine)) continue;
            for (int x = ux0; x <= ux1; ++x) {
              bool p = rowMine && x >= tx0 && x <= tx1;
              if (p) p = !(slab_d2(gTop, 0, B.qx[lane], x, x) + slab_d2(gTop, 1, B.qy[lane], y, y) + slab_d2(gTop, 2, B.qz[lane], z, z) > B.best[lane]);
              const unsigned pm = __ballot_sync(kFull, p);
              if (!pm) continue;
              const int c = rowBase + x;
              if (__ldg(&gTop.cellStart[c + 1]) == __ldg(&gTop.cellStart[c])) continue;   // an empty cell
              __syncwarp();
              if (lane == 0) {
                const int so = __ldg(&gTop.subOff[c]);
                if (so >= 0) {
                  sub_view(gTop, x, y, z, so, v);
                } else {   // a plain cell as a grid of one cell
                  const int cc[3] = {x, y, z};
                  for (int a = 0; a < 3; ++a) {
                    v.lo[a] = gTop.lo[a] + cc[a] * gTop.h[a]; v.h[a] = gTop.h[a]; v.inv_h[a] = gTop.inv_h[a];
                    v.hi[a] = v.lo[a] + gTop.h[a]; v.G[a] = 1;
                  }
                  v.n = 0; v.cellStart = gTop.cellStart + c; v.sites = gTop.sites;
                  v.heavyPrefix = nullptr; v.subOff = nullptr; v.subStart = nullptr; v.countAlg = 0; v.delta = nullptr; v.stepMode = 0;
                  v.sitesW = gTop.sitesW; v.siteWid = gTop.siteWid; v.sites32 = gTop.sites32; v.f32M = gTop.f32M;
                }
              }
              __syncwarp();
              looseMask |= batch_pass<false>(v, B, nq, pm, st);   // (a ball of many sub-rows: the single-query path finishes it)
            }
          }
      }
    }
  }
  VD_STAT(st.queries += (unsigned)(nq - __popc(looseMask));)
  if (counts_alg(gTop)) {
    // D_alg of the batched queries (the loose ones count inside nearest())
    unsigned v = 0;
    if (lane < nq && !((looseMask >> lane) & 1u)) v = ball_sites(gTop, B.qx[lane], B.qy[lane], B.qz[lane], B.best[lane]);
    v = (unsigned)warp_sum((int)v);
    extra_cnt_add(4, v);
  }
#ifdef VD_COUNT_LOOSE
  extra_cnt_add(3, (unsigned)__popc(looseMask));   // (experiment: reported as step_probes)
#endif
  if constexpr (!FALLBACK) {
    return looseMask;
  } else {
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
    return 0u;
  }
}

}  // namespace vd
