// vd_clip2d.cuh -- S4 for triangles (2D domains and surface meshes): one warp computes the
// polygon P_{a,i} = T_a ∩ Omega_i.  The polygon is an ordered loop of corners, edge c runs from corner
// c to corner c+1 and carries a flag and its supporting plane (for a surface: the bisector plane,
// or the plane through a triangle edge perpendicular to the triangle).  Every corner is the solution
// of (edge plane, edge plane, triangle plane), so coordinates do not depend on the clip order.
// The nearest-site queries are warp-cooperative; the few-corner loop surgery is done by lane 0.
#pragma once
#include "vd_clip3d.cuh"

namespace vd {

template <int K>
struct Poly2 {
  double cx[K], cy[K], cz[K];
  double enx[K], eny[K], enz[K], ed[K];
  int eflag[K], cnn[K];
  unsigned char cstate[K];
  // scratch copy used while rebuilding the loop
  double tx[K], ty[K], tz[K], tnx[K], tny[K], tnz[K], td[K];
  int tflag[K], tnn[K];
  unsigned char tstate[K];
  double u[14];   // per-pair constants: origin, v_i absolute, v_i local, witness local, [12] = 0 (the additive term of 3-D power diagrams)
  int nc;
  double scratch[(kSearchScratchBytes + 7) / 8];   // the search's batch of one and its frame
};

// fallback position of a new corner (ill-conditioned planes): where the edge from the removed corner c to
// the surviving corner b meets the line, by interpolation
__device__ __forceinline__ void lerp_to_plane(double cx, double cy, double cz, double bx, double by, double bz, double nx, double ny,
                                              double nz, double d, double& x, double& y, double& z) {
  const double sc = nx * cx + ny * cy + nz * cz - d, sn = nx * bx + ny * by + nz * bz - d;
  double t = (sc - sn) > 0.0 ? sc / (sc - sn) : 0.0;
  t = fmin(fmax(t, 0.0), 1.0);
  x = cx + t * (bx - cx); y = cy + t * (by - cy); z = cz + t * (bz - cz);
}

// P <- P clipped by the line (n, d) with flag j, starting from the outside corner p; s = the known-inside neighbour
// of p when the clip comes from a search on the real edge p_s p (else -1).  The few-corner loop surgery is done by
// lane 0.  Returns 0, or 1 when the loop outgrows K.
template <int K>
__device__ __forceinline__ int apply_clip_2d(Poly2<K>& S, int p, int s, double nx, double ny, double nz, double d, int j,
                                             double pnx, double pny, double pnz) {
  const int lane = lane_id();
  const int nc = S.nc;
  __syncwarp();
  VD_WORK(extra_cnt_add(0, (unsigned)nc); extra_cnt_add(1, 2u);)
  int rc = 0;
  if (lane == 0) {
    // outside run around p (P:L391's R_p for a loop): corners beyond the line, not known inside
    int r0 = p, r1 = p, len = 1;
    while (len < nc) {
      const int q = (r0 + nc - 1) % nc;
      const double sd = nx * S.cx[q] + ny * S.cy[q] + nz * S.cz[q] - d;
      if (!(sd > 0.0 && S.cstate[q] != ST_IN)) break;
      r0 = q; ++len;
    }
    while (len < nc) {
      const int q = (r1 + 1) % nc;
      const double sd = nx * S.cx[q] + ny * S.cy[q] + nz * S.cz[q] - d;
      if (!(sd > 0.0 && S.cstate[q] != ST_IN)) break;
      r1 = q; ++len;
    }
    if (len >= nc) {
      S.nc = 0;
    } else if (nc - len + 2 > K) {
      rc = 1;
    } else {
      const int pv = (r0 + nc - 1) % nc, nxt = (r1 + 1) % nc;
      int k = 0;
      for (int c = nxt;; c = (c + 1) % nc) {   // survivors nxt .. pv keep corner and edge
        S.tx[k] = S.cx[c]; S.ty[k] = S.cy[c]; S.tz[k] = S.cz[c];
        S.tnx[k] = S.enx[c]; S.tny[k] = S.eny[c]; S.tnz[k] = S.enz[c]; S.td[k] = S.ed[c];
        S.tflag[k] = S.eflag[c]; S.tnn[k] = S.cnn[c]; S.tstate[k] = S.cstate[c];
        ++k;
        if (c == pv) break;
      }
      // X = edge(pv) ∩ B_ij : start of the new edge, which takes flag j
      if (!solve3(S.enx[pv], S.eny[pv], S.enz[pv], S.ed[pv], nx, ny, nz, d, pnx, pny, pnz, 0.0, S.tx[k], S.ty[k], S.tz[k]))
        lerp_to_plane(S.cx[r0], S.cy[r0], S.cz[r0], S.cx[pv], S.cy[pv], S.cz[pv], nx, ny, nz, d, S.tx[k], S.ty[k], S.tz[k]);
      S.tnx[k] = nx; S.tny[k] = ny; S.tnz[k] = nz; S.td[k] = d; S.tflag[k] = j; S.tnn[k] = -1;
      S.tstate[k] = (s == pv && p == r0) ? ST_IN : ST_UNKNOWN;   // on the searched real edge
      ++k;
      // E = B_ij ∩ edge(r1) : the rest of edge r1 keeps its plane and flag
      if (!solve3(nx, ny, nz, d, S.enx[r1], S.eny[r1], S.enz[r1], S.ed[r1], pnx, pny, pnz, 0.0, S.tx[k], S.ty[k], S.tz[k]))
        lerp_to_plane(S.cx[r1], S.cy[r1], S.cz[r1], S.cx[nxt], S.cy[nxt], S.cz[nxt], nx, ny, nz, d, S.tx[k], S.ty[k], S.tz[k]);
      S.tnx[k] = S.enx[r1]; S.tny[k] = S.eny[r1]; S.tnz[k] = S.enz[r1]; S.td[k] = S.ed[r1];
      S.tflag[k] = S.eflag[r1]; S.tnn[k] = -1;
      S.tstate[k] = (s == nxt && p == r1) ? ST_IN : ST_UNKNOWN;
      ++k;
      for (int c = 0; c < k; ++c) {
        S.cx[c] = S.tx[c]; S.cy[c] = S.ty[c]; S.cz[c] = S.tz[c];
        S.enx[c] = S.tnx[c]; S.eny[c] = S.tny[c]; S.enz[c] = S.tnz[c]; S.ed[c] = S.td[c];
        S.eflag[c] = S.tflag[c]; S.cnn[c] = S.tnn[c]; S.cstate[c] = S.tstate[c];
      }
      S.nc = k;
    }
  }
  rc = shfl(rc, 0);
  __syncwarp();
  return rc;
}

// ---- the fast tier (polygons of at most 32 corners: all but a handful): ONE LANE PER CORNER ------------------------------
// The loop surgery above runs on lane 0 while 31 lanes repeat its reads; pieces of 3-8 corners spent 57 % of their
// instructions there (profiles/r01_k_clip_c4.md).  Here every per-corner step is one warp-wide operation: the corners beyond
// a line are a bit mask (ballot), the outside run around p comes from two bit scans, survivors move to their new slots in
// one step, the two new corners are solved by two lanes side by side, and the point-in-cell tests of all unclassified
// corners share one batched pass (vd_batch.cuh), as in 3D.
struct Poly2P {
  double cx[kLanes], cy[kLanes], cz[kLanes];
  double enx[kLanes], eny[kLanes], enz[kLanes], ed[kLanes];
  int eflag[kLanes], cnn[kLanes];
  unsigned char cstate[kLanes];
  int k0[kLanes], k1[kLanes];                           // finish: the ascending flag pair of a corner
  double u[14];                                          // per-pair constants (as Poly2::u)
  double scratch[(kSearchScratchBytes + 7) / 8];         // the batch of queries; the search's frame
};

// P <- P clipped by the line (n, d) with flag j from the outside corner p (s: the known-inside neighbour of p on a searched real
// edge, else -1).  nc is updated (0: nothing of P is left).  Returns 0, or 1 when the loop would outgrow 32 corners.
__device__ __forceinline__ int apply_clip_2d_par(Poly2P& S, int& nc, int p, int s, double nx, double ny, double nz, double d, int j,
                                                 double pnx, double pny, double pnz) {
  const int lane = lane_id();
  VD_WORK(extra_cnt_add(0, (unsigned)nc); extra_cnt_add(1, 2u);)
  // this lane's corner and edge
  double x = 0, y = 0, z = 0, ex = 0, ey = 0, ez = 0, e_d = 0;
  int fl = 0, nn = 0, stt = 0;
  bool out = false;
  if (lane < nc) {
    x = S.cx[lane]; y = S.cy[lane]; z = S.cz[lane];
    ex = S.enx[lane]; ey = S.eny[lane]; ez = S.enz[lane]; e_d = S.ed[lane];
    fl = S.eflag[lane]; nn = S.cnn[lane]; stt = S.cstate[lane];
    out = (nx * x + ny * y + nz * z - d > 0.0) && stt != ST_IN;
  }
  const unsigned full = nc >= 32 ? 0xffffffffu : ((1u << nc) - 1u);
  const unsigned m = (__ballot_sync(kFull, out) | (1u << p)) & full;
  // the outside run around p (P:L391's R_p for a loop): bit k of rot = corner (p + k) mod nc
  const unsigned rot = p == 0 ? m : (((m >> p) | (m << (nc - p))) & full);
  if (rot == full) { nc = 0; return 0; }
  const int fwd = __ffs((int)~rot) - 1;                 // corners p, p+1, ... beyond the line
  const unsigned zeros = ~rot & full;
  const int bwd = nc - 1 - (31 - __clz((int)zeros));    // corners p-1, p-2, ... beyond the line
  const int len = fwd + bwd;
  const int k = nc - len;                               // survivors
  if (k + 2 > kLanes) return 1;
  int r0 = p - bwd; if (r0 < 0) r0 += nc;
  int r1 = p + fwd - 1; if (r1 >= nc) r1 -= nc;
  const int pv = r0 == 0 ? nc - 1 : r0 - 1, nxt = r1 + 1 == nc ? 0 : r1 + 1;
  int idx = lane - nxt; if (idx < 0) idx += nc;         // position among the survivors nxt .. pv
  const bool survive = lane < nc && idx < k;
  // the two new corners, by the lanes that own the cut edges: X = edge(pv) ∩ B_ij, E = B_ij ∩ edge(r1)
  double qx = 0, qy = 0, qz = 0;
  if (lane == pv) {
    if (!solve3(ex, ey, ez, e_d, nx, ny, nz, d, pnx, pny, pnz, 0.0, qx, qy, qz))
      lerp_to_plane(S.cx[r0], S.cy[r0], S.cz[r0], x, y, z, nx, ny, nz, d, qx, qy, qz);
  } else if (lane == r1) {
    if (!solve3(nx, ny, nz, d, ex, ey, ez, e_d, pnx, pny, pnz, 0.0, qx, qy, qz))
      lerp_to_plane(x, y, z, S.cx[nxt], S.cy[nxt], S.cz[nxt], nx, ny, nz, d, qx, qy, qz);
  }
  __syncwarp();   // every lane holds what it needs: the slots may be rewritten
  if (survive) {
    S.cx[idx] = x; S.cy[idx] = y; S.cz[idx] = z;
    S.enx[idx] = ex; S.eny[idx] = ey; S.enz[idx] = ez; S.ed[idx] = e_d;
    S.eflag[idx] = fl; S.cnn[idx] = nn; S.cstate[idx] = (unsigned char)stt;
  }
  if (lane == pv) {          // X starts the new edge, which takes flag j
    S.cx[k] = qx; S.cy[k] = qy; S.cz[k] = qz;
    S.enx[k] = nx; S.eny[k] = ny; S.enz[k] = nz; S.ed[k] = d;
    S.eflag[k] = j; S.cnn[k] = -1;
    S.cstate[k] = (s == pv && p == r0) ? ST_IN : ST_UNKNOWN;   // on the searched real edge
  } else if (lane == r1) {   // E: the rest of edge r1 keeps its plane and flag
    S.cx[k + 1] = qx; S.cy[k + 1] = qy; S.cz[k + 1] = qz;
    S.enx[k + 1] = ex; S.eny[k + 1] = ey; S.enz[k + 1] = ez; S.ed[k + 1] = e_d;
    S.eflag[k + 1] = fl; S.cnn[k + 1] = -1;
    S.cstate[k + 1] = (s == nxt && p == r1) ? ST_IN : ST_UNKNOWN;
  }
  __syncwarp();
  nc = k + 2;
  return 0;
}

// One (triangle, site) pair on the lane-per-corner structure: Alg. 3 / Alg. 1 as in clip_pair_2d below, step for step.
// Returns 0 = done, 1 = the polygon outgrew 32 corners (the caller defers the pair to the large tier).
template <bool HV, bool BOX>
__device__ int clip_pair_2d_par(Poly2P& S, const GridIndex& g, const ClipArgs& A, int64_t pairIdx, StRef st, LocalCnt& lc) {
  const int lane = lane_id();
  const Pair pr = load_pair(A, pairIdx);
  const int a = pr.a, i = pr.i;
  const double six = __ldg(&A.sites[(int64_t)i * 3 + 0]), siy = __ldg(&A.sites[(int64_t)i * 3 + 1]),
               siz = __ldg(&A.sites[(int64_t)i * 3 + 2]);
  double ox, oy, oz, pnx, pny, pnz;
  int nc;
  if constexpr (BOX) {
    ox = __ldg(&A.verts[0]); oy = __ldg(&A.verts[1]); oz = __ldg(&A.verts[2]);
    const double e0 = __ldg(&A.verts[9]) - ox, e1 = __ldg(&A.verts[10]) - oy;
    pnx = 0.0; pny = 0.0; pnz = 1.0;
    if (lane < 4) {
      const int k = lane, vid = k ^ (k >> 1);
      S.cx[k] = (vid & 1) ? e0 : 0.0; S.cy[k] = (vid & 2) ? e1 : 0.0; S.cz[k] = 0.0;
      S.enx[k] = k == 1 ? 1.0 : (k == 3 ? -1.0 : 0.0);
      S.eny[k] = k == 2 ? 1.0 : (k == 0 ? -1.0 : 0.0);
      S.enz[k] = 0.0;
      S.ed[k] = k == 1 ? e0 : (k == 2 ? e1 : 0.0);
      S.eflag[k] = ~A.m;
      const int nn = __ldg(&A.vnn[vid]);
      S.cnn[k] = nn;
      S.cstate[k] = (nn == i) ? ST_IN : ST_OUT;
    }
    nc = 4;
  } else {
    int tv[3];
    double tx[3], ty[3], tz[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      tv[k] = __ldg(&A.simp[(int64_t)a * 3 + k]);
      tx[k] = __ldg(&A.verts[(int64_t)tv[k] * 3 + 0]);
      ty[k] = __ldg(&A.verts[(int64_t)tv[k] * 3 + 1]);
      tz[k] = __ldg(&A.verts[(int64_t)tv[k] * 3 + 2]);
    }
    ox = tx[0]; oy = ty[0]; oz = tz[0];
    {
      const double ax = tx[1] - ox, ay = ty[1] - oy, az = tz[1] - oz, bx = tx[2] - ox, by = ty[2] - oy, bz = tz[2] - oz;
      pnx = ay * bz - az * by; pny = az * bx - ax * bz; pnz = ax * by - ay * bx;
      const double inv = 1.0 / sqrt(pnx * pnx + pny * pny + pnz * pnz);
      pnx *= inv; pny *= inv; pnz *= inv;
    }
    if (lane < 3) {
      const int k = lane, k1 = (k + 1) % 3, k2 = (k + 2) % 3;
      S.cx[k] = tx[k] - ox; S.cy[k] = ty[k] - oy; S.cz[k] = tz[k] - oz;
      const double ex = tx[k1] - tx[k], ey = ty[k1] - ty[k], ez = tz[k1] - tz[k];
      double nx = ey * pnz - ez * pny, ny = ez * pnx - ex * pnz, nz = ex * pny - ey * pnx;   // e x n
      const double side = nx * (tx[k2] - tx[k]) + ny * (ty[k2] - ty[k]) + nz * (tz[k2] - tz[k]);
      if (side > 0) { nx = -nx; ny = -ny; nz = -nz; }
      S.enx[k] = nx; S.eny[k] = ny; S.enz[k] = nz;
      S.ed[k] = nx * (tx[k] - ox) + ny * (ty[k] - oy) + nz * (tz[k] - oz);
      S.eflag[k] = ~__ldg(&A.adj[(int64_t)a * 3 + k2]);
      const int nn = __ldg(&A.vnn[tv[k]]);
      S.cnn[k] = nn;
      S.cstate[k] = (nn == i) ? ST_IN : ST_OUT;
    }
    nc = 3;
  }
  const double vix = six - ox, viy = siy - oy, viz = siz - oz;
  const double wx = pr.wx - ox, wy = pr.wy - oy, wz = pr.wz - oz;
  if (lane == 0) {
    S.u[0] = ox; S.u[1] = oy; S.u[2] = oz; S.u[3] = six; S.u[4] = siy; S.u[5] = siz;
    S.u[6] = vix; S.u[7] = viy; S.u[8] = viz; S.u[9] = wx; S.u[10] = wy; S.u[11] = wz; S.u[12] = 0.0; S.u[13] = 0.0;
  }
  __syncwarp();
  bool failed = false;
  // ---- clips that need no search: B_iu, then B_iw of the two edges adjacent to the discovering edge
  if (A.firstClip && pr.u >= 0 && pr.u != i) {
    const Pair* pp = &A.pairs[pairIdx];
    const int w0 = __ldcg(&pp->w[0]), w1 = __ldcg(&pp->w[1]);
    bool complete = true;
    for (int t = 0; t < 3 && nc > 0; ++t) {
      const int j = t == 0 ? pr.u : (t == 1 ? w0 : w1);
      if (j < 0) continue;
      if (j == i) { complete = false; continue; }
      const double wjx = __ldg(&A.sites[(int64_t)j * 3 + 0]) - ox, wjy = __ldg(&A.sites[(int64_t)j * 3 + 1]) - oy,
                   wjz = __ldg(&A.sites[(int64_t)j * 3 + 2]) - oz;
      const double nx = wjx - vix, ny = wjy - viy, nz = wjz - viz;
      const double d = 0.5 * (nx * (vix + wjx) + ny * (viy + wjy) + nz * (viz + wjz));
      const double tol = 1e-9 * (nx * nx + ny * ny + nz * nz);
      double far = 0.0;
      int p = 0x7fffffff;
      bool own = false;
      if (lane < nc) {
        const double sd = nx * S.cx[lane] + ny * S.cy[lane] + nz * S.cz[lane] - d;
        if (sd > tol && S.cstate[lane] != ST_IN) { far = -sd; p = lane; }
        own = S.eflag[lane] == j;
      }
      warp_argmin(far, p);   // the corner farthest beyond the line starts the outside run
      if (p == 0x7fffffff || __any_sync(kFull, own)) { complete = false; continue; }   // the line does not cut P
      VD_WORK(lc.clips += 1; lc.pre_clips += 1;)
      if (apply_clip_2d_par(S, nc, p, -1, nx, ny, nz, d, j, pnx, pny, pnz)) return 1;
    }
    if (complete && nc > 0) {   // P's edge on B_iu is the discovering edge itself: its two end points are in Omega_i
      const unsigned hit = __ballot_sync(kFull, lane < nc && S.eflag[lane] == pr.u);
      const int prev = lane == 0 ? nc - 1 : lane - 1;
      if (lane < nc && (((hit >> lane) | (hit >> prev)) & 1u)) S.cstate[lane] = ST_IN;
      __syncwarp();
    }
  }
  QBatch& Q = *reinterpret_cast<QBatch*>(S.scratch);
  for (int guard = 0; guard < 4 * kLanes && nc > 0; ++guard) {
    // ---- point-in-cell tests of the unclassified corners (section IV-A), up to kQB per batched pass
    for (;;) {
      const bool unk = lane < nc && S.cstate[lane] == ST_UNKNOWN;
      const unsigned um = __ballot_sync(kFull, unk);
      if (!um) break;
      const int slot = __popc(um & ((1u << lane) - 1u));
      const int nq = min(kQB, __popc(um));
      if (unk && slot < kQB) {
        const double qx = S.cx[lane] + ox, qy = S.cy[lane] + oy, qz = S.cz[lane] + oz;
        const double dx = qx - six, dy = qy - siy, dz = qz - siz;
        Q.item[slot] = lane;
        Q.qx[slot] = qx; Q.qy[slot] = qy; Q.qz[slot] = qz;
        Q.best[slot] = dx * dx + dy * dy + dz * dz;
        Q.bestId[slot] = i;
      }
      __syncwarp();
      batch_nearest<HV>(g, Q, nq, st);
      if (lane < nq) {
        const int c = Q.item[lane], id = Q.bestId[lane];
        const double dx = Q.qx[lane] - six, dy = Q.qy[lane] - siy, dz = Q.qz[lane] - siz;
        const double di2 = dx * dx + dy * dy + dz * dz, best = Q.best[lane];
        // closed cell: a tie up to rounding is inside; a near tie is when the other site owns an edge of P (U6, U17)
        bool inside = id == i || best >= di2 * (1.0 - 1e-13);
        if (!inside && best >= di2 * (1.0 - 1e-9))
          for (int f = 0; f < nc && !inside; ++f) inside = S.eflag[f] == id;
        S.cstate[c] = inside ? ST_IN : ST_OUT;
        S.cnn[c] = id;
      }
      __syncwarp();
    }
    // ---- an outside corner p, preferring one with a neighbour p_s in Omega_i (real edge, Alg. 1 line 3)
    const bool out = lane < nc && S.cstate[lane] == ST_OUT;
    const unsigned om = __ballot_sync(kFull, out);
    if (!om) break;
    int sn = -1;
    if (out && A.realEdges) {
      const int pv = lane == 0 ? nc - 1 : lane - 1, nx2 = lane + 1 == nc ? 0 : lane + 1;
      if (S.cstate[pv] == ST_IN) sn = pv;
      else if (S.cstate[nx2] == ST_IN) sn = nx2;
    }
    const unsigned mr = __ballot_sync(kFull, sn >= 0);
    const int p = mr ? __ffs((int)mr) - 1 : __ffs((int)om) - 1;
    const int s = mr ? shfl(sn, p) : -1;
    double psx = wx, psy = wy, psz = wz;
    if (s >= 0) { psx = S.cx[s]; psy = S.cy[s]; psz = S.cz[s]; }
    double nx, ny, nz, d;
    const int j = find_bisector<HV>(A, g, i, S.cnn[p], S.u, psx, psy, psz, S.cx[p], S.cy[p], S.cz[p], S.eflag, nc,
                                    nx, ny, nz, d, st, lc, S.scratch);
    if (j < 0) { failed = true; atomicOr(&A.ctl->err, ERR_NOCONVERGE); break; }
    if (__any_sync(kFull, lane < nc && S.eflag[lane] == j)) {   // B_ij already bounds P: p lies on it up to rounding
      if (lane == 0) S.cstate[p] = ST_IN;
      __syncwarp();
      continue;
    }
    VD_WORK(lc.clips += 1;)
    if (apply_clip_2d_par(S, nc, p, s, nx, ny, nz, d, j, pnx, pny, pnz)) return 1;
  }
  // ---- finish
  Piece pc;
  pc.site = i; pc.simplex = a; pc.nverts = 0; pc.nnbr = 0; pc.vbase = 0; pc.nbase = 0;
  pc.measure = 0; pc.mx = pc.my = pc.mz = 0;
  lc.pairs += 1;
  if (failed || nc < 3) {
    if (lane == 0) A.pieces[pairIdx] = pc;
    return 0;
  }
  // area and first moment: fan from corner 0, one lane per fan triangle (0, t, t+1), signed along the triangle's unit normal
  double area = 0, mx = 0, my = 0, mz = 0;
  if (lane >= 1 && lane + 1 < nc) {
    const double x0 = S.cx[0], y0 = S.cy[0], z0 = S.cz[0];
    const double ux = S.cx[lane] - x0, uy = S.cy[lane] - y0, uz = S.cz[lane] - z0;
    const double vx = S.cx[lane + 1] - x0, vy = S.cy[lane + 1] - y0, vz = S.cz[lane + 1] - z0;
    area = 0.5 * ((uy * vz - uz * vy) * pnx + (uz * vx - ux * vz) * pny + (ux * vy - uy * vx) * pnz);
    mx = area * (x0 + (ux + vx) * (1.0 / 3.0));
    my = area * (y0 + (uy + vy) * (1.0 / 3.0));
    mz = area * (z0 + (uz + vz) * (1.0 / 3.0));
  }
  area = warp_sum(area); mx = warp_sum(mx); my = warp_sum(my); mz = warp_sum(mz);
  VD_WORK(extra_cnt_add(2, (unsigned)(nc - 2));)
  if (area < 0) { area = -area; mx = -mx; my = -my; mz = -mz; }
  if (!(area > 0)) {
    if (lane == 0) A.pieces[pairIdx] = pc;
    return 0;
  }
  const bool pos = lane < nc && S.eflag[lane] >= 0;
  const unsigned posm = __ballot_sync(kFull, pos);
  const int nnbr = __popc(posm);
  unsigned long long nb0 = 0, vb0 = 0;
  if (lane == 0) {
    nb0 = atomicAdd(&A.ctl->nbrTail, (unsigned long long)nnbr);
    vb0 = atomicAdd(&A.ctl->vertTail, (unsigned long long)nc);
  }
  nb0 = shfl(nb0, 0);
  vb0 = shfl(vb0, 0);
  if ((int64_t)(nb0 + nnbr) > A.nbrCap || (int64_t)(vb0 + nc) > A.vertCap) {
    if (lane == 0) {
      atomicOr(&A.ctl->err, (int64_t)(vb0 + nc) > A.vertCap ? ERR_VERT_CAP : ERR_NBR_CAP);
      A.pieces[pairIdx] = pc;
    }
    return 0;
  }
  // corners with their two edge flags, ascending (for the ranking below); neighbours and propagation: one lane per edge
  if (lane < nc) {
    const int prev = lane == 0 ? nc - 1 : lane - 1, next = lane + 1 == nc ? 0 : lane + 1;
    const int fp = S.eflag[prev], fc = S.eflag[lane], fn = S.eflag[next];
    S.k0[lane] = fp < fc ? fp : fc;
    S.k1[lane] = fp < fc ? fc : fp;
    if (pos) {
      A.poolNbr[nb0 + __popc(posm & ((1u << lane) - 1u))] = fc;
      // witness: the edge midpoint lies in T_a ∩ Omega_i ∩ Omega_j; with the tuple (u, f) of P:L211: this cell, and the
      // positive flags of the two edges adjacent to this one
      push_pair(A, a, fc, 0.5 * (S.cx[lane] + S.cx[next]) + ox, 0.5 * (S.cy[lane] + S.cy[next]) + oy,
                0.5 * (S.cz[lane] + S.cz[next]) + oz, i, fp >= 0 ? fp : -1, fn >= 0 ? fn : -1);
    }
  }
  __syncwarp();
  if (lane < nc) {
    const int q0 = S.k0[lane], q1 = S.k1[lane];
    int rank = 0;
    for (int o = 0; o < nc; ++o) {
      const int o0 = S.k0[o], o1 = S.k1[o];
      rank += (o0 < q0 || (o0 == q0 && (o1 < q1 || (o1 == q1 && o < lane)))) ? 1 : 0;
    }
    const int64_t v = (int64_t)vb0 + rank;
    A.poolXYZ[v * 3 + 0] = S.cx[lane] + ox; A.poolXYZ[v * 3 + 1] = S.cy[lane] + oy; A.poolXYZ[v * 3 + 2] = S.cz[lane] + oz;
    A.poolFlags[v * 2 + 0] = q0; A.poolFlags[v * 2 + 1] = q1;
  }
  if (lane == 0) {
    pc.nverts = nc; pc.nnbr = nnbr; pc.vbase = (int64_t)vb0; pc.nbase = (int64_t)nb0;
    pc.measure = area;
    pc.mx = mx + area * ox; pc.my = my + area * oy; pc.mz = mz + area * oz;
    A.pieces[pairIdx] = pc;
    atomicAdd(&A.sitePieces[i], 1);
    atomicAdd(&A.siteNbrRaw[i], nnbr);
  }
  lc.pieces += 1;
  __syncwarp();
  return 0;
}

template <int K, bool HV, bool BOX>
__device__ int clip_pair_2d(Poly2<K>& S, const GridIndex& g, const ClipArgs& A, int64_t pairIdx, StRef st, LocalCnt& lc) {
  const int lane = lane_id();
  const Pair pr = load_pair(A, pairIdx);
  const int a = pr.a, i = pr.i;
  const double six = __ldg(&A.sites[(int64_t)i * 3 + 0]), siy = __ldg(&A.sites[(int64_t)i * 3 + 1]),
               siz = __ldg(&A.sites[(int64_t)i * 3 + 2]);
  double ox, oy, oz, pnx, pny, pnz;
  if constexpr (BOX) {
    // simple domain (section V-B): P <- the rectangle; verts holds its 4 corners (bits x, y), the loop
    // runs 0 -> 1 -> 3 -> 2, edge k from corner k to k+1: bottom, right, top, left
    ox = __ldg(&A.verts[0]); oy = __ldg(&A.verts[1]); oz = __ldg(&A.verts[2]);
    const double e0 = __ldg(&A.verts[9]) - ox, e1 = __ldg(&A.verts[10]) - oy;
    pnx = 0.0; pny = 0.0; pnz = 1.0;
    if (lane < 4) {
      const int k = lane, vid = k ^ (k >> 1);
      S.cx[k] = (vid & 1) ? e0 : 0.0; S.cy[k] = (vid & 2) ? e1 : 0.0; S.cz[k] = 0.0;
      S.enx[k] = k == 1 ? 1.0 : (k == 3 ? -1.0 : 0.0);
      S.eny[k] = k == 2 ? 1.0 : (k == 0 ? -1.0 : 0.0);
      S.enz[k] = 0.0;
      S.ed[k] = k == 1 ? e0 : (k == 2 ? e1 : 0.0);
      S.eflag[k] = ~A.m;
      const int nn = __ldg(&A.vnn[vid]);
      S.cnn[k] = nn;
      S.cstate[k] = (nn == i) ? ST_IN : ST_OUT;
    }
    if (lane == 0) S.nc = 4;
  } else {
    int tv[3];
    double tx[3], ty[3], tz[3];
  #pragma unroll
    for (int k = 0; k < 3; ++k) {
      tv[k] = __ldg(&A.simp[(int64_t)a * 3 + k]);
      tx[k] = __ldg(&A.verts[(int64_t)tv[k] * 3 + 0]);
      ty[k] = __ldg(&A.verts[(int64_t)tv[k] * 3 + 1]);
      tz[k] = __ldg(&A.verts[(int64_t)tv[k] * 3 + 2]);
    }
    ox = tx[0]; oy = ty[0]; oz = tz[0];
    // triangle plane (local): unit normal, offset 0 (corner 0 is the origin)
    {
      const double ax = tx[1] - ox, ay = ty[1] - oy, az = tz[1] - oz, bx = tx[2] - ox, by = ty[2] - oy, bz = tz[2] - oz;
      pnx = ay * bz - az * by; pny = az * bx - ax * bz; pnz = ax * by - ay * bx;
      const double inv = 1.0 / sqrt(pnx * pnx + pny * pny + pnz * pnz);
      pnx *= inv; pny *= inv; pnz *= inv;
    }
    // ---- P <- T: corner k = vertex k, edge k = (k -> k+1) lies opposite vertex k+2
    if (lane < 3) {
      const int k = lane, k1 = (k + 1) % 3, k2 = (k + 2) % 3;
      S.cx[k] = tx[k] - ox; S.cy[k] = ty[k] - oy; S.cz[k] = tz[k] - oz;
      const double ex = tx[k1] - tx[k], ey = ty[k1] - ty[k], ez = tz[k1] - tz[k];
      double nx = ey * pnz - ez * pny, ny = ez * pnx - ex * pnz, nz = ex * pny - ey * pnx;   // e x n
      const double side = nx * (tx[k2] - tx[k]) + ny * (ty[k2] - ty[k]) + nz * (tz[k2] - tz[k]);
      if (side > 0) { nx = -nx; ny = -ny; nz = -nz; }
      S.enx[k] = nx; S.eny[k] = ny; S.enz[k] = nz;
      S.ed[k] = nx * (tx[k] - ox) + ny * (ty[k] - oy) + nz * (tz[k] - oz);
      S.eflag[k] = ~__ldg(&A.adj[(int64_t)a * 3 + k2]);
      const int nn = __ldg(&A.vnn[tv[k]]);
      S.cnn[k] = nn;
      S.cstate[k] = (nn == i) ? ST_IN : ST_OUT;
    }
    if (lane == 0) S.nc = 3;
  }
  const double vix = six - ox, viy = siy - oy, viz = siz - oz;
  const double wx = pr.wx - ox, wy = pr.wy - oy, wz = pr.wz - oz;
  if (lane == 0) {
    S.u[0] = ox; S.u[1] = oy; S.u[2] = oz; S.u[3] = six; S.u[4] = siy; S.u[5] = siz;
    S.u[6] = vix; S.u[7] = viy; S.u[8] = viz; S.u[9] = wx; S.u[10] = wy; S.u[11] = wz; S.u[12] = 0.0; S.u[13] = 0.0;
  }
  __syncwarp();
  bool failed = false;
#ifdef VD_TRACE
  {
    double b = 2e300; int bi = 0x7fffffff; QueryStats s2 = {0};
    nearest<HV>(g, pr.wx, pr.wy, pr.wz, b, bi, s2);
    const double dx = pr.wx - six, dy = pr.wy - siy, dz = pr.wz - siz;
    const double di = dx * dx + dy * dy + dz * dz;
    if (lane == 0 && bi != i && di - b > 1e-13) printf("BAD WITNESS pair(%d,%d) w=(%g,%g) nearest=%d di2=%g best=%g\n", a, i, pr.wx, pr.wy, bi, di, b);
  }
#endif
  // ---- clips that need no search (as for tets: vd_clip3d.cuh preclip_3d): a pair discovered through the
  // edge e of P_{a,u} on B_ui starts with B_iu, then B_iw for the (at most two) edges of P_{a,u} adjacent to e with a
  // positive flag w.  When all of them cut, P's edge on B_iu is e itself, and its two end points are in Omega_i.
  if (A.firstClip && pr.u >= 0 && pr.u != i) {
    const Pair* pp = &A.pairs[pairIdx];
    const int w0 = __ldcg(&pp->w[0]), w1 = __ldcg(&pp->w[1]);
    bool complete = true;
    for (int t = 0; t < 3 && S.nc > 0; ++t) {
      const int j = t == 0 ? pr.u : (t == 1 ? w0 : w1);
      if (j < 0) continue;
      if (j == i) { complete = false; continue; }
      const double wjx = __ldg(&A.sites[(int64_t)j * 3 + 0]) - ox, wjy = __ldg(&A.sites[(int64_t)j * 3 + 1]) - oy,
                   wjz = __ldg(&A.sites[(int64_t)j * 3 + 2]) - oz;
      const double nx = wjx - vix, ny = wjy - viy, nz = wjz - viz;
      const double d = 0.5 * (nx * (vix + wjx) + ny * (viy + wjy) + nz * (viz + wjz));
      const double tol = 1e-9 * (nx * nx + ny * ny + nz * nz);
      const int nc = S.nc;
      double far = tol;
      int p = -1;
      bool owned = false;
      for (int c = 0; c < nc; ++c) {   // the corner farthest beyond the line starts the outside run
        const double sd = nx * S.cx[c] + ny * S.cy[c] + nz * S.cz[c] - d;
        if (sd > far && S.cstate[c] != ST_IN) { far = sd; p = c; }
        owned |= (S.eflag[c] == j);
      }
      if (p < 0 || owned) { complete = false; continue; }   // the line does not cut P
      VD_WORK(lc.clips += 1; lc.pre_clips += 1;)
      if (apply_clip_2d(S, p, -1, nx, ny, nz, d, j, pnx, pny, pnz)) return 1;
    }
    __syncwarp();
    if (complete && lane == 0) {
      const int nc = S.nc;
      for (int c = 0; c < nc; ++c)
        if (S.eflag[c] == pr.u) { S.cstate[c] = ST_IN; S.cstate[(c + 1) % nc] = ST_IN; }
    }
    __syncwarp();
  }
  for (int guard = 0; guard < 4 * K; ++guard) {
    const int nc = S.nc;
    // point-in-cell tests of unclassified corners (section IV-A)
    for (int c = 0; c < nc; ++c) {
      if (S.cstate[c] != ST_UNKNOWN) continue;
      const double qx = S.cx[c] + ox, qy = S.cy[c] + oy, qz = S.cz[c] + oz;
      const double dx = qx - six, dy = qy - siy, dz = qz - siz;
      const double di2 = dx * dx + dy * dy + dz * dz;
      double best = di2;
      int bestId = i;
      nearest<HV>(g, qx, qy, qz, best, bestId, st, true);
      // closed cell: a tie up to rounding is inside; a near tie is when the other site owns an edge of P (U6, U17)
      bool inside = bestId == i || best >= di2 * (1.0 - 1e-13);
      if (!inside && best >= di2 * (1.0 - 1e-9)) {
        bool own = false;
        for (int f = lane; f < nc; f += kLanes) own |= (S.eflag[f] == bestId);
        inside = __any_sync(kFull, own);   // flag rule (reading U6)
      }
      __syncwarp();
      if (lane == 0) { S.cstate[c] = inside ? ST_IN : ST_OUT; S.cnn[c] = bestId; }
#ifdef VD_TRACE
      if (lane == 0) printf("pair(%d,%d) classify c=%d q=(%g,%g) best=%g id=%d inside=%d\n", a, i, c, qx, qy, best, bestId, (int)inside);
#endif
      __syncwarp();
    }
    // select the outside corner p and, if possible, a neighbour p_s in Omega_i (real edge)
    int p = -1, s = -1;
    for (int c = 0; c < nc; ++c) {
      if (S.cstate[c] != ST_OUT) continue;
      if (p < 0) p = c;
      if (A.realEdges) {
        const int pv = (c + nc - 1) % nc, nx = (c + 1) % nc;
        if (S.cstate[pv] == ST_IN) { p = c; s = pv; break; }
        if (S.cstate[nx] == ST_IN) { p = c; s = nx; break; }
      }
    }
    if (p < 0) break;
    double psx = wx, psy = wy, psz = wz;
    if (s >= 0) { psx = S.cx[s]; psy = S.cy[s]; psz = S.cz[s]; }
    double nx, ny, nz, d;
    const int j = find_bisector<HV>(A, g, i, S.cnn[p], S.u, psx, psy, psz, S.cx[p], S.cy[p], S.cz[p], S.eflag, nc,
                                nx, ny, nz, d, st, lc, S.scratch);
    if (j < 0) { failed = true; atomicOr(&A.ctl->err, ERR_NOCONVERGE); break; }
    bool own = false;
    for (int c = 0; c < nc; ++c) own |= (S.eflag[c] == j);
    if (own) {
      __syncwarp();
      if (lane == 0) S.cstate[p] = ST_IN;
      __syncwarp();
      continue;
    }
#ifdef VD_TRACE
    if (lane == 0) printf("pair(%d,%d) clip p=%d s=%d j=%d nc=%d\n", a, i, p, s, j, nc);
#endif
    VD_WORK(lc.clips += 1;)
    __syncwarp();
    int rc = apply_clip_2d(S, p, s, nx, ny, nz, d, j, pnx, pny, pnz);
#ifdef VD_TRACE
    if (lane == 0) { printf("   loop:"); for (int c = 0; c < S.nc; ++c) printf(" (%.4f,%.4f|f%d|s%d)", S.cx[c]+ox, S.cy[c]+oy, S.eflag[c], (int)S.cstate[c]); printf("\n"); }
#endif
    if (rc) return 1;
    if (S.nc == 0) break;
  }
  // ---- finish
  const int nc = S.nc;
  Piece pc;
  pc.site = i; pc.simplex = a; pc.nverts = 0; pc.nnbr = 0; pc.vbase = 0; pc.nbase = 0;
  pc.measure = 0; pc.mx = pc.my = pc.mz = 0;
  lc.pairs += 1;
  if (failed || nc < 3) {
    if (lane == 0) A.pieces[pairIdx] = pc;
    return 0;
  }
  // area and first moment: fan from corner 0, signed along the triangle's unit normal
  double area = 0, mx = 0, my = 0, mz = 0;
  for (int c = 1; c + 1 < nc; ++c) {
    const double ux = S.cx[c] - S.cx[0], uy = S.cy[c] - S.cy[0], uz = S.cz[c] - S.cz[0];
    const double vx = S.cx[c + 1] - S.cx[0], vy = S.cy[c + 1] - S.cy[0], vz = S.cz[c + 1] - S.cz[0];
    const double ar = 0.5 * ((uy * vz - uz * vy) * pnx + (uz * vx - ux * vz) * pny + (ux * vy - uy * vx) * pnz);
    area += ar;
    mx += ar * (S.cx[0] + (ux + vx) * (1.0 / 3.0));
    my += ar * (S.cy[0] + (uy + vy) * (1.0 / 3.0));
    mz += ar * (S.cz[0] + (uz + vz) * (1.0 / 3.0));
  }
  VD_WORK(extra_cnt_add(2, (unsigned)(nc - 2));)
  if (area < 0) { area = -area; mx = -mx; my = -my; mz = -mz; }
  if (!(area > 0)) {
    if (lane == 0) A.pieces[pairIdx] = pc;
    return 0;
  }
  int nnbr = 0;
  for (int c = 0; c < nc; ++c) nnbr += S.eflag[c] >= 0 ? 1 : 0;
  unsigned long long nb0 = 0, vb0 = 0;
  if (lane == 0) {
    nb0 = atomicAdd(&A.ctl->nbrTail, (unsigned long long)nnbr);
    vb0 = atomicAdd(&A.ctl->vertTail, (unsigned long long)nc);
  }
  nb0 = shfl(nb0, 0);
  vb0 = shfl(vb0, 0);
  if ((int64_t)(nb0 + nnbr) > A.nbrCap || (int64_t)(vb0 + nc) > A.vertCap) {
    if (lane == 0) {
      atomicOr(&A.ctl->err, (int64_t)(vb0 + nc) > A.vertCap ? ERR_VERT_CAP : ERR_NBR_CAP);
      A.pieces[pairIdx] = pc;
    }
    return 0;
  }
  if (lane == 0) {
    int k = 0;
    for (int c = 0; c < nc; ++c) {
      if (S.eflag[c] < 0) continue;
      A.poolNbr[nb0 + k++] = S.eflag[c];
      const int c1 = (c + 1) % nc;
      // witness: the edge midpoint lies in T_a ∩ Omega_i ∩ Omega_j
      // with the tuple (u, f) of P:L211: this cell, and the positive flags of the two edges adjacent to edge c
      const int fp = S.eflag[(c + nc - 1) % nc], fn = S.eflag[c1];
      push_pair(A, a, S.eflag[c], 0.5 * (S.cx[c] + S.cx[c1]) + ox, 0.5 * (S.cy[c] + S.cy[c1]) + oy,
                0.5 * (S.cz[c] + S.cz[c1]) + oz, i, fp >= 0 ? fp : -1, fn >= 0 ? fn : -1);
    }
  }
  // corners with their two edge flags, ascending; ranked lexicographically
  for (int c = lane; c < nc; c += kLanes) {
    int f0 = S.eflag[(c + nc - 1) % nc], f1 = S.eflag[c];
    if (f0 > f1) { const int t = f0; f0 = f1; f1 = t; }
    S.tflag[c] = f0; S.tnn[c] = f1;
  }
  __syncwarp();
  for (int c = lane; c < nc; c += kLanes) {
    const int k0 = S.tflag[c], k1 = S.tnn[c];
    int rank = 0;
    for (int o = 0; o < nc; ++o) {
      const int o0 = S.tflag[o], o1 = S.tnn[o];
      rank += (o0 < k0 || (o0 == k0 && (o1 < k1 || (o1 == k1 && o < c)))) ? 1 : 0;
    }
    const int64_t v = (int64_t)vb0 + rank;
    A.poolXYZ[v * 3 + 0] = S.cx[c] + ox; A.poolXYZ[v * 3 + 1] = S.cy[c] + oy; A.poolXYZ[v * 3 + 2] = S.cz[c] + oz;
    A.poolFlags[v * 2 + 0] = k0; A.poolFlags[v * 2 + 1] = k1;
  }
  if (lane == 0) {
    pc.nverts = nc; pc.nnbr = nnbr; pc.vbase = (int64_t)vb0; pc.nbase = (int64_t)nb0;
    pc.measure = area;
    pc.mx = mx + area * ox; pc.my = my + area * oy; pc.mz = mz + area * oz;
    A.pieces[pairIdx] = pc;
    atomicAdd(&A.sitePieces[i], 1);
    atomicAdd(&A.siteNbrRaw[i], nnbr);
  }
  lc.pieces += 1;
  __syncwarp();
  return 0;
}

}  // namespace vd
