// vd_clip3d.cuh -- S4 for tetrahedra: one warp computes P_{a,i} = T_a ∩ Omega_i by Alg. 3
// / Alg. 1 on the cell structure of section VI-C: an array of planes and an
// array of corners, each corner the intersection of three planes = a triangle of the dual mesh.
#pragma once
#include "vd_batch.cuh"
#include "vd_clip_args.cuh"

namespace vd {

// Member order matters to the phased schedule (vd_phase.cu), which parks polytopes in HBM between kernels: first
// what the point-in-cell tests read, then the rest of the polytope, scratch last (never copied).  Every array
// starts on a 16-byte boundary.
// A warp's private chunks of the corner pool and the face-flag pool (phased finish kernel).
struct WarpPool {
  unsigned long long vbase, nbase;
  int vleft, nleft, vchunk, nchunk;
};

template <int P, int C>
struct alignas(16) Poly3 {
  double u[14];                           // per-pair constants: origin o, site v_i (absolute, local), witness (local), [12] = the site's additive term (power diagrams), [13] spare
  int pflag[P];                           // flag of plane f
  double cx[C], cy[C], cz[C];             // corner coordinates (local)
  unsigned char cstate[C];
  int cnn[C];                             // nearest site of an outside corner            <- end of what the tests touch
  double pnx[P], pny[P], pnz[P], pd[P];   // plane f: n.x <= d, coordinates local to the tet's corner 0
  unsigned short cp[C][3];                // the corner's three planes, cyclically ordered
  unsigned short cadj[C][3];              // corner across the polytope edge (cp[t], cp[t+1])
  int key[C + 16][3];                     // scratch from here on (sized for the query batch: static_assert in classify_unknown_3d): flag triple of a corner (output order); rim points during a clip
  unsigned short remap[C];                // index of a surviving corner after the clip
  unsigned short pa[P], pb[P];            // new corner whose rim edge starts / ends at a plane
  unsigned short be[P][4];                // rim edges of R_p: (a, b, inside neighbour, flags)
  unsigned char cmark[C];
};

// What the point-in-cell tests of a piece touch: the leading members of Poly3, at the same offsets, and room for the
// batch state.  k_ph_verify holds this (2.8 KB per warp) instead of the whole polytope (5.2 KB): the shared memory
// it does not take is L1 for the site records the tests stream through.
template <int P, int C>
struct alignas(16) PolyTest3 {
  double u[14];
  int pflag[P];
  double cx[C], cy[C], cz[C];
  unsigned char cstate[C];
  int cnn[C];
  int key[(sizeof(QBatch) + 40 + 11) / 12 + 1][3];   // scratch: the batch of queries (k_ph_verify searches nothing: no frame)
};

// returns false when the three planes are (numerically) parallel to a common line
__device__ __forceinline__ bool solve3(double ax, double ay, double az, double ad, double bx, double by, double bz, double bd,
                                       double cx, double cy, double cz, double cd, double& x, double& y, double& z) {
  // Cramer: x = (ad (b x c) + bd (c x a) + cd (a x b)) / det[a, b, c]
  const double bcx = by * cz - bz * cy, bcy = bz * cx - bx * cz, bcz = bx * cy - by * cx;
  const double cax = cy * az - cz * ay, cay = cz * ax - cx * az, caz = cx * ay - cy * ax;
  const double abx = ay * bz - az * by, aby = az * bx - ax * bz, abz = ax * by - ay * bx;
  const double det = ax * bcx + ay * bcy + az * bcz;
  const double inv = 1.0 / det;
  x = (ad * bcx + bd * cax + cd * abx) * inv;
  y = (ad * bcy + bd * cay + cd * aby) * inv;
  z = (ad * bcz + bd * caz + cd * abz) * inv;
  const double na = ax * ax + ay * ay + az * az, nb = bx * bx + by * by + bz * bz, nc = cx * cx + cy * cy + cz * cz;
  return det * det > 1e-24 * na * nb * nc;
}

// P <- P clipped by the half-space n.x <= d with flag j (Alg. 3 line 4), steps of P:L389: (1) the
// corners outside the plane, restricted to the connected component R_p that contains the known-outside
// corner p; (2) the rim of R_p; (3) R_p removed, one new corner per rim edge.
// np, nc are updated.  Returns 0 ok, 1 capacity, 2 the rim is not a simple loop.
template <int P, int C>
__device__ int apply_clip_3d(Poly3<P, C>& S, int& np, int& nc, int p, int s, double nx, double ny, double nz, double d, int j) {
  const int lane = lane_id();
  const int N = np;   // index of the new plane
  if (nc <= kLanes) {
    // ---- Pieces of at most 32 corners (every tet piece; most whole cells): one corner per lane, the corner sets
    // are bit masks in registers, and when the clip adds at least as many corners as it removes (always, unless
    // R_p swallows a whole face) the new corners take the slots of the removed ones: nothing else moves.
    const int c = lane;
    const bool live = c < nc;
    const unsigned lt = (1u << lane) - 1u;
    int a0 = 0, a1 = 0, a2 = 0;
    bool cand = false;
    if (live) {
      const double sd = nx * S.cx[c] + ny * S.cy[c] + nz * S.cz[c] - d;
      cand = (c == p) || (sd > 0.0 && S.cstate[c] != ST_IN);
      a0 = S.cadj[c][0]; a1 = S.cadj[c][1]; a2 = S.cadj[c][2];
    }
    // (1) R_p: flood from p over polytope edges among the candidates
    const unsigned nbm = live ? ((1u << a0) | (1u << a1) | (1u << a2)) : 0u;
    unsigned R = 1u << p;
    for (;;) {
      const unsigned grow = __ballot_sync(kFull, cand && !((R >> c) & 1u) && (nbm & R) != 0u);
      if (!grow) break;
      R |= grow;
    }
    // (2) rim edges of the removed corners
    const bool rem = live && ((R >> c) & 1u);
    const bool r0 = rem && !((R >> a0) & 1u), r1 = rem && !((R >> a1) & 1u), r2 = rem && !((R >> a2) & 1u);
    const int cnt = (int)r0 + (int)r1 + (int)r2;
    const unsigned b0 = __ballot_sync(kFull, cnt & 1), b1 = __ballot_sync(kFull, cnt & 2);
    const int L = __popc(b0) + 2 * __popc(b1), k = __popc(R);
    if (L == 0) { nc = 0; np = N + 1; return 0; }   // nothing of P is left
    if (L > P || nc - k + L > C) return 1;
    if (L >= k) {
      VD_WORK(extra_cnt_add(0, (unsigned)nc); extra_cnt_add(1, (unsigned)L);)
      const int base = __popc(b0 & lt) + 2 * __popc(b1 & lt);
      if (lane == 0) { S.pnx[N] = nx; S.pny[N] = ny; S.pnz[N] = nz; S.pd[N] = d; S.pflag[N] = j; }
      if (rem) S.remap[__popc(R & lt)] = (unsigned short)c;   // slot list: the e-th new corner takes the e-th removed slot
      // which of the surviving neighbour's three slots points back at c (read before anybody rewrites them)
      int q0 = 0, q1 = 0, q2 = 0;
      if (r0) q0 = (S.cadj[a0][0] == c) ? 0 : ((S.cadj[a0][1] == c) ? 1 : 2);
      if (r1) q1 = (S.cadj[a1][0] == c) ? 0 : ((S.cadj[a1][1] == c) ? 1 : 2);
      if (r2) q2 = (S.cadj[a2][0] == c) ? 0 : ((S.cadj[a2][1] == c) ? 1 : 2);
      for (int f = lane; f <= N; f += kLanes) { S.pa[f] = 0xffff; S.pb[f] = 0xffff; }
      __syncwarp();
      if (rem) {
#pragma unroll
        for (int t = 0; t < 3; ++t) {
          const bool rt = t == 0 ? r0 : (t == 1 ? r1 : r2);
          if (!rt) continue;
          const int nb = t == 0 ? a0 : (t == 1 ? a1 : a2);
          const int q = t == 0 ? q0 : (t == 1 ? q1 : q2);
          const int e = base + (t == 0 ? 0 : (t == 1 ? (int)r0 : (int)r0 + (int)r1));
          const int slot = e < k ? (int)S.remap[e] : nc + (e - k);
          S.be[e][0] = S.cp[c][t]; S.be[e][1] = S.cp[c][(t + 1) % 3]; S.be[e][2] = (unsigned short)nb;
          S.be[e][3] = (unsigned short)(c | ((c == p && nb == s) ? 0x8000 : 0));
          S.cadj[nb][q] = (unsigned short)slot;   // the surviving neighbour now points at the new corner
        }
      }
      __syncwarp();
      // (2b) + (3) one lane per rim edge (a -> b): the new corner (a, b, N), its position, its neighbours along N
      bool bad = false;
      int t = 0, ea = 0, eb = 0, nb = 0, fl = 0;
      double x = 0, y = 0, z = 0;
      const int e = lane;
      if (e < L) {
        t = e < k ? (int)S.remap[e] : nc + (e - k);
        ea = S.be[e][0]; eb = S.be[e][1]; nb = S.be[e][2]; fl = S.be[e][3];
        const bool ok = solve3(S.pnx[ea], S.pny[ea], S.pnz[ea], S.pd[ea], S.pnx[eb], S.pny[eb], S.pnz[eb], S.pd[eb], nx, ny, nz, d, x, y, z);
        if (!ok) {   // ill-conditioned planes: where the polytope edge (removed corner, neighbour) meets the new plane
          const int rc = fl & 0x7fff;
          const double sc = nx * S.cx[rc] + ny * S.cy[rc] + nz * S.cz[rc] - d;
          const double sn = nx * S.cx[nb] + ny * S.cy[nb] + nz * S.cz[nb] - d;
          double tt = (sc - sn) > 0.0 ? sc / (sc - sn) : 0.0;
          tt = fmin(fmax(tt, 0.0), 1.0);
          x = S.cx[rc] + tt * (S.cx[nb] - S.cx[rc]);
          y = S.cy[rc] + tt * (S.cy[nb] - S.cy[rc]);
          z = S.cz[rc] + tt * (S.cz[nb] - S.cz[rc]);
        }
        if (S.pa[ea] != 0xffff || S.pb[eb] != 0xffff) bad = true;   // (racy duplicates are caught below)
        S.pa[ea] = (unsigned short)t;
        S.pb[eb] = (unsigned short)t;
      }
      __syncwarp();   // every read of a removed corner is done: its slot may be rewritten
      if (e < L) {
        S.cp[t][0] = (unsigned short)ea; S.cp[t][1] = (unsigned short)eb; S.cp[t][2] = (unsigned short)N;
        S.cadj[t][0] = (unsigned short)nb;
        const int nxt = S.pa[eb];   // edge (b -> N) is shared with the corner whose rim edge starts at b
        const int prv = S.pb[ea];   // edge (N -> a) with the corner whose rim edge ends at a
        if (nxt == 0xffff || prv == 0xffff || S.pa[ea] != t || S.pb[eb] != t) bad = true;
        S.cadj[t][1] = (unsigned short)nxt;
        S.cadj[t][2] = (unsigned short)prv;
        S.cx[t] = x; S.cy[t] = y; S.cz[t] = z;
        S.cnn[t] = -1;
        S.cstate[t] = (fl & 0x8000) ? ST_IN : ST_UNKNOWN;   // on the searched real edge p_s p: in Omega_i
      }
      __syncwarp();
      nc = nc - k + L;
      np = N + 1;
      return __any_sync(kFull, bad) ? 2 : 0;
    }
  }
  // ---- general form: any number of corners, survivors compacted to the front
  // (1) candidates: strictly outside the plane and not known to be in Omega_i; p itself always
  for (int c = lane; c < nc; c += kLanes) {
    const double sd = nx * S.cx[c] + ny * S.cy[c] + nz * S.cz[c] - d;
    const bool cand = (c == p) || (sd > 0.0 && S.cstate[c] != ST_IN);
    S.cmark[c] = (c == p) ? 2 : (cand ? 1 : 0);   // 2 = in R_p, 1 = candidate, 0 = stays
  }
  if (lane == 0) {
    S.pnx[N] = nx; S.pny[N] = ny; S.pnz[N] = nz; S.pd[N] = d; S.pflag[N] = j;
  }
  __syncwarp();
  for (int it = 0; it < C; ++it) {   // flood over polytope edges
    bool grew = false;
    for (int c = lane; c < nc; c += kLanes) {
      if (S.cmark[c] == 1 && (S.cmark[S.cadj[c][0]] == 2 || S.cmark[S.cadj[c][1]] == 2 || S.cmark[S.cadj[c][2]] == 2)) {
        S.cmark[c] = 2;
        grew = true;
      }
    }
    __syncwarp();
    if (!__any_sync(kFull, grew)) break;
  }
  // (2) rim edges: edge (cp[t], cp[t+1]) of a removed corner whose neighbour across it stays
  int L = 0, nRemoved = 0;
  for (int c0 = 0; c0 < nc; c0 += kLanes) {
    const int c = c0 + lane;
    const bool rem = c < nc && S.cmark[c] == 2;
    // rim edge t of c: the neighbour across (cp[t], cp[t+1]) stays.  No arrays indexed at run time here: they
    // would live in local memory
    int nb0 = 0, nb1 = 0, nb2 = 0;
    bool r0 = false, r1 = false, r2 = false;
    if (rem) {
      nb0 = S.cadj[c][0]; nb1 = S.cadj[c][1]; nb2 = S.cadj[c][2];
      r0 = S.cmark[nb0] != 2; r1 = S.cmark[nb1] != 2; r2 = S.cmark[nb2] != 2;
    }
    const int cnt = (int)r0 + (int)r1 + (int)r2;
    const int incl = warp_incl_scan(cnt);
    const int base = L + incl - cnt;
    const int tot = shfl(incl, kLanes - 1);
    if (L + tot > P) return 1;
    if (rem) {
#pragma unroll
      for (int t = 0; t < 3; ++t) {
        const bool rt = t == 0 ? r0 : (t == 1 ? r1 : r2);
        if (!rt) continue;
        const int nb = t == 0 ? nb0 : (t == 1 ? nb1 : nb2);
        const int e = base + (t == 0 ? 0 : (t == 1 ? (int)r0 : (int)r0 + (int)r1));
        S.be[e][0] = S.cp[c][t]; S.be[e][1] = S.cp[c][(t + 1) % 3]; S.be[e][2] = (unsigned short)nb;
        // the removed corner, and whether (c, nb) is the searched real edge p_s p
        S.be[e][3] = (unsigned short)(c | ((c == p && nb == s) ? 0x8000 : 0));
        // the surviving neighbour's slot that pointed at c will point at the new corner
#pragma unroll
        for (int q = 0; q < 3; ++q)
          if (S.cadj[nb][q] == c) S.cadj[nb][q] = (unsigned short)(0x8000 | e);
      }
    }
    L += tot;
    nRemoved += __popc(__ballot_sync(kFull, rem));
  }
  __syncwarp();
  const int nSurv = nc - nRemoved;
  if (L == 0) { nc = 0; np = N + 1; return 0; }   // nothing of P is left
  if (nSurv + L > C) return 1;
  VD_WORK(extra_cnt_add(0, (unsigned)nc); extra_cnt_add(1, (unsigned)L);)
  // (2b) where the new corners are: rim edge (a -> b) gives the corner (a, b, N), the solution of its three planes;
  // one lane per rim edge, while the removed corners are still in place for the fallback
  for (int e = lane; e < L; e += kLanes) {
    const int ea = S.be[e][0], eb = S.be[e][1];
    double x, y, z;
    const bool ok = solve3(S.pnx[ea], S.pny[ea], S.pnz[ea], S.pd[ea], S.pnx[eb], S.pny[eb], S.pnz[eb], S.pd[eb], nx, ny, nz, d, x, y, z);
    if (!ok) {
      // ill-conditioned planes (degenerate inputs, e.g. regular grids): where the polytope edge (c, neighbour)
      // meets the new plane, by interpolation
      const int c = S.be[e][3] & 0x7fff, nb = S.be[e][2];
      const double sc = nx * S.cx[c] + ny * S.cy[c] + nz * S.cz[c] - d;
      const double sn = nx * S.cx[nb] + ny * S.cy[nb] + nz * S.cz[nb] - d;
      double tt = (sc - sn) > 0.0 ? sc / (sc - sn) : 0.0;
      tt = fmin(fmax(tt, 0.0), 1.0);
      x = S.cx[c] + tt * (S.cx[nb] - S.cx[c]);
      y = S.cy[c] + tt * (S.cy[nb] - S.cy[c]);
      z = S.cz[c] + tt * (S.cz[nb] - S.cz[c]);
    }
    double* rim = reinterpret_cast<double*>(&S.key[0][0]) + 3 * e;
    rim[0] = x; rim[1] = y; rim[2] = z;
  }
  __syncwarp();
  // (3a) compact the surviving corners to the front
  int run = 0;
  for (int c0 = 0; c0 < nc; c0 += kLanes) {
    const int c = c0 + lane;
    const bool keep = c < nc && S.cmark[c] != 2;
    const unsigned m = __ballot_sync(kFull, keep);
    if (keep) S.remap[c] = (unsigned short)(run + __popc(m & ((1u << lane) - 1u)));
    run += __popc(m);
  }
  __syncwarp();
  for (int c0 = 0; c0 < nc; c0 += kLanes) {
    const int c = c0 + lane;
    const bool keep = c < nc && S.cmark[c] != 2;
    double x = 0, y = 0, z = 0;
    int nn = 0, st = 0;
    unsigned short cp0 = 0, cp1 = 0, cp2 = 0, a0 = 0, a1 = 0, a2 = 0;
    if (keep) {
      x = S.cx[c]; y = S.cy[c]; z = S.cz[c]; nn = S.cnn[c]; st = S.cstate[c];
      cp0 = S.cp[c][0]; cp1 = S.cp[c][1]; cp2 = S.cp[c][2];
      a0 = S.cadj[c][0]; a1 = S.cadj[c][1]; a2 = S.cadj[c][2];
      a0 = (a0 & 0x8000) ? (unsigned short)(nSurv + (a0 & 0x7fff)) : S.remap[a0];
      a1 = (a1 & 0x8000) ? (unsigned short)(nSurv + (a1 & 0x7fff)) : S.remap[a1];
      a2 = (a2 & 0x8000) ? (unsigned short)(nSurv + (a2 & 0x7fff)) : S.remap[a2];
    }
    __syncwarp();
    if (keep) {
      const int t = S.remap[c];
      S.cx[t] = x; S.cy[t] = y; S.cz[t] = z; S.cnn[t] = nn; S.cstate[t] = (unsigned char)st;
      S.cp[t][0] = cp0; S.cp[t][1] = cp1; S.cp[t][2] = cp2;
      S.cadj[t][0] = a0; S.cadj[t][1] = a1; S.cadj[t][2] = a2;
    }
    __syncwarp();
  }
  // (3b) new corners: rim edge (a -> b) becomes the corner (a, b, N)
  for (int f = lane; f <= N; f += kLanes) { S.pa[f] = 0xffff; S.pb[f] = 0xffff; }
  __syncwarp();
  bool bad = false;
  for (int e = lane; e < L; e += kLanes) {
    const int ea = S.be[e][0], eb = S.be[e][1];
    if (S.pa[ea] != 0xffff || S.pb[eb] != 0xffff) bad = true;   // (racy duplicates are caught below)
    S.pa[ea] = (unsigned short)(nSurv + e);
    S.pb[eb] = (unsigned short)(nSurv + e);
  }
  __syncwarp();
  for (int e = lane; e < L; e += kLanes) {
    const int t = nSurv + e;
    const int ea = S.be[e][0], eb = S.be[e][1];
    S.cp[t][0] = (unsigned short)ea; S.cp[t][1] = (unsigned short)eb; S.cp[t][2] = (unsigned short)N;
    S.cadj[t][0] = S.remap[S.be[e][2]];
    const int nxt = S.pa[eb];   // edge (b -> N) is shared with the corner whose rim edge starts at b
    const int prv = S.pb[ea];   // edge (N -> a) with the corner whose rim edge ends at a
    if (nxt == 0xffff || prv == 0xffff || S.pa[ea] != t || S.pb[eb] != t) bad = true;
    S.cadj[t][1] = (unsigned short)nxt;
    S.cadj[t][2] = (unsigned short)prv;
    const double* rim = reinterpret_cast<const double*>(&S.key[0][0]) + 3 * e;
    S.cx[t] = rim[0]; S.cy[t] = rim[1]; S.cz[t] = rim[2];
    S.cnn[t] = -1;
    // the new corner on the searched real edge p_s p is in Omega_i ∩ Omega_j
    S.cstate[t] = (S.be[e][3] & 0x8000) ? ST_IN : ST_UNKNOWN;
  }
  __syncwarp();
  nc = nSurv + L;
  np = N + 1;
  return __any_sync(kFull, bad) ? 2 : 0;
}

// Drop the planes that no corner lies on any more (box faces and early bisectors cut away by later ones): P's
// plane list is a capacity (P planes in the fast tier) and the flag rules loop over it.
template <int P, int C>
static __device__ __noinline__ void compact_planes_3d(Poly3<P, C>& S, int& np, int nc) {
  const int lane = lane_id();
  for (int f = lane; f < np; f += kLanes) S.pa[f] = 0;
  __syncwarp();
  for (int c = lane; c < nc; c += kLanes) { S.pa[S.cp[c][0]] = 1; S.pa[S.cp[c][1]] = 1; S.pa[S.cp[c][2]] = 1; }
  __syncwarp();
  int run = 0;
  for (int f0 = 0; f0 < np; f0 += kLanes) {
    const int f = f0 + lane;
    const bool live = f < np && S.pa[f] != 0;
    const unsigned m = __ballot_sync(kFull, live);
    const int t = run + __popc(m & ((1u << lane) - 1u));
    double a = 0, b = 0, c = 0, d = 0;
    int fl = 0;
    if (live) { a = S.pnx[f]; b = S.pny[f]; c = S.pnz[f]; d = S.pd[f]; fl = S.pflag[f]; }
    __syncwarp();   // targets t <= f lie in this chunk or in earlier ones, already read
    if (live) { S.pnx[t] = a; S.pny[t] = b; S.pnz[t] = c; S.pd[t] = d; S.pflag[t] = fl; S.pb[f] = (unsigned short)t; }
    run += __popc(m);
    __syncwarp();
  }
  for (int c = lane; c < nc; c += kLanes) {
    S.cp[c][0] = S.pb[S.cp[c][0]]; S.cp[c][1] = S.pb[S.cp[c][1]]; S.cp[c][2] = S.pb[S.cp[c][2]];
  }
  __syncwarp();
  np = run;
}

// Record the finished piece: measure and first moment (fan tetrahedra over every face, S6 input),
// corners with their flag triples in canonical order, face flags, and the propagation of P:L266-273.
template <int P, int C>
__device__ int finish_piece_3d(Poly3<P, C>& S, const ClipArgs& A, int64_t pairIdx, int a, int i, int np, int nc, double ox,
                               double oy, double oz, bool failed, LocalCnt& lc, WarpPool* wp = nullptr) {
  const int lane = lane_id();
  Piece pc;
  pc.site = i; pc.simplex = a; pc.nverts = 0; pc.nnbr = 0; pc.vbase = 0; pc.nbase = 0;
  pc.measure = 0; pc.mx = pc.my = pc.mz = 0;
  lc.pairs += 1;
  if (failed || nc < 4) {
#ifdef VD_TRACE
    if (lane == 0) printf("pair(%d,%d) dropped: failed=%d nc=%d np=%d\n", a, i, (int)failed, nc, np);
#endif
    if (lane == 0) A.pieces[pairIdx] = pc;
    return 0;
  }
  // one corner of every live plane (a plane is live iff some corner lies on it)
  for (int f = lane; f < np; f += kLanes) S.pa[f] = 0xffff;
  __syncwarp();
  for (int c = lane; c < nc; c += kLanes) {
    S.pa[S.cp[c][0]] = (unsigned short)c; S.pa[S.cp[c][1]] = (unsigned short)c; S.pa[S.cp[c][2]] = (unsigned short)c;
  }
  __syncwarp();
  const double rx = S.cx[0], ry = S.cy[0], rz = S.cz[0];   // reference point of the fan: corner 0
  double vol = 0, mx = 0, my = 0, mz = 0;
  int nnbr = 0, nlive = 0;
  for (int f0 = 0; f0 < np; f0 += kLanes) {
    const int f = f0 + lane;
    const bool live = f < np && S.pa[f] != 0xffff;
    double fx = 0, fy = 0, fz = 0;
    int fk = 0;
    // the planes of the faces adjacent to f, eight bits each: decoded only for a pair that is really pushed
    unsigned long long awp = 0ull;
    int naw = 0;
    if (live) {
      // walk the face loop: from a corner, the edge that starts at plane f leads to the next corner
      const int c0 = S.pa[f];
      const double ux = S.cx[c0] - rx, uy = S.cy[c0] - ry, uz = S.cz[c0] - rz;
      fx = S.cx[c0]; fy = S.cy[c0]; fz = S.cz[c0]; fk = 1;
      int c = c0;
      double vx = 0, vy = 0, vz = 0;
      for (int step = 0; step < nc; ++step) {
        const int t = (S.cp[c][0] == f) ? 0 : ((S.cp[c][1] == f) ? 1 : 2);
        {
          // the edge about to be walked separates f from the next plane of c's cyclic triple
          if (naw < 8) awp |= (unsigned long long)S.cp[c][t == 2 ? 0 : t + 1] << (8 * naw);
          ++naw;
        }
        c = S.cadj[c][t];
        if (c == c0) break;
        const double wx = S.cx[c] - rx, wy = S.cy[c] - ry, wz = S.cz[c] - rz;
        fx += S.cx[c]; fy += S.cy[c]; fz += S.cz[c]; ++fk;
        if (step > 0) {
          const double tv = (ux * (vy * wz - vz * wy) + uy * (vz * wx - vx * wz) + uz * (vx * wy - vy * wx)) * (1.0 / 6.0);
          vol += tv;
          mx += tv * (rx + 0.25 * (ux + vx + wx));
          my += tv * (ry + 0.25 * (uy + vy + wy));
          mz += tv * (rz + 0.25 * (uz + vz + wz));
        }
        vx = wx; vy = wy; vz = wz;
      }
    }
    const bool pos = live && S.pflag[f] >= 0;
    const unsigned pm = __ballot_sync(kFull, pos);
    nlive += __popc(__ballot_sync(kFull, live));
    // the face flags travel in key[][] (free until the corners are ranked): flag, then witness
    if (pos) {
      const int slot = nnbr + __popc(pm & ((1u << lane) - 1u));
      if (slot < C) {
        S.key[slot][0] = S.pflag[f];
        const double inv = 1.0 / fk;
        // witness: the face's corner average lies in T_a ∩ Omega_i ∩ Omega_j
        if (!A.dissolve) push_pair_faces(A, a, S.pflag[f], fx * inv + ox, fy * inv + oy, fz * inv + oz, i, awp, naw, S.pflag);
      }
    }
    if (A.dissolve && a != A.wholeA && live && S.pflag[f] < 0 && ~S.pflag[f] < A.m) {
      // Alg. 5 lines 20-24: the face of P on the face T_a shares with T_b lies in Omega_i, so (T_b, v_i) is a
      // non-empty pair; its witness is that face's corner average
      const double inv = 1.0 / fk;
      push_pair(A, ~S.pflag[f], i, fx * inv + ox, fy * inv + oy, fz * inv + oz);
    }
    nnbr += __popc(pm);
  }
  vol = warp_sum(vol); mx = warp_sum(mx); my = warp_sum(my); mz = warp_sum(mz);
  VD_WORK(extra_cnt_add(2, (unsigned)(3 * nc - 2 * nlive));)   // fan tetrahedra: every face of k corners gives k - 2; corners lie on 3 faces
  if (vol < 0) { vol = -vol; mx = -mx; my = -my; mz = -mz; }
  if (!(vol > 0)) {
#ifdef VD_TRACE
    if (lane == 0) printf("pair(%d,%d) dropped: vol=%g nc=%d\n", a, i, vol, nc);
#endif
    if (lane == 0) A.pieces[pairIdx] = pc;
    return 0;
  }
  if (nnbr > C) nnbr = C;
  // face flags -> pool
  unsigned long long nb0 = 0, vb0 = 0;
  if (wp) {
    // the two pool cursors are single addresses that every piece of the step would hit: a warp takes a chunk
    // at a time and hands out of it (the pools get holes; S6 gathers by (base, count) per piece)
    if (wp->nleft < nnbr) {
      const int take = max(wp->nchunk, nnbr);
      if (lane == 0) nb0 = atomicAdd(&A.ctl->nbrTail, (unsigned long long)take);
      wp->nbase = shfl(nb0, 0); wp->nleft = take;
    }
    if (wp->vleft < nc) {
      const int take = max(wp->vchunk, nc);
      if (lane == 0) vb0 = atomicAdd(&A.ctl->vertTail, (unsigned long long)take);
      wp->vbase = shfl(vb0, 0); wp->vleft = take;
    }
    nb0 = wp->nbase; wp->nbase += nnbr; wp->nleft -= nnbr;
    vb0 = wp->vbase; wp->vbase += nc; wp->vleft -= nc;
  } else {
    if (lane == 0) nb0 = atomicAdd(&A.ctl->nbrTail, (unsigned long long)nnbr);
    nb0 = shfl(nb0, 0);
    if (lane == 0) vb0 = atomicAdd(&A.ctl->vertTail, (unsigned long long)nc);
    vb0 = shfl(vb0, 0);
  }
  if ((int64_t)(nb0 + nnbr) > A.nbrCap || (int64_t)(vb0 + nc) > A.vertCap) {
    if (lane == 0) {
      atomicOr(&A.ctl->err, (int64_t)(vb0 + nc) > A.vertCap ? ERR_VERT_CAP : ERR_NBR_CAP);
      A.pieces[pairIdx] = pc;
    }
    return 0;
  }
  for (int k = lane; k < nnbr; k += kLanes) A.poolNbr[nb0 + k] = S.key[k][0];
  __syncwarp();
  // corners: ascending flag triple, corners ranked lexicographically by it.  Two 64-bit keys per corner (flags biased
  // to unsigned; the corner index breaks ties) in the scratch arrays key / remap / pa / pb, all free by now
  using PolyPC = Poly3<P, C>;
  static_assert(offsetof(PolyPC, be) - offsetof(PolyPC, key) >= 16 * (size_t)C, "room for two 64-bit keys per corner");
  ulonglong2* K = reinterpret_cast<ulonglong2*>(&S.key[0][0]);
  __syncwarp();
  for (int c = lane; c < nc; c += kLanes) {
    int f0 = S.pflag[S.cp[c][0]], f1 = S.pflag[S.cp[c][1]], f2 = S.pflag[S.cp[c][2]];
    int t;
    if (f0 > f1) { t = f0; f0 = f1; f1 = t; }
    if (f1 > f2) { t = f1; f1 = f2; f2 = t; }
    if (f0 > f1) { t = f0; f0 = f1; f1 = t; }
    ulonglong2 k;
    k.x = ((unsigned long long)((unsigned)f0 ^ 0x80000000u) << 32) | (unsigned long long)((unsigned)f1 ^ 0x80000000u);
    k.y = ((unsigned long long)((unsigned)f2 ^ 0x80000000u) << 32) | (unsigned long long)(unsigned)c;
    K[c] = k;
  }
  __syncwarp();
  for (int c = lane; c < nc; c += kLanes) {
    const ulonglong2 k = K[c];
    int rank = 0;
    for (int o = 0; o < nc; ++o) {
      const ulonglong2 q = K[o];
      rank += (q.x < k.x || (q.x == k.x && q.y < k.y)) ? 1 : 0;
    }
    const int k0 = (int)((unsigned)(k.x >> 32) ^ 0x80000000u), k1 = (int)((unsigned)k.x ^ 0x80000000u),
              k2 = (int)((unsigned)(k.y >> 32) ^ 0x80000000u);
    const int64_t v = (int64_t)vb0 + rank;
    A.poolXYZ[v * 3 + 0] = S.cx[c] + ox; A.poolXYZ[v * 3 + 1] = S.cy[c] + oy; A.poolXYZ[v * 3 + 2] = S.cz[c] + oz;
    A.poolFlags[v * 3 + 0] = k0; A.poolFlags[v * 3 + 1] = k1; A.poolFlags[v * 3 + 2] = k2;
  }
  if (lane == 0) {
    pc.nverts = nc; pc.nnbr = nnbr; pc.vbase = (int64_t)vb0; pc.nbase = (int64_t)nb0;
    pc.measure = vol;
    pc.mx = mx + vol * ox; pc.my = my + vol * oy; pc.mz = mz + vol * oz;
    A.pieces[pairIdx] = pc;
    atomicAdd(&A.sitePieces[i], 1);
    atomicAdd(&A.siteNbrRaw[i], nnbr);
  }
  lc.pieces += 1;
  return 0;
}

// ---- the steps of Alg. 3 on one (simplex, site) pair, as separate functions: the one-kernel path (clip_pair_3d)
// and the phased path (vd_phase.cu: one small kernel per step, the polytope parked in HBM between them) share them.

#define VD_POLY_REFS                                                                                               \
  const double &ox = S.u[0], &oy = S.u[1], &oz = S.u[2], &six = S.u[3], &siy = S.u[4], &siz = S.u[5];            \
  const double &vix = S.u[6], &viy = S.u[7], &viz = S.u[8], &wx = S.u[9], &wy = S.u[10], &wz = S.u[11];          \
  (void)ox; (void)oy; (void)oz; (void)six; (void)siy; (void)siz; (void)vix; (void)viy; (void)viz; (void)wx; (void)wy; (void)wz

// P <- T_a or the box (Alg. 3 line 1) and the per-pair constants S.u
template <int P, int C, bool BOX>
__device__ __forceinline__ void init_poly_3d(Poly3<P, C>& S, const ClipArgs& A, const Pair& pr, int& np, int& nc) {
  const int lane = lane_id();
  const int a = pr.a, i = pr.i;
  // ---- P <- T (Alg. 3 line 1): 4 planes (flags from the simplex adjacency), 4 corners.  Lane k < 4
  // loads tet vertex k; coordinates are local to vertex 0.  The per-pair constants live in shared memory
  // (S.u), not in registers: they would be spilled around every call of the query routines.
  np = 4; nc = 4;
  if (BOX || a == A.wholeA) {
    // simple domain (section V-B): P <- the box; verts holds its 8 corners, corner c = bits (x, y, z),
    // planes 0..5 = -x +x -y +y -z +z, local origin = lo
    double vx = 0, vy = 0, vz = 0;
    if (lane < 8) { vx = __ldg(&A.boxVerts[lane * 3 + 0]); vy = __ldg(&A.boxVerts[lane * 3 + 1]); vz = __ldg(&A.boxVerts[lane * 3 + 2]); }
    const double o0 = shfl(vx, 0), o1 = shfl(vy, 0), o2 = shfl(vz, 0);
    const double e0 = shfl(vx, 7) - o0, e1 = shfl(vy, 7) - o1, e2 = shfl(vz, 7) - o2;
    if (lane == 0) {
      const double s0 = __ldg(&A.sites[(int64_t)i * 3 + 0]), s1 = __ldg(&A.sites[(int64_t)i * 3 + 1]), s2 = __ldg(&A.sites[(int64_t)i * 3 + 2]);
      S.u[0] = o0; S.u[1] = o1; S.u[2] = o2;
      S.u[3] = s0; S.u[4] = s1; S.u[5] = s2;
      S.u[6] = s0 - o0; S.u[7] = s1 - o1; S.u[8] = s2 - o2;
      S.u[9] = pr.wx - o0; S.u[10] = pr.wy - o1; S.u[11] = pr.wz - o2;
      S.u[12] = (VD_EXT && A.siteW) ? __ldg(&A.siteW[i]) : 0.0; S.u[13] = 0.0;
    }
    if (lane < 6) {
      const int axis = lane >> 1, hiSide = lane & 1;
      const double sg = hiSide ? 1.0 : -1.0;
      S.pnx[lane] = axis == 0 ? sg : 0.0; S.pny[lane] = axis == 1 ? sg : 0.0; S.pnz[lane] = axis == 2 ? sg : 0.0;
      S.pd[lane] = hiSide ? (axis == 0 ? e0 : (axis == 1 ? e1 : e2)) : 0.0;
      S.pflag[lane] = ~A.m;
    }
    if (lane < 8) {
      const int c = lane;
      S.cx[c] = (c & 1) ? e0 : 0.0; S.cy[c] = (c & 2) ? e1 : 0.0; S.cz[c] = (c & 4) ? e2 : 0.0;
      const int px = (c & 1) ? 1 : 0, py = (c & 2) ? 3 : 2, pz = (c & 4) ? 5 : 4;
      // cyclic plane order mirrored at odd corners, so that neighbours traverse the shared edge in opposite directions
      const bool odd = __popc(c) & 1;
      S.cp[c][0] = (unsigned short)px; S.cp[c][1] = (unsigned short)(odd ? pz : py); S.cp[c][2] = (unsigned short)(odd ? py : pz);
      S.cadj[c][0] = (unsigned short)(odd ? (c ^ 2) : (c ^ 4));
      S.cadj[c][1] = (unsigned short)(c ^ 1);
      S.cadj[c][2] = (unsigned short)(odd ? (c ^ 4) : (c ^ 2));
      const int nn = __ldg(&A.boxVnn[c]);
      S.cnn[c] = nn;
      S.cstate[c] = (nn == i) ? ST_IN : ST_OUT;
    }
    np = 6; nc = 8;
  } else {
    double vx = 0, vy = 0, vz = 0;
    int vk = 0;
    if (lane < 4) {
      vk = __ldg(&A.simp[(int64_t)a * 4 + lane]);
      vx = __ldg(&A.verts[(int64_t)vk * 3 + 0]); vy = __ldg(&A.verts[(int64_t)vk * 3 + 1]); vz = __ldg(&A.verts[(int64_t)vk * 3 + 2]);
    }
    {
      const double o0 = shfl(vx, 0), o1 = shfl(vy, 0), o2 = shfl(vz, 0);
      if (lane < 4) { S.cx[lane] = vx - o0; S.cy[lane] = vy - o1; S.cz[lane] = vz - o2; }
      if (lane == 0) {
        const double s0 = __ldg(&A.sites[(int64_t)i * 3 + 0]), s1 = __ldg(&A.sites[(int64_t)i * 3 + 1]), s2 = __ldg(&A.sites[(int64_t)i * 3 + 2]);
        S.u[0] = o0; S.u[1] = o1; S.u[2] = o2;
        S.u[3] = s0; S.u[4] = s1; S.u[5] = s2;
        S.u[6] = s0 - o0; S.u[7] = s1 - o1; S.u[8] = s2 - o2;
        S.u[9] = pr.wx - o0; S.u[10] = pr.wy - o1; S.u[11] = pr.wz - o2;
        S.u[12] = (VD_EXT && A.siteW) ? __ldg(&A.siteW[i]) : 0.0; S.u[13] = 0.0;
      }
    }
    __syncwarp();
    if (lane < 4) {
      const int k = lane;
      const int q0 = (k + 1) & 3, q1 = (k + 2) & 3, q2 = (k + 3) & 3;
      const double ax = S.cx[q1] - S.cx[q0], ay = S.cy[q1] - S.cy[q0], az = S.cz[q1] - S.cz[q0];
      const double bx = S.cx[q2] - S.cx[q0], by = S.cy[q2] - S.cy[q0], bz = S.cz[q2] - S.cz[q0];
      double nx = ay * bz - az * by, ny = az * bx - ax * bz, nz = ax * by - ay * bx;
      const double side = nx * (S.cx[k] - S.cx[q0]) + ny * (S.cy[k] - S.cy[q0]) + nz * (S.cz[k] - S.cz[q0]);
      if (side > 0) { nx = -nx; ny = -ny; nz = -nz; }
      S.pnx[k] = nx; S.pny[k] = ny; S.pnz[k] = nz;
      S.pd[k] = nx * S.cx[q0] + ny * S.cy[q0] + nz * S.cz[q0];
      S.pflag[k] = ~__ldg(&A.adj[(int64_t)a * 4 + k]);
      // corner k = tet vertex k = the three faces other than k, cyclically ordered so that neighbouring
      // corners traverse their shared edge in opposite directions: (1,3,2) (0,2,3) (0,3,1) (0,1,2)
      const int t0 = (k == 0) ? 1 : 0;
      const int t1 = (k == 0) ? 3 : ((k == 1) ? 2 : ((k == 2) ? 3 : 1));
      const int t2 = (k == 0) ? 2 : ((k == 1) ? 3 : ((k == 2) ? 1 : 2));
      S.cp[k][0] = (unsigned short)t0; S.cp[k][1] = (unsigned short)t1; S.cp[k][2] = (unsigned short)t2;
      S.cadj[k][0] = (unsigned short)(6 - k - t0 - t1);
      S.cadj[k][1] = (unsigned short)(6 - k - t1 - t2);
      S.cadj[k][2] = (unsigned short)(6 - k - t2 - t0);
      // corners of T are classified from the per-vertex nearest site (S3): in Omega_i iff N_p = v_i
      const int nn = __ldg(&A.vnn[vk]);
      S.cnn[k] = nn;
      S.cstate[k] = (nn == i) ? ST_IN : ST_OUT;
    }
    __syncwarp();
  }
  __syncwarp();
}

// P <- P clipped by the bisector B_ij of a GIVEN site j, no search: any B_ij is a valid clip of Omega_i (Eq. 1).  A
// plane that does not cut P is skipped.  Returns 0, 1 (capacity), 2 (topology), -1 (skipped).
// (sx, sy, sz, sw: site j's coordinates and additive term, loaded by the caller -- for a whole list of sites at once, one per lane)
template <int P, int C>
__device__ __forceinline__ int clip_by_site_3d(Poly3<P, C>& S, const ClipArgs& A, int j, double sx, double sy, double sz, double sw, int& np, int& nc,
                                               LocalCnt& lc) {
  const int lane = lane_id();
  VD_POLY_REFS;
  const double wjx = sx - ox, wjy = sy - oy, wjz = sz - oz;
  const double nx = wjx - vix, ny = wjy - viy, nz = wjz - viz;
  const double d = 0.5 * (nx * (vix + wjx) + ny * (viy + wjy) + nz * (viz + wjz) + (sw - S.u[12]));
  // any corner clearly beyond the plane starts R_p: the corners of a convex polytope beyond a plane are connected over its
  // edges, so the flood of apply_clip_3d reaches the same set from each of them (a ballot instead of a warp argmin of the
  // farthest one)
  int p = -1;
  const double tol = 1e-9 * (nx * nx + ny * ny + nz * nz);
  for (int c0 = 0; c0 < nc && p < 0; c0 += kLanes) {
    const int c = c0 + lane;
    const bool beyond = c < nc && (nx * S.cx[c] + ny * S.cy[c] + nz * S.cz[c] - d > tol) && S.cstate[c] != ST_IN;
    const unsigned m = __ballot_sync(kFull, beyond);
    if (m) p = c0 + __ffs((int)m) - 1;
  }
  if (p < 0) return -1;   // the plane does not cut P
  if (np >= P) {
    compact_planes_3d(S, np, nc);
    if (np >= P) return 1;
  }
  VD_WORK(lc.clips += 1; lc.pre_clips += 1;)
  return apply_clip_3d(S, np, nc, p, -1, nx, ny, nz, d, j);
}

// Clips that need no search, before the point-in-cell loop of Alg. 3 starts:
// (a) a pair (a, i) discovered through the face of P_{a,u} on B_ui: that face lies in T_a, so B_iu bounds P_{a,i} --
//     the first clip of G_{a,j} (Fig. 6), taken from the tuple (u, f) the pair carries; then B_iw for
//     every face of P_{a,u} adjacent to f with a positive flag w ("clip by B_{j,w} for each adjacent face of f",
//     P:L211): cells u, i, w meet along that edge of f, which lies in T_a, so B_iw bounds P_{a,i} too;
// (b) reading U19: the bisectors of the sites nearest to v_i.  Most of them bound the cell, and what is left for the
//     point-in-cell loop is a small polytope around the cell.
// Returns 0, 1 (capacity), 2 (topology).
template <int P, int C>
__device__ __forceinline__ int preclip_3d(Poly3<P, C>& S, const ClipArgs& A, int a, int i, int u, const Pair* pp, int& np, int& nc, LocalCnt& lc) {
  const int lane = lane_id();
  if (A.firstClip && u >= 0 && u != i) {
    // lane 0: u; lanes 1 .. kPairW: the adjacent faces' sites (each bounds Omega_i along an edge of f that lies in T_a)
    int mine = -1;
    if (lane == 0) mine = u;
    else if (lane <= kPairW) mine = __ldcg(&pp->w[lane - 1]);
    // When every one of them cut P, the face of P on B_iu IS f: a convex polygon is the intersection of the
    // half-planes of its edges, f's edges come from exactly these faces (and faces of T_a, which P has), and on
    // B_iu the half-spaces H_iw and H_uw agree.  f is a face of the finished P_{a,u}, so its corners are in Omega_i:
    // they need no point-in-cell test.
    bool complete = true;
    const int pu = np;   // B_iu's plane index, if it cuts
    // every lane loads its own site: one round trip to L2 for the whole list instead of one per clip
    double sx = 0.0, sy = 0.0, sz = 0.0, sw = 0.0;
    if (mine >= 0) {
      sx = __ldg(&A.sites[(int64_t)mine * 3 + 0]); sy = __ldg(&A.sites[(int64_t)mine * 3 + 1]); sz = __ldg(&A.sites[(int64_t)mine * 3 + 2]);
      if (VD_EXT && A.siteW) sw = __ldg(&A.siteW[mine]);
    }
    for (int t = 0; t <= kPairW && nc > 0; ++t) {
      const int j = shfl(mine, t);
      if (j == -2) complete = false;   // f had more adjacent faces than a pair carries
      if (j < 0) break;
      if (j == i) { complete = false; continue; }
      const int rc = clip_by_site_3d(S, A, j, shfl(sx, t), shfl(sy, t), shfl(sz, t), (VD_EXT && A.siteW) ? shfl(sw, t) : 0.0, np, nc, lc);
      if (rc > 0) return rc;
      if (rc < 0) complete = false;
    }
    if (complete && nc > 0 && np < P) {   // (np == P: the plane list may have been compacted, pu renumbered)
      for (int c = lane; c < nc; c += kLanes)
        if (S.cp[c][0] == pu || S.cp[c][1] == pu || S.cp[c][2] == pu) S.cstate[c] = ST_IN;
      __syncwarp();
    }
  }
  if (A.nearList && nc > 0 && (!A.dissolve || a == A.wholeA)) {   // (dissolve mode: whole cells only)
    const int K = A.nearClips;
    int mine = lane < K ? __ldg(&A.nearList[(int64_t)i * K + lane]) : -1;
    {   // the list ends at its first negative entry (what follows may never have been written)
      const unsigned neg = __ballot_sync(kFull, mine < 0);
      if (neg && lane >= __ffs((int)neg) - 1) mine = -1;
    }
    double sx = 0.0, sy = 0.0, sz = 0.0, sw = 0.0;
    if (mine >= 0) {
      sx = __ldg(&A.sites[(int64_t)mine * 3 + 0]); sy = __ldg(&A.sites[(int64_t)mine * 3 + 1]); sz = __ldg(&A.sites[(int64_t)mine * 3 + 2]);
      if (VD_EXT && A.siteW) sw = __ldg(&A.siteW[mine]);
    }
    // which of the listed bisectors cut P as it stands?  One lane per plane, all planes at once (P only shrinks from here on, so a
    // plane that misses it now misses it for good); only those take their turn in the loop below -- on a mesh whose simplices are
    // smaller than the cells most of the list misses most pairs
    unsigned cand;
    {
      VD_POLY_REFS;
      bool cuts = false;
      if (mine >= 0) {
        const double wjx = sx - ox, wjy = sy - oy, wjz = sz - oz;
        const double nx = wjx - vix, ny = wjy - viy, nz = wjz - viz;
        const double d = 0.5 * (nx * (vix + wjx) + ny * (viy + wjy) + nz * (viz + wjz) + (sw - S.u[12]));
        const double tol = 1e-9 * (nx * nx + ny * ny + nz * nz);
        for (int c = 0; c < nc && !cuts; ++c) cuts = (nx * S.cx[c] + ny * S.cy[c] + nz * S.cz[c] - d > tol) && S.cstate[c] != ST_IN;
      }
      cand = __ballot_sync(kFull, cuts);
    }
    while (cand) {
      const int t = __ffs((int)cand) - 1;
      cand &= cand - 1;
      const int j = shfl(mine, t);
      const int rc = clip_by_site_3d(S, A, j, shfl(sx, t), shfl(sy, t), shfl(sz, t), (VD_EXT && A.siteW) ? shfl(sw, t) : 0.0, np, nc, lc);
      if (rc > 0) return rc;
      if (nc == 0) break;
    }
  }
  return 0;
}

// An outside corner p, preferring one with a neighbour p_s in Omega_i (a real edge, Alg. 1 line 3); -1 if no
// corner is known to be outside.
template <int P, int C>
__device__ __forceinline__ int select_out_3d(const Poly3<P, C>& S, const ClipArgs& A, int nc, int& sOut) {
  const int lane = lane_id();
  int p = -1, s = -1;
  for (int c0 = 0; c0 < nc && p < 0; c0 += kLanes) {
    const int c = c0 + lane;
    const bool out = c < nc && S.cstate[c] == ST_OUT;
    int sn = -1;
    if (out && A.realEdges) {
#pragma unroll
      for (int t = 0; t < 3; ++t)
        if (S.cstate[S.cadj[c][t]] == ST_IN) sn = S.cadj[c][t];
    }
    const unsigned mr = __ballot_sync(kFull, sn >= 0);
    const unsigned mo = __ballot_sync(kFull, out);
    if (mr) { const int src = __ffs(mr) - 1; p = c0 + src; s = shfl(sn, src); }
    else if (mo) { p = c0 + __ffs(mo) - 1; }
  }
  sOut = s;
  return p;
}

// Point-in-cell tests of the unclassified corners (section IV-A), up to kQB at a time in one batched
// pass (vd_batch.cuh); the batch state lives in the scratch area S.key.  Returns whether there were any.
// PolyT: Poly3<P, C>, or PolyTest3<P, C> (the members the tests touch, nothing else: k_ph_verify)
// DEFER (refined index, fast pass): corners whose test needs the single-query path are marked ST_LOOSE and left alone;
// *deferred tells whether there were any.  Without DEFER such marks count as unclassified.
template <class PolyT, bool HV, bool DEFER = false>
__device__ __forceinline__ bool classify_unknown_3d(PolyT& S, const GridIndex& g, int i, int np, int nc, StRef st, bool* deferred = nullptr) {
  const int lane = lane_id();
  VD_POLY_REFS;
  static_assert(sizeof(QBatch) + 40 <= sizeof(S.key), "the batch state must fit the scratch area");
  QBatch& Q = *reinterpret_cast<QBatch*>(&S.key[0][0]);
  bool any = false;
  for (;;) {
    int nq = 0;
    for (int c0 = 0; c0 < nc && nq < kQB; c0 += kLanes) {
      const int c = c0 + lane;
      const bool unk = c < nc && (S.cstate[c] == ST_UNKNOWN || (!DEFER && S.cstate[c] == ST_LOOSE));
      const unsigned m = __ballot_sync(kFull, unk);
      const int slot = nq + __popc(m & ((1u << lane) - 1u));
      if (unk && slot < kQB) {
        const double qx = S.cx[c] + ox, qy = S.cy[c] + oy, qz = S.cz[c] + oz;
        const double dx = qx - six, dy = qy - siy, dz = qz - siz;
        Q.item[slot] = c;
        Q.qx[slot] = qx; Q.qy[slot] = qy; Q.qz[slot] = qz;
        Q.best[slot] = dx * dx + dy * dy + dz * dz + S.u[12];
        Q.bestId[slot] = i;
      }
      nq = min(kQB, nq + __popc(m));
    }
    if (nq == 0) break;
    any = true;
    __syncwarp();
    const unsigned unanswered = batch_nearest<HV, !DEFER>(g, Q, nq, st);
    if (DEFER && unanswered) {
      if (lane < nq && ((unanswered >> lane) & 1u)) S.cstate[Q.item[lane]] = ST_LOOSE;
      *deferred = true;
    }
    if (lane < nq && !((unanswered >> lane) & 1u)) {
      const int c = Q.item[lane], id = Q.bestId[lane];
      // q in Omega_i iff no site is nearer than v_i (Eq. 1: the cell is closed).  A tie up to rounding (1e-13
      // relative in the squared distance) counts as inside; a near tie (1e-9) does when the other site already
      // owns a plane of P -- the flag rule in the form of reading U6.  A clearly nearer site (any
      // such site ends the query, U17) means outside.
      const double dx = Q.qx[lane] - six, dy = Q.qy[lane] - siy, dz = Q.qz[lane] - siz;
      const double di2 = dx * dx + dy * dy + dz * dz + S.u[12], best = Q.best[lane];
      bool inside = id == i || best >= di2 * (1.0 - 1e-13);
      if (!inside && best >= di2 * (1.0 - 1e-9))
        for (int f = 0; f < np && !inside; ++f) inside = (S.pflag[f] == id);
      S.cstate[c] = inside ? ST_IN : ST_OUT;
      S.cnn[c] = id;
#ifdef VD_TRACE
      printf("pair(?,%d) classify c=%d q=(%g,%g,%g) best=%g di2=%g id=%d inside=%d\n", i, c, Q.qx[lane], Q.qy[lane], Q.qz[lane], best, di2, id, (int)inside);
#endif
    }
    __syncwarp();
  }
  return any;
}

// One clipping from the known-outside corner p (Alg. 3 lines 3-4): bisector search on the real edge p_s p or on the
// virtual edge w p, then the clip.  Returns 0 ok, 1 capacity, 2 topology, 3 search cap.
// Returns 0 ok, 1 capacity, 2 topology, 3 search cap, 4 (DEFER only) the search needs the single-query path: nothing changed.
template <int P, int C, bool HV, bool DEFER = false>
__device__ __forceinline__ int clip_from_3d(Poly3<P, C>& S, const GridIndex& g, const ClipArgs& A, int i, int p, int s, int& np,
                                            int& nc, StRef st, LocalCnt& lc) {
  const int lane = lane_id();
  VD_POLY_REFS;
  if (np >= P) {
    compact_planes_3d(S, np, nc);
    if (np >= P) return 1;
  }
  static_assert(kSearchScratchBytes <= (int)sizeof(S.key), "the batch state and the search frame must fit the scratch area");
  double psx = wx, psy = wy, psz = wz;
  if (s >= 0) { psx = S.cx[s]; psy = S.cy[s]; psz = S.cz[s]; }
  double nx, ny, nz, d;
  const int j = find_bisector<HV, DEFER>(A, g, i, S.cnn[p], S.u, psx, psy, psz, S.cx[p], S.cy[p], S.cz[p], S.pflag, np,
                                         nx, ny, nz, d, st, lc, reinterpret_cast<double*>(&S.key[0][0]));
  if (DEFER && j == -2) return 4;
  if (j < 0) return 3;
  bool own = false;
  for (int f = lane; f < np; f += kLanes) own |= (S.pflag[f] == j);
  if (__any_sync(kFull, own)) {   // B_ij already bounds P: p lies on it up to rounding
    if (lane == 0) S.cstate[p] = ST_IN;
    __syncwarp();
    return 0;
  }
#ifdef VD_TRACE
  if (lane == 0) printf("pair(?,%d) clip p=%d(%g,%g,%g) s=%d j=%d nc=%d np=%d\n", i, p, S.cx[p]+ox, S.cy[p]+oy, S.cz[p]+oz, s, j, nc, np);
#endif
  VD_WORK(lc.clips += 1;)
  return apply_clip_3d(S, np, nc, p, s, nx, ny, nz, d, j);
}

// returns 0 = done (piece or empty recorded), 1 = capacity exceeded (caller defers the pair)
template <int P, int C, bool HV, bool BOX>
__device__ int clip_pair_3d(Poly3<P, C>& S, const GridIndex& g, const ClipArgs& A, int64_t pairIdx, StRef st, LocalCnt& lc) {
  const Pair pr = load_pair(A, pairIdx);
  const int a = pr.a, i = pr.i;
  int np, nc;
  init_poly_3d<P, C, BOX>(S, A, pr, np, nc);
  bool failed = false;
  {
    const int rc = preclip_3d(S, A, a, i, pr.u, &A.pairs[pairIdx], np, nc, lc);
    if (rc == 1) return 1;
    if (rc == 2) { failed = true; atomicOr(&A.ctl->err, ERR_TOPOLOGY); }
  }
  // ---- while P has a corner outside Omega_i (Alg. 3 line 2).  A corner known to be outside is clipped away
  // first; only when none is left are the unclassified corners tested: a clip removes unclassified corners
  // beyond its plane for free (they are candidates of R_p)
  for (int guard = 0; guard < 8 * P + 32 && !failed; ++guard) {
    int s;
    const int p = select_out_3d(S, A, nc, s);
    if (p < 0) {
      if (!classify_unknown_3d<Poly3<P, C>, HV>(S, g, i, np, nc, st)) break;   // every corner is in Omega_i
      continue;
    }
    const int rc = clip_from_3d<P, C, HV>(S, g, A, i, p, s, np, nc, st, lc);
    if (rc == 1) return 1;
    if (rc) { failed = true; atomicOr(&A.ctl->err, rc == 2 ? ERR_TOPOLOGY : ERR_NOCONVERGE); }
  }
  return finish_piece_3d(S, A, pairIdx, a, i, np, nc, S.u[0], S.u[1], S.u[2], failed, lc);
}

}  // namespace vd
