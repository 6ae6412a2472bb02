// vd_clip_args.cuh -- kernel arguments and small helpers shared by the 2D/surface and 3D clip kernels.
#pragma once
#include "vd_internal.h"
#include "vd_nearest.cuh"
#include "vd_batch.cuh"

#ifndef VD_SEARCH_BATCH
#define VD_SEARCH_BATCH 1   // refined index: a search's queries go through the batched multi-view pass (0: the single-query path)
#endif
#ifndef VD_ONE_SHOT_HV
#define VD_ONE_SHOT_HV 0
#endif
namespace vd {

struct ClipArgs {
  const GridIndex* grid;
  const double* sites;     // [n][3] original order
  const double* siteW;     // [n] additive term eta - w_i of every site (power diagrams of 3-D sites), or nullptr
  const double* verts;     // [nv][3]
  const int* simp;         // [m][nc]
  const int* adj;          // [m][nc]
  const int* vnn;          // [nv] nearest site of every mesh vertex
  const int* nearList;     // [n][nearClips] or nullptr
  int n, m, kind;
  int realEdges, ballCells, nearClips;
  int firstClip;           // 1: a discovered pair (a, i) is first clipped by B_iu, u the discovering site
  int aBegin, aEnd;        // simplices seeded by this context (vd_options.simplex_begin / simplex_end; a rank's block of M)
  // Whole cells (section V-B; Alg. 5 line 6): a pair whose simplex id is wholeA starts from the box boxVerts (8 corners, corner
  // c = bits x, y, z; their nearest sites in boxVnn) instead of a simplex.  VD_BOX_3D: wholeA = 0, the box is the domain.
  // Dissolve mode of VD_TET_3D (Alg. 5): wholeA = m, the box is the mesh's bounding box; such pairs push nothing, and tet
  // pairs propagate over NEGATIVE flags (same site, adjacent tet: Alg. 5 lines 20-24).  Otherwise wholeA = -1.
  int wholeA, dissolve;
  const double* boxVerts;
  const int* boxVnn;
  int queue;               // 1: the pair list is read by a running kernel (device-side queue): publish slots with a fence
  Control* ctl;
  Pair* pairs;
  Piece* pieces;
  unsigned long long* visited;
  uint64_t hashMask;
  int64_t pairCap, vertCap, nbrCap, ovfCap;
  int* ovf;
  double* poolXYZ;
  int* poolFlags;
  int* poolNbr;
  int* sitePieces;
  int* siteNbrRaw;
};

enum { ST_UNKNOWN = 0, ST_IN = 1, ST_OUT = 2,
       ST_LOOSE = 3 };   // unclassified, and its point-in-cell test needs the single-query path (left for the second pass)

// State of one WAVE PROGRAM (vd_clip.cu): the fixed sequence of launches that processes one wavefront of pairs with no
// host in between.  Its first kernel (k_wave_begin) looks at the pair list and decides what the wave is; every other
// kernel of the program reads that decision, and the counts it needs, from here.
constexpr int kMaxRounds = 6;
enum { WAVE_NONE = 0,     // nothing to do (the list is exhausted, or an error is pending)
       WAVE_PHASED = 1,   // 3D kinds: one kernel per step of Alg. 3, polytopes parked in HBM (vd_phase.cu)
       WAVE_QUEUE = 2,    // the one-kernel form as a device-side queue: drains this wave and everything it discovers
       WAVE_SINGLE = 3 }; // the one-kernel form over exactly this wave
struct PhaseCtl {
  unsigned mode, count;             // WAVE_*, pairs of this wave (phased: at most the parking capacity)
  unsigned long long begin;         // first pair of the wave in the pair list
  unsigned nDone, pad;
  unsigned nClip[kMaxRounds + 2];   // pairs with a corner outside after the tests of round r
  unsigned nLoose[kMaxRounds + 2];  // refined index: pairs whose tests / searches of round r need the single-query path
  unsigned nLooseFix[kMaxRounds + 2];
  unsigned ticket[4 * kMaxRounds + 4];   // one work cursor per launch of the program
};

struct LocalCnt {
  unsigned pairs, pieces, search_iters, clips, search_evals, pre_clips;
};

__device__ __forceinline__ void flush_counters(Control* ctl, const QueryStats&, const LocalCnt& lc, int kind = CNT_OTHER) {
  __syncwarp();
  if (lane_id() == 0) {
    const WarpStats st = warp_stats();
    Counters* cnt = &ctl->cnt[kind];
    atomicAdd(&cnt->pairs, (unsigned long long)lc.pairs);
    atomicAdd(&cnt->pieces, (unsigned long long)lc.pieces);
    atomicAdd(&cnt->search_iters, (unsigned long long)lc.search_iters);
    atomicAdd(&cnt->clips, (unsigned long long)lc.clips);
    if (lc.search_evals) atomicAdd(&cnt->search_evals, (unsigned long long)lc.search_evals);
    if (lc.pre_clips) atomicAdd(&cnt->pre_clips, (unsigned long long)lc.pre_clips);
    atomicAdd(&cnt->queries, (unsigned long long)st.queries);
    atomicAdd(&cnt->dist_evals, (unsigned long long)st.dist_evals);
    atomicAdd(&cnt->rows, (unsigned long long)st.rows);
    const unsigned* x = sExtraCnt[(threadIdx.x / kLanes) % kWarpsPerBlock];
    if (x[0]) atomicAdd(&cnt->clip_corners, (unsigned long long)x[0]);
    if (x[1]) atomicAdd(&cnt->new_corners, (unsigned long long)x[1]);
    if (x[2]) atomicAdd(&cnt->fan_simplices, (unsigned long long)x[2]);
    if (x[3]) atomicAdd(&cnt->step_probes, (unsigned long long)x[3]);
    if (x[4]) atomicAdd(&cnt->alg_evals, (unsigned long long)x[4]);
    if (x[5]) atomicAdd(&cnt->f32_survivors, (unsigned long long)x[5]);
  }
}

// Propagation (Alg. 4 lines 11-15): a positive flag j on an edge/face of P_{a,i} means
// Omega_j meets T_a; push (a, j) once, with a witness point on that edge/face.
__device__ __forceinline__ void push_pair(const ClipArgs& A, int a, int j, double wx, double wy, double wz, int u = -1,
                                          int w0 = -1, int w1 = -1, int w2 = -1, int w3 = -1, int w4 = -1, int w5 = -1, int w6 = -1) {
  if (!visit(A.visited, A.hashMask, a, j)) return;
  const unsigned long long slot = atomicAdd(&A.ctl->pairTail, 1ull);
  if ((int64_t)slot >= A.pairCap) { atomicOr(&A.ctl->err, ERR_PAIR_CAP); return; }
  // the simplex id doubles as the slot's ready flag for the device-side queue: written last, after a fence
  Pair* p = &A.pairs[slot];
  p->i = j; p->wx = wx; p->wy = wy; p->wz = wz;
  if (u >= 0) {   // the list was filled with -1 (S3)
    p->u = u;
    p->w[0] = w0; p->w[1] = w1; p->w[2] = w2; p->w[3] = w3; p->w[4] = w4; p->w[5] = w5; p->w[6] = w6;
  }
  if (A.queue) __threadfence();   // other schedules read the list in a later launch
  *reinterpret_cast<volatile int*>(&p->a) = a;
}

// The same for a pair discovered through a face f of a finished 3D piece: the adjacent faces arrive as plane indices
// (eight bits each in `planes`, `nplanes` of them, at most eight kept) and are turned into sites here, after the
// visited test -- four out of five pushes end there.
__device__ __forceinline__ void push_pair_faces(const ClipArgs& A, int a, int j, double wx, double wy, double wz, int u,
                                                unsigned long long planes, int nplanes, const int* pflag) {
  if (!visit(A.visited, A.hashMask, a, j)) return;
  const unsigned long long slot = atomicAdd(&A.ctl->pairTail, 1ull);
  if ((int64_t)slot >= A.pairCap) { atomicOr(&A.ctl->err, ERR_PAIR_CAP); return; }
  Pair* p = &A.pairs[slot];
  p->i = j; p->wx = wx; p->wy = wy; p->wz = wz;
  p->u = u;
  int cnt = 0;
  const int kept = nplanes < 8 ? nplanes : 8;
  for (int k = 0; k < kept; ++k) {
    const int fl = pflag[(int)((planes >> (8 * k)) & 0xffull)];
    if (fl >= 0) {
      if (cnt < kPairW) p->w[cnt] = fl;   // (the list was filled with -1: S3)
      ++cnt;
    }
  }
  // more adjacent faces than a pair carries: the mark sits right behind the last site (the reader stops at the first
  // negative entry)
  if (nplanes > 8 || cnt > kPairW) p->w[cnt < kPairW ? cnt : kPairW - 1] = -2;
  if (A.queue) __threadfence();
  *reinterpret_cast<volatile int*>(&p->a) = a;
}

// A pair may have been written by another SM a moment ago: read it past the (incoherent) L1.
__device__ __forceinline__ Pair load_pair(const ClipArgs& A, int64_t idx) {
  const Pair* p = &A.pairs[idx];
  Pair r;
  r.a = __ldcg(&p->a); r.i = __ldcg(&p->i);
  r.wx = __ldcg(&p->wx); r.wy = __ldcg(&p->wy); r.wz = __ldcg(&p->wz);
  r.u = __ldcg(&p->u);   // w[] is read lane by lane where it is used (preclip_3d)
  return r;
}

// Next unit of work for this warp, or -1.  Wave mode: tickets begin .. end-1 of the current wave (Alg. 4's
// "for each pair in L1 in parallel").  Persistent mode: the pair list is a device-side queue; a
// ticket beyond the tail waits until the pair is pushed, and the kernel ends when every dispatched pair
// has finished (then nobody can push any more): no host round trip per wave.
template <bool BIG>
__device__ __forceinline__ int64_t next_ticket(const ClipArgs& A, int64_t begin, int64_t end, bool persist) {
  long long t = 0;
  if (lane_id() == 0) {
    t = (long long)atomicAdd(&A.ctl->fetch[BIG ? 1 : 0], 1ull) + begin;
    if (!persist) {
      if (t >= end) t = -1;
    } else {
      for (;;) {
        const unsigned long long fin = *reinterpret_cast<volatile unsigned long long*>(&A.ctl->finished);
        unsigned long long tail = *reinterpret_cast<volatile unsigned long long*>(&A.ctl->pairTail);
        if (tail > (unsigned long long)A.pairCap) tail = (unsigned long long)A.pairCap;
        if ((unsigned long long)t < tail) break;
        if (fin >= tail) { t = -1; break; }
        __nanosleep(256);
      }
      if (t >= 0) {
        while (*reinterpret_cast<volatile int*>(&A.pairs[t].a) < 0) __nanosleep(64);
        __threadfence();
      }
    }
  }
  return (int64_t)shfl(t, 0);
}

__device__ __forceinline__ void pair_done(const ClipArgs& A) {
  __syncwarp();
  if (lane_id() == 0) {
    __threadfence();
    atomicAdd(&A.ctl->finished, 1ull);
  }
}

// Whole-cell kinds (reading U19): up to k of the sites nearest to v_i among the 3 x 3 x 3 grid cells around it,
// nearest first, into out[]; returns how many.  Any bisector B_ij is a valid clip of Omega_i (Eq. 1), and the
// nearest few sites are almost always Voronoi neighbours, so clipping the box by them first costs no search and
// leaves a small polytope whose corners are all close to the cell.  Selection is approximate on purpose: each
// lane keeps the two nearest of the candidates it saw, the k best of those 64 win.
#ifndef VD_NEAR_R
#define VD_NEAR_R 1   // half width, in cells, of the window near_sites looks around in (at most 2)
#endif
#ifndef VD_NEAR_LIMIT
#define VD_NEAR_LIMIT 256   // (measured on C3: 16 -> 207 ms, 64 -> 177, 256 -> 174, 1024 -> 174)
#endif
// A site in a refined cell (clustered sites) looks around in that cell's sub-grid instead: the 27 top cells around it hold
// thousands of sites there, of which the first 512 in storage order are no one's nearest.
static __device__ __noinline__ int near_sites(const GridIndex& gTop, double vx, double vy, double vz, int i, int k, int* out, StRef st) {
  __shared__ int sBaseN[kWarpsPerBlock][kLanes];
  const int lane = lane_id();
  int* base = sBaseN[(threadIdx.x / kLanes) % kWarpsPerBlock];
  const GridIndex* gp = &gTop;
  if (gTop.subOff) {
    const int tx = cell_of(gTop, 0, vx), ty = cell_of(gTop, 1, vy), tz = cell_of(gTop, 2, vz);
    const int so = __ldg(&gTop.subOff[(tz * gTop.G[1] + ty) * gTop.G[0] + tx]);
    if (so >= 0) {
      GridIndex& v = warp_view();
      __syncwarp();
      if (lane == 0) sub_view(gTop, tx, ty, tz, so, v);
      __syncwarp();
      gp = &v;
    }
  }
  const GridIndex& g = *gp;
  const int cx = cell_of(g, 0, vx), cy = cell_of(g, 1, vy), cz = cell_of(g, 2, vz);
  const int x0 = max(cx - VD_NEAR_R, 0), x1 = min(cx + VD_NEAR_R, g.G[0] - 1);
  const int y0 = max(cy - VD_NEAR_R, 0), y1 = min(cy + VD_NEAR_R, g.G[1] - 1);
  const int z0 = max(cz - VD_NEAR_R, 0), z1 = min(cz + VD_NEAR_R, g.G[2] - 1);
  const int ny = y1 - y0 + 1, nrows = ny * (z1 - z0 + 1);   // (at most 25: one lane per row)
  int s = 0, cnt = 0;
  if (lane < nrows) {
    const int rz = lane / ny;
    const int rowBase = ((z0 + rz) * g.G[1] + y0 + (lane - rz * ny)) * g.G[0];
    s = __ldg(&g.cellStart[rowBase + x0]);
    cnt = __ldg(&g.cellStart[rowBase + x1 + 1]) - s;
  }
  double md = 2e300, md2 = 2e300;   // the nearest and the second nearest this lane saw
  int mi = 0x7fffffff, mi2 = 0x7fffffff;
  const int total = for_each_packed(s, cnt, base, VD_NEAR_LIMIT * kLanes /* a dense neighbourhood: the first VD_NEAR_LIMIT x 32 candidates will do */, [](int) {},
                                    [&](bool valid, int pos, int) {
    if (valid) {
      const double4 p = g.sites[pos];
      const int id = (int)(__double_as_longlong(p.w) & 0x7fffffff);
      const double dx = vx - p.x, dy = vy - p.y, dz = vz - p.z;
      const double d2 = dx * dx + dy * dy + dz * dz;
      if (id != i && d2 > 0.0) {
        if (closer(d2, id, md, mi)) { md2 = md; mi2 = mi; md = d2; mi = id; }
        else if (closer(d2, id, md2, mi2)) { md2 = d2; mi2 = id; }
      }
    }
  });
  VD_STAT(st.dist_evals += (unsigned)total;)
  int found = 0;
  for (; found < k; ++found) {
    double bd = md;
    int bi = mi;
    warp_argmin(bd, bi);
    if (bi == 0x7fffffff) break;
    if (lane == 0) out[found] = bi;
    if (mi == bi) { md = md2; mi = mi2; md2 = 2e300; mi2 = 0x7fffffff; }
  }
  __syncwarp();
  return found;
}

// One-shot form of the edge-based bisector search (reading U18).  Along p_s -> p_t every g_k(t) = |x-v_k|^2 -
// |x-v_i|^2 is linear and >= 0 at p_s, so the target bisector is the one with the smallest crossing parameter
// t_k.  With q = B_ij ∩ segment (parameter tq), every site whose bisector crosses before q is nearer to q than
// v_i, i.e. lies in the ball (q, |q - v_i|): one complete scan of that ball, keeping the smallest t_k, ends the
// search -- P:L137's iteration would visit a chain of such sites one nearest-site query at a time.  Sites nearer
// only within rounding do not compete (1e-13 relative; 1e-9 when the site owns a flag of P: the flag rule of
// P:L109-111, readings U6/U17).  Returns false, doing nothing, when the ball covers too many grid cells (q still
// far from Omega_i): the caller then takes an ordinary step.  Coordinates are absolute.  Warp-uniform result.
// Refined index (HV): the scan needs plain cells -- a ball inside one refined cell is scanned in that cell's sub-grid (viewed
// as a grid of its own); a ball that touches a refined cell otherwise is declined.
template <bool HV>
static __device__ __noinline__ bool scan_ball_min_t(const GridIndex& gTop, double qx, double qy, double qz, double r2, double psx,
                                                    double psy, double psz, double dis2, double tq, int i, int j, const int* flags,
                                                    int nflags, int maxCells, double& tbest, int& jbest, StRef st) {
  __shared__ int sBaseT[kWarpsPerBlock][kLanes];
  const int lane = lane_id();
  int* base = sBaseT[(threadIdx.x / kLanes) % kWarpsPerBlock];
  const double r = sqrt(r2);
  const GridIndex* gp = &gTop;
  bool checkRefined = HV;
  if (HV) {
    const int hx = cell_of(gTop, 0, qx), hy = cell_of(gTop, 1, qy), hz = cell_of(gTop, 2, qz);
    const int so = __ldg(&gTop.subOff[(hz * gTop.G[1] + hy) * gTop.G[0] + hx]);
    if (so >= 0) {
      if (!ball_in_cell(gTop, hx, hy, hz, qx, qy, qz, r)) return false;
      GridIndex& v = warp_view();
      __syncwarp();
      if (lane == 0) sub_view(gTop, hx, hy, hz, so, v);
      __syncwarp();
      gp = &v;
      checkRefined = false;
    }
  }
  const GridIndex& g = *gp;
  const int x0 = cell_of(g, 0, qx - r - 1e-6 * g.h[0]), x1 = cell_of(g, 0, qx + r + 1e-6 * g.h[0]);
  const int y0 = cell_of(g, 1, qy - r - 1e-6 * g.h[1]), y1 = cell_of(g, 1, qy + r + 1e-6 * g.h[1]);
  const int z0 = cell_of(g, 2, qz - r - 1e-6 * g.h[2]), z1 = cell_of(g, 2, qz + r + 1e-6 * g.h[2]);
  const int ny = y1 - y0 + 1;
  const int nrows = ny * (z1 - z0 + 1);
  if (nrows > kLanes || nrows * (x1 - x0 + 1) > maxCells) return false;
  int s = 0, cnt = 0;
  bool refined = false;
  if (lane < nrows) {
    const int rz = lane / ny;
    const int y = y0 + (lane - rz * ny), z = z0 + rz;
    const double rd2 = slab_d2(g, 1, qy, y, y) + slab_d2(g, 2, qz, z, z);
    if (!(rd2 > r2)) {
      const double w = sqrt(r2 - rd2);
      const int xa = max(x0, (int)floor((qx - w - g.lo[0]) * g.inv_h[0] - 1e-6));
      const int xb = min(x1, (int)floor((qx + w - g.lo[0]) * g.inv_h[0] + 1e-6));
      if (xa <= xb) {
        const int rowBase = (z * g.G[1] + y) * g.G[0];
        s = __ldg(&g.cellStart[rowBase + xa]);
        cnt = __ldg(&g.cellStart[rowBase + xb + 1]) - s;
        if (HV && checkRefined && cnt > kHeavy)
          refined = __ldg(&g.heavyPrefix[rowBase + xb + 1]) != __ldg(&g.heavyPrefix[rowBase + xa]);
      }
    }
  }
  if (HV && __any_sync(kFull, refined)) return false;
  VD_STAT(st.queries += 1;)
  VD_STAT(st.rows += (unsigned)nrows;)
  double tb = 2.0;
  int jb = 0x7fffffff;
  const int total = for_each_packed(s, cnt, base, 0x7fffffff, [](int) {}, [&](bool valid, int pos, int) {
    if (valid) {
      const double4 p = g.sites[pos];
      const int id = (int)(__double_as_longlong(p.w) & 0x7fffffff);
      const double dx = qx - p.x, dy = qy - p.y, dz = qz - p.z;
      const double pw = has_weights(g) ? __ldg(&g.sitesW[pos]) : 0.0;
      const double dq2 = dx * dx + dy * dy + dz * dz + pw;
      bool cand = id != i && id != j && dq2 < r2 * (1.0 - 1e-13);
      if (cand && !(dq2 < r2 * (1.0 - 1e-9)))
        for (int f = 0; f < nflags; ++f) cand = cand && (flags[f] != id);
      if (cand) {
        const double ex = psx - p.x, ey = psy - p.y, ez = psz - p.z;
        const double gs = ex * ex + ey * ey + ez * ez + pw - dis2, gq = dq2 - r2;
        const double tk = gs > 0.0 ? tq * gs / (gs - gq) : 0.0;
        if (closer(tk, id, tb, jb)) { tb = tk; jb = id; }
      }
    }
  });
  VD_STAT(st.dist_evals += (unsigned)total;)
  warp_argmin(tb, jb);
  if (closer(tb, jb, tbest, jbest)) { tbest = tb; jbest = jb; }
  if (counts_alg(gTop)) extra_cnt_add(4, lane == 0 ? ball_sites(gTop, qx, qy, qz, r2) : 0u);   // the search needs every site of this ball
  return true;
}

// Improved search of section VI-A (Fig. 8): before the search on a long segment p_s p_t, step out from p_s in
// multiples of delta_i (S1b): g = p_s + lambda delta_i dir, lambda = 2, 3, ... (stepMode 2: lambda doubles), while
// g is still in Omega_i; the first g outside, with its nearest site, replaces p_t -- the search then runs on the short
// segment p_s g.  g never passes p_t (reading U7); a probe that meets the end of the segment leaves p_t as it is.  Coordinates
// local to o = u[0..2]; the new end point and its site come back through pt[3] / j.  Returns the number of probes.
template <bool HV>
static __device__ __noinline__ int step_out(const GridIndex& g, int i, int& j, const double* u, double psx, double psy, double psz, double* pt,
                                            const int* flags, int nflags, StRef st) {
  const double delta = __ldg(&g.delta[i]);
  const double sx = pt[0] - psx, sy = pt[1] - psy, sz = pt[2] - psz;
  const double len = sqrt(sx * sx + sy * sy + sz * sz);
  int probes = 0;
  if (!(delta > 0.0) || !(len > 2.0 * delta)) return 0;
  const double inv = 1.0 / len;
  double lambda = 2.0;
  for (int k = 0; k < 64; ++k) {
    const double s = lambda * delta;
    if (!(s < len)) break;
    const double gx = psx + sx * inv * s, gy = psy + sy * inv * s, gz = psz + sz * inv * s;
    const double ax = gx + u[0], ay = gy + u[1], az = gz + u[2];
    const double dx = ax - u[3], dy = ay - u[4], dz = az - u[5];
    const double di2 = dx * dx + dy * dy + dz * dz + u[12];
    double best = di2;
    int bestId = i;
    nearest<HV>(g, ax, ay, az, best, bestId, st, true);
    probes += 1;
    bool outside = bestId != i && best < di2 * (1.0 - 1e-9);   // clearly nearer to another site (U8): g has left Omega_i
    if (outside) { pt[0] = gx; pt[1] = gy; pt[2] = gz; j = bestId; break; }
    lambda = g.stepMode == 1 ? lambda + 1.0 : lambda * 2.0;
  }
  (void)flags; (void)nflags;
  return probes;
}

// Edge-based bisector search (section IV-B) on the segment p_s -> p_t, all in coordinates
// local to the origin o.  p_s is in Omega_i, the nearest site of p_t is j != i.  Iterates
// q = B_ij ∩ segment, k = N_q, until k is i or j; then B_ij is the target bisector.  Along the segment
// every g_k(t) = |x-v_k|^2 - |x-v_i|^2 is linear, so this is Newton's iteration on the concave
// piecewise-linear min_k g_k from t = 1 (reading U7).  flags[0..nflags) are the flags of P's edges/faces:
// the segment lies in P, and P is inside H_ik for every site k that owns one of them, so N_q = v_k can
// only be a tie and also means q in Omega_i -- the flag rule of P:L109-111 for a point on an edge/face of P
// (a real edge, or a virtual edge that runs inside a bisector face).  Returns j, or -1 at the cap.
// The state of one search (warp-uniform): it lives in the warp's shared-memory scratch behind the batch of queries, NOT in
// registers -- the doubles that the loop carries across its calls of the (not inlined) query routines were the largest
// source of spill loads / stores of the step kernels.  Lane 0 writes, the warp synchronises before anyone reads and again
// before the next write (the lanes of a warp need not be in step after a call).
struct SearchFrame {
  double plane[4];        // out: the bisector (n, d) of the site returned
  double ps[3], pt[3];    // the segment, local to o
  double q[3];            // the intersecting point of the current iteration
  double di2, dj2;
  unsigned iters, pad;
};
constexpr int kSearchScratchBytes = ((int)sizeof(QBatch) + 7) / 8 * 8 + (int)sizeof(SearchFrame);

template <bool HV, bool DEFER = false>
// DEFER (refined index, fast pass): a query that needs the single-query path ends the search with -2, nothing changed.
// The arguments are scalars and pointers on purpose: a struct passed by reference to this (not inlined) function
// would be copied into every thread's local memory.  The segment comes in and the plane goes out through the frame.
static __device__ __noinline__ int find_bisector_impl(const double* __restrict__ sites, int ballCells, const GridIndex& g, int i, int j,
                                             const double* u,   // per-pair constants (shared memory): origin, v_i absolute, v_i local
                                             SearchFrame* sf, const int* flags, int nflags, QBatch* qb, StRef st) {
  const double &ox = u[0], &oy = u[1], &oz = u[2], &vix = u[6], &viy = u[7], &viz = u[8];
  if (has_step_out(g)) {   // section VI-A (vd_options.step_out): shorten the segment first
    double pt[3] = {sf->pt[0], sf->pt[1], sf->pt[2]};
    const int probes = step_out<HV>(g, i, j, u, sf->ps[0], sf->ps[1], sf->ps[2], pt, flags, nflags, st);
    __syncwarp();
    if (probes) { if (lane_id() == 0) { sf->pt[0] = pt[0]; sf->pt[1] = pt[1]; sf->pt[2] = pt[2]; } extra_cnt_add(3, (unsigned)probes); }
    __syncwarp();
  }
  for (int it = 0; it < 96; ++it) {
    double ax, ay, az;
    {
      const double psx = sf->ps[0], psy = sf->ps[1], psz = sf->ps[2], ptx = sf->pt[0], pty = sf->pt[1], ptz = sf->pt[2];
      const double vjx = __ldg(&sites[(int64_t)j * 3 + 0]) - ox, vjy = __ldg(&sites[(int64_t)j * 3 + 1]) - oy,
                   vjz = __ldg(&sites[(int64_t)j * 3 + 2]) - oz;
      const double wi = u[12], wj = site_w(g, j);   // power diagram: the lifted sites' fourth coordinates, squared (else 0)
      const double nx = vjx - vix, ny = vjy - viy, nz = vjz - viz;
      const double d = 0.5 * (nx * (vix + vjx) + ny * (viy + vjy) + nz * (viz + vjz) + (wj - wi));
      const double gs = d - (nx * psx + ny * psy + nz * psz);
      const double gt = d - (nx * ptx + ny * pty + nz * ptz);
      const double den = gs - gt;
      double t = den > 0.0 ? gs / den : 1.0;
      t = fmin(fmax(t, 0.0), 1.0);
      const double qx = psx + t * (ptx - psx), qy = psy + t * (pty - psy), qz = psz + t * (ptz - psz);
      // point-in-cell test of the intersecting point: N_q in {i, j} means q is in Omega_i
      ax = qx + ox; ay = qy + oy; az = qz + oz;
      const double dix = ax - u[3], diy = ay - u[4], diz = az - u[5];
      const double djx = ax - (vjx + ox), djy = ay - (vjy + oy), djz = az - (vjz + oz);
      const double di2 = dix * dix + diy * diy + diz * diz + wi, dj2 = djx * djx + djy * djy + djz * djz + wj;
      __syncwarp();   // every lane has read the segment (and, in the previous iteration, q and the bounds)
      if (lane_id() == 0) {
        sf->plane[0] = nx; sf->plane[1] = ny; sf->plane[2] = nz; sf->plane[3] = d;
        sf->q[0] = qx; sf->q[1] = qy; sf->q[2] = qz;
        sf->di2 = di2; sf->dj2 = dj2;
        sf->iters = (unsigned)(it + 1);
      }
      __syncwarp();
      if ((!HV || VD_ONE_SHOT_HV) && ballCells > 0) {   // (on the refined index the one-shot scan measured slower: C3 583 -> 632 ms)
        // close enough to Omega_i for a complete scan of the ball: the site whose bisector crosses first ends the search
        double tb = 2.0;
        int jb = 0x7fffffff;
        const double sx = psx + ox - u[3], sy = psy + oy - u[4], sz = psz + oz - u[5];
        if (scan_ball_min_t<HV>(g, ax, ay, az, di2, psx + ox, psy + oy, psz + oz, sx * sx + sy * sy + sz * sz + wi, t, i, j, flags, nflags,
                            ballCells, tb, jb, st)) {
          if (jb != 0x7fffffff) {
            j = jb;
            const double wjx = __ldg(&sites[(int64_t)j * 3 + 0]) - ox, wjy = __ldg(&sites[(int64_t)j * 3 + 1]) - oy,
                         wjz = __ldg(&sites[(int64_t)j * 3 + 2]) - oz;
            const double mx = wjx - vix, my = wjy - viy, mz = wjz - viz;
            const double md = 0.5 * (mx * (vix + wjx) + my * (viy + wjy) + mz * (viz + wjz) + (site_w(g, j) - u[12]));
            __syncwarp();
            if (lane_id() == 0) { sf->plane[0] = mx; sf->plane[1] = my; sf->plane[2] = mz; sf->plane[3] = md; }
          }
          __syncwarp();
          return j;
        }
        ax = sf->q[0] + ox; ay = sf->q[1] + oy; az = sf->q[2] + oz;   // (the same sums again, not kept across the call)
      }
    }
    double best = sf->di2;
    int bestId = i;
    if (closer(sf->dj2, j, best, bestId)) { best = sf->dj2; bestId = j; }
    if (HV && qb && VD_SEARCH_BATCH) {
      // refined index: the query as a batch of one -- the cell-by-cell pass over sub-grids (vd_batch.cuh) instead of the
      // general single-query search
      if (lane_id() == 0) { qb->qx[0] = ax; qb->qy[0] = ay; qb->qz[0] = az; qb->best[0] = best; qb->bestId[0] = bestId; }
      __syncwarp();
      const unsigned unanswered = batch_nearest<HV, !DEFER>(g, *qb, 1, st);
      if (DEFER && unanswered) return -2;
      __syncwarp();
      best = qb->best[0]; bestId = qb->bestId[0];
      __syncwarp();
    } else {
      nearest<HV>(g, ax, ay, az, best, bestId, st, true);
    }
    const double bound = fmin(sf->di2, sf->dj2);
    if (bestId == i || bestId == j || best >= bound * (1.0 - 1e-13)) return j;   // nothing nearer, up to rounding
    if (best >= bound * (1.0 - 1e-9)) {   // a (near) tie with a site that owns a plane of P: flag rule
      bool own = false;
      for (int f = lane_id(); f < nflags; f += kLanes) own |= (flags[f] == bestId);
      if (__any_sync(kFull, own)) return j;
    }
    j = bestId;
    __syncwarp();   // the bounds have been read by every lane
    if (lane_id() == 0) { sf->pt[0] = sf->q[0]; sf->pt[1] = sf->q[1]; sf->pt[2] = sf->q[2]; }
    __syncwarp();
  }
  return -1;
}

// scratch: the warp's shared-memory scratch (kSearchScratchBytes: the batch of queries, then the search frame)
template <bool HV, bool DEFER = false>
__device__ __forceinline__ int find_bisector(const ClipArgs& A, const GridIndex& g, int i, int j, const double* u, double psx, double psy,
                                             double psz, double ptx, double pty, double ptz, const int* flags, int nflags, double& nx,
                                             double& ny, double& nz, double& d, StRef st, LocalCnt& lc, double* scratch) {
  const unsigned e0 = warp_stats().dist_evals;
  QBatch* qb = reinterpret_cast<QBatch*>(scratch);
  SearchFrame* sf = reinterpret_cast<SearchFrame*>(scratch + (sizeof(QBatch) + 7) / 8);
  __syncwarp();
  if (lane_id() == 0) {
    sf->ps[0] = psx; sf->ps[1] = psy; sf->ps[2] = psz; sf->pt[0] = ptx; sf->pt[1] = pty; sf->pt[2] = ptz;
    sf->iters = 0u;
  }
  __syncwarp();
  const int r = find_bisector_impl<HV, DEFER>(A.sites, A.ballCells, g, i, j, u, sf, flags, nflags, qb, st);
  __syncwarp();
  nx = sf->plane[0]; ny = sf->plane[1]; nz = sf->plane[2]; d = sf->plane[3];
  const unsigned iters = sf->iters;
  VD_WORK(lc.search_iters += iters;)
  (void)iters;
  __syncwarp();
  VD_WORK(lc.search_evals += warp_stats().dist_evals - e0;)
  (void)e0;
  return r;
}

}  // namespace vd
