// vd_clip_args.cuh -- kernel arguments and small helpers shared by the 2D/surface and 3D clip kernels.
#pragma once
#include "vd_internal.h"
#include "vd_nearest.cuh"

namespace vd {

struct ClipArgs {
  const GridIndex* grid;
  const double* sites;     // [n][3] original order
  const double* verts;     // [nv][3]
  const int* simp;         // [m][nc]
  const int* adj;          // [m][nc]
  const int* vnn;          // [nv] nearest site of every mesh vertex
  int n, m, kind;
  int realEdges, stepOut;
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

enum { ST_UNKNOWN = 0, ST_IN = 1, ST_OUT = 2 };

struct LocalCnt {
  unsigned pairs, pieces, search_iters, clips;
};

__device__ __forceinline__ void flush_counters(Control* ctl, const QueryStats& st, const LocalCnt& lc) {
  if (lane_id() == 0) {
    atomicAdd(&ctl->cnt.pairs, (unsigned long long)lc.pairs);
    atomicAdd(&ctl->cnt.pieces, (unsigned long long)lc.pieces);
    atomicAdd(&ctl->cnt.search_iters, (unsigned long long)lc.search_iters);
    atomicAdd(&ctl->cnt.clips, (unsigned long long)lc.clips);
    atomicAdd(&ctl->cnt.queries, (unsigned long long)st.queries);
    atomicAdd(&ctl->cnt.dist_evals, (unsigned long long)st.dist_evals);
    atomicAdd(&ctl->cnt.rows, (unsigned long long)st.rows);
  }
}

// Propagation (Alg. 4 lines 11-15): a positive flag j on an edge/face of P_{a,i} means
// Omega_j meets T_a; push (a, j) once, with a witness point on that edge/face.
__device__ __forceinline__ void push_pair(const ClipArgs& A, int a, int j, double wx, double wy, double wz) {
  if (!visit(A.visited, A.hashMask, a, j)) return;
  const unsigned long long slot = atomicAdd(&A.ctl->pairTail, 1ull);
  if ((int64_t)slot >= A.pairCap) { atomicOr(&A.ctl->err, ERR_PAIR_CAP); return; }
  // the simplex id doubles as the slot's ready flag for the device-side queue: written last, after a fence
  Pair* p = &A.pairs[slot];
  p->i = j; p->wx = wx; p->wy = wy; p->wz = wz;
  __threadfence();
  *reinterpret_cast<volatile int*>(&p->a) = a;
}

// A pair may have been written by another SM a moment ago: read it past the (incoherent) L1.
__device__ __forceinline__ Pair load_pair(const ClipArgs& A, int64_t idx) {
  const Pair* p = &A.pairs[idx];
  Pair r;
  r.a = __ldcg(&p->a); r.i = __ldcg(&p->i);
  r.wx = __ldcg(&p->wx); r.wy = __ldcg(&p->wy); r.wz = __ldcg(&p->wz);
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

// Edge-based bisector search (section IV-B) on the segment p_s -> p_t, all in coordinates
// local to the origin o.  p_s is in Omega_i, the nearest site of p_t is j != i.  Iterates
// q = B_ij ∩ segment, k = N_q, until k is i or j; then B_ij is the target bisector.  Along the segment
// every g_k(t) = |x-v_k|^2 - |x-v_i|^2 is linear, so this is Newton's iteration on the concave
// piecewise-linear min_k g_k from t = 1 (reading U7).  flags[0..nflags) are the flags of P's edges/faces:
// the segment lies in P, and P is inside H_ik for every site k that owns one of them, so N_q = v_k can
// only be a tie and also means q in Omega_i -- the flag rule of P:L109-111 for a point on an edge/face of P
// (a real edge, or a virtual edge that runs inside a bisector face).  Returns j, or -1 at the cap.
template <bool HV>
static __device__ __noinline__ int find_bisector(const ClipArgs& A, const GridIndex& g, int i, int j,
                                             const double* u,   // per-pair constants (shared memory): origin, v_i absolute, v_i local
                                             double psx, double psy, double psz, double ptx, double pty, double ptz, const int* flags, int nflags,
                                             double& nx, double& ny, double& nz, double& d, QueryStats& st, LocalCnt& lc) {
  const double &ox = u[0], &oy = u[1], &oz = u[2], &vix = u[6], &viy = u[7], &viz = u[8];
  for (int it = 0; it < 96; ++it) {
    lc.search_iters += 1;
    const double vjx = __ldg(&A.sites[(int64_t)j * 3 + 0]) - ox, vjy = __ldg(&A.sites[(int64_t)j * 3 + 1]) - oy,
                 vjz = __ldg(&A.sites[(int64_t)j * 3 + 2]) - oz;
    nx = vjx - vix; ny = vjy - viy; nz = vjz - viz;
    d = 0.5 * (nx * (vix + vjx) + ny * (viy + vjy) + nz * (viz + vjz));
    const double gs = d - (nx * psx + ny * psy + nz * psz);
    const double gt = d - (nx * ptx + ny * pty + nz * ptz);
    const double den = gs - gt;
    double t = den > 0.0 ? gs / den : 1.0;
    t = fmin(fmax(t, 0.0), 1.0);
    const double qx = psx + t * (ptx - psx), qy = psy + t * (pty - psy), qz = psz + t * (ptz - psz);
    // point-in-cell test of the intersecting point: N_q in {i, j} means q is in Omega_i
    const double ax = qx + ox, ay = qy + oy, az = qz + oz;
    const double dix = ax - u[3], diy = ay - u[4], diz = az - u[5];
    const double djx = ax - (vjx + ox), djy = ay - (vjy + oy), djz = az - (vjz + oz);
    const double di2 = dix * dix + diy * diy + diz * diz, dj2 = djx * djx + djy * djy + djz * djz;
    double best = di2;
    int bestId = i;
    if (closer(dj2, j, best, bestId)) { best = dj2; bestId = j; }
    nearest<HV>(g, ax, ay, az, best, bestId, st, true);
#ifdef VD_TRACE
    if (lane_id() == 0) printf("      search i=%d j=%d t=%.17g q=(%g,%g) gs=%g gt=%g -> N_q=%d\n", i, j, t, ax, ay, gs, gt, bestId);
#endif
    const double bound = fmin(di2, dj2);
    if (bestId == i || bestId == j || best >= bound * (1.0 - 1e-13)) return j;   // nothing nearer, up to rounding
    if (best >= bound * (1.0 - 1e-9)) {   // a (near) tie with a site that owns a plane of P: flag rule
      bool own = false;
      for (int f = lane_id(); f < nflags; f += kLanes) own |= (flags[f] == bestId);
      if (__any_sync(kFull, own)) return j;
    }
    j = bestId;
    ptx = qx; pty = qy; ptz = qz;
  }
  return -1;
}

}  // namespace vd
