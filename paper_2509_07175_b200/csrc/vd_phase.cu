// vd_phase.cu -- S4 as a sequence of small kernels ("phased" mode, vd_options.persistent = 2) for the 3D kinds.
//
// The one-kernel clip path (vd_clip.cu) is bound by instruction fetch: ~100 KB of code whose 24 warps per SM sit
// in different steps of Alg. 3, against a 32 KB L1.5 instruction cache.  Here every step of Alg. 3 is its own
// kernel over all pairs of a wave, and the polytope of each pair is parked in HBM between the steps (5.2 KB per
// pair; a round over 1 M pairs moves ~10 GB, ~1.5 ms of HBM time -- bandwidth is what a B200 has to spare):
//
//   k_ph_init    P <- T_a or the box (Alg. 3 line 1), then the clips by the nearest sites (reading U19)
//   k_ph_verify  point-in-cell tests of all unclassified corners (section IV-A)          --+  rounds, until no
//   k_ph_fix     per pair with a corner outside: bisector search + clip (Alg. 3 l. 3-4)  --+  corner is outside
//   k_ph_finish  measure, moments, corners, flags, propagation
//
// Pairs pushed by k_ph_finish form the next wave (Alg. 4's L1/L2 swap).  Pairs that outgrow the fast tier
// go to the large-capacity kernel of vd_clip.cu, as in the other modes.
#include "vd_clip3d.cuh"

namespace vd {

#ifndef VD_PH_BLOCKS
#define VD_PH_BLOCKS 4   // resident blocks per SM of the verify / fix kernels (plain index)
#endif
#ifndef VD_PHV_BLOCKS
#define VD_PHV_BLOCKS VD_PH_BLOCKS   // the verify kernel's own (its shared memory would allow more than fix's)
#endif
constexpr int P3 = 32, C3 = 64;
constexpr int kTailPairs = 65536;   // a round with at most this many pairs left is finished by k_ph_tail
using PolyF = Poly3<P3, C3>;
using PolyT = PolyTest3<P3, C3>;   // k_ph_verify's view of a parked polytope

struct CellState {
  PolyF S;
  int np, nc;      // np < 0: the pair left the phased path (capacity: large tier)
  int a, i;
  int failed, pad[3];
};
static_assert(sizeof(CellState) % 16 == 0 && sizeof(PolyF) % 16 == 0, "copied in 16-byte words");

constexpr int kTestBytes = (int)offsetof(PolyF, pnx);    // what k_ph_verify reads (and, for cstate and cnn, writes back)
constexpr int kPolyBytes = (int)offsetof(PolyF, key);    // the polytope without its scratch arrays
static_assert(kTestBytes % 16 == 0 && kPolyBytes % 16 == 0, "copied in 16-byte words");
static_assert(offsetof(PolyT, key) == kTestBytes && offsetof(PolyT, cnn) == offsetof(PolyF, cnn) && offsetof(PolyT, cstate) == offsetof(PolyF, cstate),
              "PolyTest3 mirrors the head of Poly3");

struct PhaseCtl {
  unsigned ticket, nClip, nDone, pad;
};

// warp copy in 16-byte words, eight (then four) loads in flight per lane
__device__ __forceinline__ void copy_words(void* dst, const void* src, int bytes) {
  const uint4* s = reinterpret_cast<const uint4*>(src);
  uint4* d = reinterpret_cast<uint4*>(dst);
  const int n = bytes / 16, lane = lane_id();
  int k = lane;
  for (; k + 7 * kLanes < n; k += 8 * kLanes) {
    uint4 v[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) v[q] = s[k + q * kLanes];
#pragma unroll
    for (int q = 0; q < 8; ++q) d[k + q * kLanes] = v[q];
  }
  for (; k + 3 * kLanes < n; k += 4 * kLanes) {
    const uint4 a = s[k], b = s[k + kLanes], c = s[k + 2 * kLanes], e = s[k + 3 * kLanes];
    d[k] = a; d[k + kLanes] = b; d[k + 2 * kLanes] = c; d[k + 3 * kLanes] = e;
  }
  for (; k < n; k += kLanes) d[k] = s[k];
}

__device__ __forceinline__ int next_item(PhaseCtl* pc, int count) {
  unsigned t = 0;
  if (lane_id() == 0) t = atomicAdd(&pc->ticket, 1u);
  t = shfl(t, 0);
  return t < (unsigned)count ? (int)t : -1;
}

__device__ __forceinline__ void defer_pair(const ClipArgs& A, int64_t idx) {
  if (lane_id() == 0) {
    const unsigned long long slot = atomicAdd(&A.ctl->ovfTail, 1ull);
    if ((int64_t)slot < A.ovfCap) A.ovf[slot] = (int)idx; else atomicOr(&A.ctl->err, ERR_PAIR_CAP);
  }
}

template <bool BOX>
__global__ void __launch_bounds__(kBlock, 3) k_ph_init(ClipArgs A, CellState* __restrict__ cells, int64_t begin, int count, PhaseCtl* pc) {
  __shared__ PolyF S[kWarpsPerBlock];
  const int w = (int)threadIdx.x / kLanes, lane = lane_id();
  QueryStats st = {0u, 0u, 0u};
  LocalCnt lc = {0u, 0u, 0u, 0u, 0u, 0u};
  extra_cnt_reset();
  for (;;) {
    const int t = next_item(pc, count);
    if (t < 0) break;
    const Pair pr = load_pair(A, begin + t);
    int np, nc;
    init_poly_3d<P3, C3, BOX>(S[w], A, pr, np, nc);
    const int rc = preclip_3d(S[w], A, pr.i, pr.u, &A.pairs[begin + t], np, nc, lc);
    int failed = 0;
    if (rc == 1) { defer_pair(A, begin + t); np = -1; }
    if (rc == 2) { failed = 1; atomicOr(&A.ctl->err, ERR_TOPOLOGY); }
    __syncwarp();
    CellState* c = &cells[t];
    if (np >= 0) copy_words(&c->S, &S[w], kPolyBytes);
    if (lane == 0) { c->np = np; c->nc = nc; c->a = pr.a; c->i = pr.i; c->failed = failed; }
    __syncwarp();
  }
  flush_counters(A.ctl, st, lc, CNT_INIT);
}

// list == nullptr: items 0 .. count-1; a negative list entry is a pair that left the path
template <bool HV>
__global__ void __launch_bounds__(kBlock, HV ? 3 : VD_PHV_BLOCKS) k_ph_verify(ClipArgs A, CellState* __restrict__ cells, const int* __restrict__ list, int count,
                                                     int* __restrict__ clipList, int* __restrict__ doneList, PhaseCtl* pc) {
  __shared__ GridIndex g;
  __shared__ PolyT S[kWarpsPerBlock];
  if (threadIdx.x == 0) g = *A.grid;
  __syncthreads();
  const int w = (int)threadIdx.x / kLanes, lane = lane_id();
  QueryStats st = {0u, 0u, 0u};
  LocalCnt lc = {0u, 0u, 0u, 0u, 0u, 0u};
  extra_cnt_reset();
  for (;;) {
    const int t = next_item(pc, count);
    if (t < 0) break;
    const int slot = list ? list[t] : t;
    if (slot < 0) continue;
    CellState* c = &cells[slot];
    const int np = c->np, nc = c->nc;
    if (np < 0) continue;
    bool out = false;
    if (!c->failed && nc > 0) {
      copy_words(&S[w], &c->S, kTestBytes);
      __syncwarp();
      const bool any = classify_unknown_3d<PolyT, HV>(S[w], g, c->i, np, nc, st);
      for (int k = lane; k < nc; k += kLanes) out |= (S[w].cstate[k] == ST_OUT);
      out = __any_sync(kFull, out);
      if (any) {
        copy_words(c->S.cnn, S[w].cnn, (nc * 4 + 15) & ~15);
        copy_words(c->S.cstate, S[w].cstate, (nc + 15) & ~15);
      }
    }
    if (lane == 0) {
      if (out) clipList[atomicAdd(&pc->nClip, 1u)] = slot;
      else doneList[atomicAdd(&pc->nDone, 1u)] = slot;
    }
    __syncwarp();
  }
  flush_counters(A.ctl, st, lc, CNT_VERIFY);
}

// every corner known to be outside is clipped away (its search, its clip); the new corners wait for the next
// round of tests.  The list is rewritten in place: the slot, or -1 when the pair left the path.
template <bool HV>
__global__ void __launch_bounds__(kBlock, HV ? 3 : VD_PH_BLOCKS) k_ph_fix(ClipArgs A, CellState* __restrict__ cells, int* __restrict__ list, int count,
                                                     int64_t begin, PhaseCtl* pc) {
  __shared__ GridIndex g;
  __shared__ PolyF S[kWarpsPerBlock];
  if (threadIdx.x == 0) g = *A.grid;
  __syncthreads();
  const int w = (int)threadIdx.x / kLanes, lane = lane_id();
  QueryStats st = {0u, 0u, 0u};
  LocalCnt lc = {0u, 0u, 0u, 0u, 0u, 0u};
  extra_cnt_reset();
  for (;;) {
    const int t = next_item(pc, count);
    if (t < 0) break;
    const int slot = list[t];
    CellState* c = &cells[slot];
    int np = c->np, nc = c->nc;
    const int i = c->i;
    copy_words(&S[w], &c->S, kPolyBytes);
    __syncwarp();
    int failed = 0;
    for (int guard = 0; guard < 4 * P3 && nc > 0; ++guard) {
      int s;
      const int p = select_out_3d(S[w], A, nc, s);
      if (p < 0) break;
      const int rc = clip_from_3d<P3, C3, HV>(S[w], g, A, i, p, s, np, nc, st, lc);
      if (rc == 1) { defer_pair(A, begin + slot); np = -1; break; }
      if (rc) { failed = 1; atomicOr(&A.ctl->err, rc == 2 ? ERR_TOPOLOGY : ERR_NOCONVERGE); break; }
    }
    __syncwarp();
    if (np >= 0) copy_words(&c->S, &S[w], kPolyBytes);
    if (lane == 0) {
      c->np = np; c->nc = nc; c->failed = failed;
      list[t] = np >= 0 ? slot : -1;
    }
    __syncwarp();
  }
  flush_counters(A.ctl, st, lc, CNT_FIX);
}

// The last few pairs of a wave (a verify round left fewer than kTailPairs with a corner outside): tests and clips
// alternate inside one launch until every corner is in Omega_i -- Alg. 3's loop as it stands --
// instead of one round trip to the host and two nearly empty launches per remaining round.  Finished pairs join the
// done list.  The whole loop in one kernel is the instruction-fetch-bound form (header of this file); on a few
// thousand pairs that does not matter.
template <bool HV>
__global__ void __launch_bounds__(kBlock, 3) k_ph_tail(ClipArgs A, CellState* __restrict__ cells, const int* __restrict__ list, int count,
                                                       int64_t begin, int* __restrict__ doneList, PhaseCtl* pc) {
  __shared__ GridIndex g;
  __shared__ PolyF S[kWarpsPerBlock];
  if (threadIdx.x == 0) g = *A.grid;
  __syncthreads();
  const int w = (int)threadIdx.x / kLanes, lane = lane_id();
  QueryStats st = {0u, 0u, 0u};
  LocalCnt lc = {0u, 0u, 0u, 0u, 0u, 0u};
  extra_cnt_reset();
  for (;;) {
    const int t = next_item(pc, count);
    if (t < 0) break;
    const int slot = list[t];
    CellState* c = &cells[slot];
    int np = c->np, nc = c->nc;
    const int i = c->i;
    copy_words(&S[w], &c->S, kPolyBytes);
    __syncwarp();
    int failed = 0;
    for (int guard = 0; guard < 8 * P3 + 32 && nc > 0; ++guard) {
      int s;
      const int p = select_out_3d(S[w], A, nc, s);
      if (p < 0) {
        if (!classify_unknown_3d<PolyF, HV>(S[w], g, i, np, nc, st)) break;   // every corner is in Omega_i
        continue;
      }
      const int rc = clip_from_3d<P3, C3, HV>(S[w], g, A, i, p, s, np, nc, st, lc);
      if (rc == 1) { defer_pair(A, begin + slot); np = -1; break; }
      if (rc) { failed = 1; atomicOr(&A.ctl->err, rc == 2 ? ERR_TOPOLOGY : ERR_NOCONVERGE); break; }
    }
    __syncwarp();
    if (np >= 0) copy_words(&c->S, &S[w], kPolyBytes);
    if (lane == 0) {
      c->np = np; c->nc = nc; c->failed = failed;
      if (np >= 0) doneList[atomicAdd(&pc->nDone, 1u)] = slot;
    }
    __syncwarp();
  }
  flush_counters(A.ctl, st, lc, CNT_TAIL);
}

__global__ void __launch_bounds__(kBlock, 3) k_ph_finish(ClipArgs A, CellState* __restrict__ cells, const int* __restrict__ list, int count,
                                                     int64_t begin, int vchunk, int nchunk) {
  __shared__ PolyF S[kWarpsPerBlock];
  const int w = (int)threadIdx.x / kLanes;
  QueryStats st = {0u, 0u, 0u};
  LocalCnt lc = {0u, 0u, 0u, 0u, 0u, 0u};
  extra_cnt_reset();
  WarpPool wp = {0ull, 0ull, 0, 0, vchunk, nchunk};
  // uniform work per piece: a static stride instead of a ticket (one same-address atomic less per piece)
  const int stride = (int)gridDim.x * kWarpsPerBlock;
  for (int t = (int)blockIdx.x * kWarpsPerBlock + w; t < count; t += stride) {
    const int slot = list[t];
    const CellState* c = &cells[slot];
    copy_words(&S[w], &c->S, kPolyBytes);
    __syncwarp();
    finish_piece_3d(S[w], A, begin + slot, c->a, c->i, c->np, c->nc, S[w].u[0], S[w].u[1], S[w].u[2], c->failed != 0, lc, &wp);
    __syncwarp();
  }
  flush_counters(A.ctl, st, lc, CNT_FINISH);
}

static vd_status reset_ctl(vd_ctx* c, PhaseCtl* pc, bool all) {
  return cuda_check(c, cudaMemsetAsync(pc, 0, all ? sizeof(PhaseCtl) : sizeof(unsigned) * 2, c->stream), "phase ctl");
}

// One wave: pairs [begin, end) of the pair list, all of one 3D kind.  Every launch is bracketed by two events;
// the elapsed times are read after the round's synchronisation (vd_get_phase_ms).
vd_status run_phases(vd_ctx* c, const ClipArgs& A, bool hv, int64_t begin, int64_t end) {
  const int64_t chunk = (int64_t)1 << 20;
  const int64_t cap = end - begin < chunk ? end - begin : chunk;
  vd_status s;
  if ((s = ensure(c, c->phaseCells, sizeof(CellState) * (size_t)cap))) return s;
  if ((s = ensure(c, c->phaseLists, sizeof(int) * 3 * (size_t)cap + sizeof(PhaseCtl)))) return s;
  for (cudaEvent_t& e : c->phaseEv)
    if (!e && cudaEventCreate(&e) != cudaSuccess) return cuda_check(c, cudaGetLastError(), "phase events");
  CellState* cells = c->phaseCells.as<CellState>();
  int* listA = c->phaseLists.as<int>();
  int* listB = listA + cap;
  int* done = listB + cap;
  PhaseCtl* pc = reinterpret_cast<PhaseCtl*>(done + cap);
  cudaStream_t st = c->stream;
  cudaEvent_t* ev = c->phaseEv;
  const int grid = sm_count() * 4;
  const int tailPairs = c->opt.tail_pairs == 0 ? kTailPairs : c->opt.tail_pairs;   // < 0: never
  auto elapsed = [&](int which, cudaEvent_t a, cudaEvent_t b) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, a, b) == cudaSuccess) c->phaseMs[which] += ms;
  };
  auto read_ctl = [&](PhaseCtl& h) -> cudaError_t {
    // through page-locked memory: a copy into pageable memory is staged by the driver (tens of microseconds, once per round)
    PhaseCtl* dst = c->pinned ? reinterpret_cast<PhaseCtl*>(c->pinned) : &h;
    cudaError_t e = cudaMemcpyAsync(dst, pc, sizeof(h), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = sync_stream(c);
    if (e == cudaSuccess && dst != &h) h = *dst;
    return e;
  };
  for (int64_t b = begin; b < end; b += chunk) {
    const int count = (int)((end - b) < chunk ? (end - b) : chunk);
    if ((s = reset_ctl(c, pc, true))) return s;
    cudaEventRecord(ev[0], st);
    if (c->kind == KIND_BOX_3D) VD_LAUNCH(k_ph_init<true>, grid, kBlock, 0, st)(A, cells, b, count, pc);
    else VD_LAUNCH(k_ph_init<false>, grid, kBlock, 0, st)(A, cells, b, count, pc);
    cudaEventRecord(ev[1], st);
    const int* cur = nullptr;
    int curCount = count;
    int* clip = listA;
    int* other = listB;
    bool initTimed = false, fixPending = false;
    PhaseCtl h;
    for (int round = 0; round < 4 * P3; ++round) {
      if ((s = reset_ctl(c, pc, false))) return s;   // ticket and nClip; nDone keeps growing
      cudaEventRecord(ev[2], st);
      if (hv) VD_LAUNCH(k_ph_verify<true>, grid, kBlock, 0, st)(A, cells, cur, curCount, clip, done, pc);
      else VD_LAUNCH(k_ph_verify<false>, grid, kBlock, 0, st)(A, cells, cur, curCount, clip, done, pc);
      cudaEventRecord(ev[3], st);
      const cudaError_t e = read_ctl(h);
      if (e != cudaSuccess) return cuda_check(c, e, "phase round");
      if (!initTimed) { elapsed(0, ev[0], ev[1]); initTimed = true; }
      if (fixPending) { elapsed(2, ev[1], ev[2]); fixPending = false; }   // previous fix: between its start mark and this verify
      elapsed(1, ev[2], ev[3]);
      if (h.nClip == 0) break;
      if ((s = cuda_check(c, cudaMemsetAsync(&pc->ticket, 0, sizeof(unsigned), st), "phase ctl"))) return s;
      if ((int)h.nClip <= tailPairs) {
        cudaEventRecord(ev[1], st);
        if (hv) VD_LAUNCH(k_ph_tail<true>, grid, kBlock, 0, st)(A, cells, clip, (int)h.nClip, b, done, pc);
        else VD_LAUNCH(k_ph_tail<false>, grid, kBlock, 0, st)(A, cells, clip, (int)h.nClip, b, done, pc);
        cudaEventRecord(ev[2], st);
        const cudaError_t e2 = read_ctl(h);
        if (e2 != cudaSuccess) return cuda_check(c, e2, "phase tail");
        elapsed(4, ev[1], ev[2]);
        break;
      }
      cudaEventRecord(ev[1], st);
      if (hv) VD_LAUNCH(k_ph_fix<true>, grid, kBlock, 0, st)(A, cells, clip, (int)h.nClip, b, pc);
      else VD_LAUNCH(k_ph_fix<false>, grid, kBlock, 0, st)(A, cells, clip, (int)h.nClip, b, pc);
      fixPending = true;
      cur = clip;
      curCount = (int)h.nClip;
      int* tmp = clip; clip = other; other = tmp;
    }
    if (h.nDone > 0) {
      // pool chunk per warp: ~1/32 of an even share of the pool, so that the slack (one open chunk per warp) stays small
      // static stride over the grid: exactly the resident blocks (3 per SM), or the last third would run alone
      const int fgrid = sm_count() * 3;
      const int64_t warps = (int64_t)fgrid * kWarpsPerBlock;
      auto chunk_of = [&](int64_t cap) { const int64_t v = cap / (warps * 32); return (int)(v > 1024 ? 1024 : v); };   // small pools: piece by piece
      cudaEventRecord(ev[0], st);
      VD_LAUNCH(k_ph_finish, fgrid, kBlock, 0, st)(A, cells, done, (int)h.nDone, b, chunk_of(c->vertCap), chunk_of(c->nbrCap));
      cudaEventRecord(ev[1], st);
      const cudaError_t e = sync_stream(c);
      if (e != cudaSuccess) return cuda_check(c, e, "phase finish");
      elapsed(3, ev[0], ev[1]);
    }
  }
  return cuda_check(c, cudaGetLastError(), "phases");
}

}  // namespace vd
