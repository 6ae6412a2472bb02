// vd_phase.cu -- S4 as a sequence of small kernels ("phased" mode, the default of the 3D kinds: vd_options.persistent = 1 / 2).
//
// The one-kernel clip path (vd_clip.cu) is bound by instruction fetch: ~100 KB of code whose 24 warps per SM sit
// in different steps of Alg. 3, against a 32 KB L1.5 instruction cache.  Here every step of Alg. 3 is its own
// kernel over all pairs of a wave, and the polytope of each pair is parked in HBM between the steps (5.2 KB per
// pair; a round over 1 M pairs moves ~10 GB, ~1.5 ms of HBM time -- bandwidth is what a B200 has to spare):
//
//   k_ph_init    P <- T_a or the box (Alg. 3 line 1), then the clips by the nearest sites (reading U19)
//   k_ph_verify  point-in-cell tests of all unclassified corners (section IV-A)          --+  rounds, until no
//   k_ph_fix     per pair with a corner outside: bisector search + clip (Alg. 3 l. 3-4)  --+  corner is outside
//   k_ph_tail    what the rounds leave: tests and clips to completion in one launch
//   k_ph_finish  measure, moments, corners, flags, propagation
//
// The kernels of a wave are enqueued as one fixed sequence (enqueue_phased, part of a "wave program": vd_clip.cu); each reads
// from PhaseCtl in device memory whether it has work and how much, so the host does not look between them.  Polytopes move
// between HBM and shared memory through the TMA unit (vd_tma.cuh).  On the refined index k_ph_verify and k_ph_fix run as a
// fast pass (without the single-query search code) and a second pass for the pairs it leaves (MODE).
// Pairs pushed by k_ph_finish form the next wave (Alg. 4's L1/L2 swap).  Pairs that outgrow the fast tier
// go to the large-capacity kernel of vd_clip.cu, as in the other modes.
#include "vd_clip3d.cuh"
#include "vd_tma.cuh"

namespace vd {
namespace VD_VARIANT {   // compiled twice: header of vd_clip.cu

#ifndef VD_PH_BLOCKS
#define VD_PH_BLOCKS 4   // resident blocks per SM of the verify / fix kernels (plain index)
#endif
#ifndef VD_PH_BLOCKS_HV
#define VD_PH_BLOCKS_HV 4   // the same for the kernels that know the refined index (measured on C3: 2 blocks 451 ms, 3 blocks 416 ms, 4 blocks 405 ms)
#endif
#ifndef VD_TWO_PASS
#define VD_TWO_PASS 1   // refined index: fast pass + second pass of the verify / fix kernels (0: one complete pass)
#endif
#ifndef VD_PH_TAIL_BLOCKS
#define VD_PH_TAIL_BLOCKS 3
#endif
#ifndef VD_PHV_BLOCKS
#define VD_PHV_BLOCKS VD_PH_BLOCKS   // the verify kernel's own (its shared memory would allow more than fix's)
#endif
#ifndef VD_PHV_BLOCKS_HV
#define VD_PHV_BLOCKS_HV VD_PH_BLOCKS_HV   // (measured on C3, verify alone: 3 blocks 100.0 ms, 4 blocks 91.1, 5 blocks 95.2, 6 blocks 100.4)
#endif
constexpr int P3 = 32, C3 = 64;
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

// Parked polytope -> shared memory through the TMA unit: lane 0 issues the bulk copy, every lane waits on the warp's mbarrier
// (whose phase parity the caller keeps).  VD_NO_TMA: the per-lane load / store loops (for comparison).
__device__ __forceinline__ void unpark(void* smem, const void* gmem, int bytes, unsigned long long* bar, unsigned& parity) {
#ifdef VD_NO_TMA
  copy_words(smem, gmem, bytes);
  __syncwarp();
#else
  __syncwarp();   // every lane is done with what the buffer held
  if (lane_id() == 0) tma_load(smem, gmem, (unsigned)bytes, bar);
  tma_wait(bar, parity);
  parity ^= 1u;
#endif
}

// Shared memory -> parked polytope; returns when the shared-memory source may be overwritten.
__device__ __forceinline__ void park(void* gmem, const void* smem, int bytes) {
#ifdef VD_NO_TMA
  copy_words(gmem, smem, bytes);
  __syncwarp();
#else
  __syncwarp();   // the warp's stores to the buffer are done
  if (lane_id() == 0) { tma_store(gmem, smem, (unsigned)bytes); tma_store_commit(); tma_store_wait_read(); }
  __syncwarp();
#endif
}

#define VD_WARP_BAR                                                        \
  __shared__ unsigned long long sBar[kWarpsPerBlock];                      \
  unsigned long long* bar = &sBar[(int)threadIdx.x / kLanes];              \
  unsigned parity = 0u;                                                    \
  if (lane_id() == 0) tma_bar_init(bar);                                   \
  __syncwarp()

__device__ __forceinline__ int next_item(PhaseCtl* pc, int slot, int count) {
  unsigned t = 0;
  if (lane_id() == 0) t = atomicAdd(&pc->ticket[slot], 1u);
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
__global__ void __launch_bounds__(kBlock, 3) k_ph_init(ClipArgs A, CellState* __restrict__ cells, PhaseCtl* pc) {
  if (pc->mode != WAVE_PHASED) return;
  const int64_t begin = (int64_t)pc->begin;
  const int count = (int)pc->count;
  __shared__ PolyF S[kWarpsPerBlock];
  const int w = (int)threadIdx.x / kLanes, lane = lane_id();
  QueryStats st = {0};
  LocalCnt lc = {0u, 0u, 0u, 0u, 0u, 0u};
  extra_cnt_reset();
  for (;;) {
    const int t = next_item(pc, 0, count);
    if (t < 0) break;
    const Pair pr = load_pair(A, begin + t);
    int np, nc;
    init_poly_3d<P3, C3, BOX>(S[w], A, pr, np, nc);
    const int rc = preclip_3d(S[w], A, pr.a, pr.i, pr.u, &A.pairs[begin + t], np, nc, lc);
    int failed = 0;
    if (rc == 1) { defer_pair(A, begin + t); np = -1; }
    if (rc == 2) { failed = 1; atomicOr(&A.ctl->err, ERR_TOPOLOGY); }
    __syncwarp();
    CellState* c = &cells[t];
    if (np >= 0) park(&c->S, &S[w], kPolyBytes);
    if (lane == 0) { c->np = np; c->nc = nc; c->a = pr.a; c->i = pr.i; c->failed = failed; }
    __syncwarp();
  }
  flush_counters(A.ctl, st, lc, CNT_INIT);
}

// Round r of a phased wave (lists[r & 1] receives the pairs that still have a corner outside).  Round 0 tests every pair of
// the wave; round r > 0 the pairs that round r-1's k_ph_fix clipped -- it runs only if that kernel ran.  A negative list
// entry is a pair that left the path.
// MODE 0: the whole step.  Refined index: MODE 1 = the fast pass (batched tests only; a pair with a corner whose test needs the
// single-query path goes to the loose list, those corners marked ST_LOOSE), MODE 2 = the second pass over the loose list with
// the complete test code.  Both passes feed the same clip / done lists.
template <bool HV, int MODE>
__global__ void __launch_bounds__(kBlock, HV ? VD_PHV_BLOCKS_HV : VD_PHV_BLOCKS) k_ph_verify(ClipArgs A, CellState* __restrict__ cells, int* __restrict__ lists, int cap,
                                                     int* __restrict__ doneList, PhaseCtl* pc, int r, int tailPairs) {
  if (pc->mode != WAVE_PHASED) return;
  if (r > 0 && (int)pc->nClip[r - 1] <= tailPairs) return;
  int* looseList = lists + 3 * (int64_t)cap;
  const int* list = MODE == 2 ? looseList : (r > 0 ? lists + ((r - 1) & 1) * (int64_t)cap : nullptr);
  const int count = MODE == 2 ? (int)pc->nLoose[r] : (r > 0 ? (int)pc->nClip[r - 1] : (int)pc->count);
  if (count == 0) return;
  int* clipList = lists + (r & 1) * (int64_t)cap;
  const int slot = 4 + 4 * r + (MODE == 2 ? 1 : 0);
  __shared__ GridIndex g;
  __shared__ PolyT S[kWarpsPerBlock];
  if (threadIdx.x == 0) g = *A.grid;
  __syncthreads();
  const int w = (int)threadIdx.x / kLanes, lane = lane_id();
  QueryStats st = {0};
  LocalCnt lc = {0u, 0u, 0u, 0u, 0u, 0u};
  extra_cnt_reset();
  VD_WARP_BAR;
  for (;;) {
    const int t = next_item(pc, slot, count);
    if (t < 0) break;
    const int item = list ? list[t] : t;
    if (item < 0) continue;
    CellState* c = &cells[item];
    const int np = c->np, nc = c->nc;
    if (np < 0) continue;
    bool out = false, loose = false;
    if (!c->failed && nc > 0) {
      unpark(&S[w], &c->S, kTestBytes, bar, parity);
      bool deferred = false;
      const bool any = classify_unknown_3d<PolyT, HV, MODE == 1>(S[w], g, c->i, np, nc, st, &deferred);
      for (int k = lane; k < nc; k += kLanes) out |= (S[w].cstate[k] == ST_OUT);
      out = __any_sync(kFull, out);
      if (MODE == 1 && deferred) loose = true;
      if (any) {
#ifdef VD_NO_TMA
        copy_words(c->S.cnn, S[w].cnn, (nc * 4 + 15) & ~15);
        copy_words(c->S.cstate, S[w].cstate, (nc + 15) & ~15);
#else
        __syncwarp();
        if (lane == 0) {
          tma_store(c->S.cnn, S[w].cnn, (unsigned)((nc * 4 + 15) & ~15));
          tma_store(c->S.cstate, S[w].cstate, (unsigned)((nc + 15) & ~15));
          tma_store_commit();
          tma_store_wait_read();
        }
        __syncwarp();
#endif
      }
    }
    if (lane == 0) {
      if (MODE == 1 && loose) looseList[atomicAdd(&pc->nLoose[r], 1u)] = item;
      else if (out) clipList[atomicAdd(&pc->nClip[r], 1u)] = item;
      else doneList[atomicAdd(&pc->nDone, 1u)] = item;
    }
    __syncwarp();
  }
  flush_counters(A.ctl, st, lc, CNT_VERIFY);
}

// every corner known to be outside is clipped away (its search, its clip); the new corners wait for the next
// round of tests.  The list is rewritten in place: the slot, or -1 when the pair left the path.
// Runs when round r's tests left more than tailPairs pairs with a corner outside (fewer: k_ph_tail finishes them).
// MODE as in k_ph_verify: the fast pass (1) stops at a search that needs the single-query path -- the pair is parked as it is
// and its position in the clip list goes to the loose list --, the second pass (2) takes those pairs to the end of the step.
template <bool HV, int MODE>
__global__ void __launch_bounds__(kBlock, HV ? VD_PH_BLOCKS_HV : VD_PH_BLOCKS) k_ph_fix(ClipArgs A, CellState* __restrict__ cells, int* __restrict__ lists, int cap,
                                                     PhaseCtl* pc, int r, int tailPairs) {
  if (pc->mode != WAVE_PHASED || (int)pc->nClip[r] <= tailPairs) return;
  int* list = lists + (r & 1) * (int64_t)cap;
  int* looseList = lists + 3 * (int64_t)cap;
  const int count = MODE == 2 ? (int)pc->nLooseFix[r] : (int)pc->nClip[r];
  if (count == 0) return;
  const int64_t begin = (int64_t)pc->begin;
  const int tslot = 6 + 4 * r + (MODE == 2 ? 1 : 0);
  __shared__ GridIndex g;
  __shared__ PolyF S[kWarpsPerBlock];
  if (threadIdx.x == 0) g = *A.grid;
  __syncthreads();
  const int w = (int)threadIdx.x / kLanes, lane = lane_id();
  QueryStats st = {0};
  LocalCnt lc = {0u, 0u, 0u, 0u, 0u, 0u};
  extra_cnt_reset();
  VD_WARP_BAR;
  for (;;) {
    int t = next_item(pc, tslot, count);
    if (t < 0) break;
    if (MODE == 2) t = looseList[t];   // the pair's position in the clip list
    const int slot = list[t];
    CellState* c = &cells[slot];
    int np = c->np, nc = c->nc;
    const int i = c->i;
    unpark(&S[w], &c->S, kPolyBytes, bar, parity);
    int failed = 0;
    for (int guard = 0; guard < 4 * P3 && nc > 0; ++guard) {
      int s;
      const int p = select_out_3d(S[w], A, nc, s);
      if (p < 0) break;
      const int rc = clip_from_3d<P3, C3, HV, MODE == 1>(S[w], g, A, i, p, s, np, nc, st, lc);
      if (MODE == 1 && rc == 4) {   // this search is for the second pass; what was clipped so far stays
        if (lane == 0) looseList[atomicAdd(&pc->nLooseFix[r], 1u)] = t;
        break;
      }
      if (rc == 1) { defer_pair(A, begin + slot); np = -1; break; }
      if (rc) { failed = 1; atomicOr(&A.ctl->err, rc == 2 ? ERR_TOPOLOGY : ERR_NOCONVERGE); break; }
    }
    if (np >= 0) park(&c->S, &S[w], kPolyBytes);
    if (lane == 0) {
      c->np = np; c->nc = nc; c->failed = failed;
      list[t] = np >= 0 ? slot : -1;
    }
    __syncwarp();
  }
  flush_counters(A.ctl, st, lc, CNT_FIX);
}

// The last few pairs of a wave (a verify round left at most `tail_pairs` (65 536) pairs with a corner outside): tests and clips
// alternate inside one launch until every corner is in Omega_i -- Alg. 3's loop as it stands --
// instead of one round trip to the host and two nearly empty launches per remaining round.  Finished pairs join the
// done list.  The whole loop in one kernel is the instruction-fetch-bound form (header of this file); on a few
// thousand pairs that does not matter.
// A program without rounds (the default on tet meshes with the plain site index, where it is the fastest form: no parking between a
// pair's clips; init and finish stay kernels of their own -- fused into this one, its code no longer fits the instruction cache and the
// step takes 23.8 instead of 17.6 ms on C2) hands every pair of the wave to this kernel straight from k_ph_init.
// One launch after the program's rounds.  The rounds stop at the first round r whose tests leave at most tailPairs pairs with
// a corner outside: those pairs (tested, not clipped) are taken to completion here.  If every round ran its clips, the last
// round's pairs (clipped, not yet re-tested) are -- so a wave always ends, whatever the number of rounds in the program.
template <bool HV>
__global__ void __launch_bounds__(kBlock, VD_PH_TAIL_BLOCKS) k_ph_tail(ClipArgs A, CellState* __restrict__ cells, const int* __restrict__ lists, int cap,
                                                       int* __restrict__ doneList, PhaseCtl* pc, int rounds, int tailPairs) {
  if (pc->mode != WAVE_PHASED) return;
  int r = 0;
  while (r < rounds - 1 && (int)pc->nClip[r] > tailPairs) ++r;
  const int count = rounds == 0 ? (int)pc->count : (int)pc->nClip[r];   // a program without rounds: every pair of the wave, straight from k_ph_init
  if (count == 0) return;
  const int* list = rounds == 0 ? nullptr : lists + (r & 1) * (int64_t)cap;
  const int64_t begin = (int64_t)pc->begin;
  const int tslot = 3;   // (cursors 4 ..: four per round -- tests, their second pass, clips, their second pass)
  __shared__ GridIndex g;
  __shared__ PolyF S[kWarpsPerBlock];
  if (threadIdx.x == 0) g = *A.grid;
  __syncthreads();
  const int w = (int)threadIdx.x / kLanes, lane = lane_id();
  QueryStats st = {0};
  LocalCnt lc = {0u, 0u, 0u, 0u, 0u, 0u};
  extra_cnt_reset();
  VD_WARP_BAR;
  for (;;) {
    const int t = next_item(pc, tslot, count);
    if (t < 0) break;
    const int slot = list ? list[t] : t;
    if (slot < 0) continue;   // (the fix kernel marked a pair that left the path)
    CellState* c = &cells[slot];
    int np = c->np, nc = c->nc;
    if (np < 0) continue;     // (k_ph_init sent the pair to the large tier)
    const int i = c->i;
    int failed = c->failed;
    const bool work = !failed && nc > 0;   // (else: an empty or failed pair from k_ph_init, which stays parked as it is)
    if (work) unpark(&S[w], &c->S, kPolyBytes, bar, parity);
    for (int guard = 0; guard < 8 * P3 + 32 && nc > 0 && !failed; ++guard) {
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
    if (np >= 0 && work) park(&c->S, &S[w], kPolyBytes);
    if (lane == 0) {
      c->np = np; c->nc = nc; c->failed = failed;
      if (np >= 0) doneList[atomicAdd(&pc->nDone, 1u)] = slot;
    }
    __syncwarp();
  }
  flush_counters(A.ctl, st, lc, CNT_TAIL);
}

__global__ void __launch_bounds__(kBlock, 3) k_ph_finish(ClipArgs A, CellState* __restrict__ cells, const int* __restrict__ list, const PhaseCtl* pc,
                                                     int vchunk, int nchunk) {
  if (pc->mode != WAVE_PHASED) return;
  const int count = (int)pc->nDone;
  const int64_t begin = (int64_t)pc->begin;
  __shared__ PolyF S[kWarpsPerBlock];
  const int w = (int)threadIdx.x / kLanes;
  QueryStats st = {0};
  LocalCnt lc = {0u, 0u, 0u, 0u, 0u, 0u};
  extra_cnt_reset();
  VD_WARP_BAR;
  WarpPool wp = {0ull, 0ull, 0, 0, vchunk, nchunk};
  // uniform work per piece: a static stride instead of a ticket (one same-address atomic less per piece)
  const int stride = (int)gridDim.x * kWarpsPerBlock;
  for (int t = (int)blockIdx.x * kWarpsPerBlock + w; t < count; t += stride) {
    const int slot = list[t];
    const CellState* c = &cells[slot];
    unpark(&S[w], &c->S, kPolyBytes, bar, parity);
    finish_piece_3d(S[w], A, begin + slot, c->a, c->i, c->np, c->nc, S[w].u[0], S[w].u[1], S[w].u[2], c->failed != 0, lc, &wp);
    __syncwarp();
  }
  flush_counters(A.ctl, st, lc, CNT_FINISH);
}

// The step kernels of ONE wave program, enqueued without looking at the device: `rounds` rounds of {tests, then clips
// or -- for a short list -- the finishing kernel}, one more finishing launch for what the last round's clips left, and
// the finish kernel.  Every kernel decides from PhaseCtl whether it has work (a launch without work costs ~3 us); the
// wave's size, its lists and its counters never visit the host (the paper's host loop is P:L257, L325).
vd_status phase_buffers(vd_ctx* c, int64_t cap) {
  vd_status s;
  if ((s = ensure(c, c->phaseCells, sizeof(CellState) * (size_t)cap))) return s;
  return ensure(c, c->phaseLists, sizeof(PhaseCtl) + sizeof(int) * 4 * (size_t)cap);   // to verify / to clip, done, loose   // the control block first (8-byte members)
}

void enqueue_phased(vd_ctx* c, const ClipArgs& A, bool hv, int64_t cap, int rounds, int tailPairs) {
  CellState* cells = c->phaseCells.as<CellState>();
  PhaseCtl* pc = c->phaseLists.as<PhaseCtl>();
  int* lists = reinterpret_cast<int*>(pc + 1);
  int* done = lists + 2 * cap;
  cudaStream_t st = c->stream;
  const int grid = sm_count() * 4;
  const int icap = (int)cap;
  phase_mark(c, 0);
  if (c->kind == KIND_BOX_3D) VD_LAUNCH(k_ph_init<true>, grid, kBlock, 0, st)(A, cells, pc);
  else VD_LAUNCH(k_ph_init<false>, grid, kBlock, 0, st)(A, cells, pc);
  for (int r = 0; r < rounds; ++r) {
    // refined index: a fast pass without the single-query search code, then a second pass for what it left (MODE)
    phase_mark(c, 1);
    if (hv && VD_TWO_PASS) {
      VD_LAUNCH((k_ph_verify<true, 1>), grid, kBlock, 0, st)(A, cells, lists, icap, done, pc, r, tailPairs);
      VD_LAUNCH((k_ph_verify<true, 2>), grid, kBlock, 0, st)(A, cells, lists, icap, done, pc, r, tailPairs);
    } else if (hv) {
      VD_LAUNCH((k_ph_verify<true, 0>), grid, kBlock, 0, st)(A, cells, lists, icap, done, pc, r, tailPairs);
    } else {
      VD_LAUNCH((k_ph_verify<false, 0>), grid, kBlock, 0, st)(A, cells, lists, icap, done, pc, r, tailPairs);
    }
    phase_mark(c, 2);
    if (hv && VD_TWO_PASS) {
      VD_LAUNCH((k_ph_fix<true, 1>), grid, kBlock, 0, st)(A, cells, lists, icap, pc, r, tailPairs);
      VD_LAUNCH((k_ph_fix<true, 2>), grid, kBlock, 0, st)(A, cells, lists, icap, pc, r, tailPairs);
    } else if (hv) {
      VD_LAUNCH((k_ph_fix<true, 0>), grid, kBlock, 0, st)(A, cells, lists, icap, pc, r, tailPairs);
    } else {
      VD_LAUNCH((k_ph_fix<false, 0>), grid, kBlock, 0, st)(A, cells, lists, icap, pc, r, tailPairs);
    }
  }
  phase_mark(c, 4);
  if (hv) VD_LAUNCH(k_ph_tail<true>, grid, kBlock, 0, st)(A, cells, lists, icap, done, pc, rounds, tailPairs);
  else VD_LAUNCH(k_ph_tail<false>, grid, kBlock, 0, st)(A, cells, lists, icap, done, pc, rounds, tailPairs);
  // pool chunk per warp: ~1/32 of an even share of the pool, so that the slack (one open chunk per warp) stays small;
  // static stride over the grid: exactly the resident blocks (3 per SM), or the last third would run alone
  const int fgrid = sm_count() * 3;
  const int64_t warps = (int64_t)fgrid * kWarpsPerBlock;
  auto chunk_of = [&](int64_t poolCap) { const int64_t v = poolCap / (warps * 32); return (int)(v > 1024 ? 1024 : v); };   // small pools: piece by piece
  phase_mark(c, 3);
  VD_LAUNCH(k_ph_finish, fgrid, kBlock, 0, st)(A, cells, done, pc, chunk_of(c->vertCap), chunk_of(c->nbrCap));
  phase_mark(c, -1);
}

PhaseCtl* phase_ctl(vd_ctx* c, int64_t) { return c->phaseLists.as<PhaseCtl>(); }

}  // namespace VD_VARIANT
}  // namespace vd
