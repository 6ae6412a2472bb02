// vd_common.cuh -- shared types and warp helpers of the CUDA path (sm_100a).
// Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#ifndef VD_LANES
#define VD_LANES 32
#endif
namespace vd { extern unsigned long long g_launches; }   // kernels launched by this library (host counter)
#ifndef VD_LAUNCH
#define VD_LAUNCH(kernel, grid, block, smem, stream) ++vd::g_launches, kernel<<<(grid), (block), (smem), (stream)>>>
#endif

namespace vd {

constexpr int kLanes = VD_LANES;
constexpr unsigned kFull = 0xffffffffu;
constexpr int kWarpsPerBlock = 8;
constexpr int kBlock = kWarpsPerBlock * kLanes;

enum { KIND_TRI_2D = 0, KIND_TRI_SURFACE = 1, KIND_TET_3D = 2, KIND_BOX_2D = 3, KIND_BOX_3D = 4 };

// device-side sticky error bits (read once at the end of vd_compute)
enum {
  ERR_PAIR_CAP = 1,      // pair list / visited set full
  ERR_VERT_CAP = 2,      // corner pool full
  ERR_NBR_CAP = 4,       // face-flag pool full
  ERR_PIECE_CAP = 8,     // a piece outgrew the large-capacity path
  ERR_NOCONVERGE = 16,   // iteration cap
  ERR_TOPOLOGY = 32,     // clip produced a non-simple boundary loop
  ERR_INPUT = 64,        // zero-measure simplex / non-manifold face / non-finite coordinate
  ERR_DUPLICATE = 128,   // two sites with equal coordinates (found inside a bucket of the site index, S1)
  ERR_WEIGHT = 256       // eta below the largest weight, or a non-finite weight (vd_create_weighted)
};

// Site index: uniform grid over the sites' bounding box; sites sorted by cell key so
// that a run of cells along x is one contiguous range.
struct GridIndex {
  double lo[3];
  double h[3];      // cell size (0 on a degenerate axis)
  double inv_h[3];  // 1/h (0 on a degenerate axis)
  double hi[3];
  int G[3];
  int n;
  const int* __restrict__ cellStart;      // [G0*G1*G2 + 1]
  const double4* __restrict__ sites;      // sorted; w = original id (as int bits)
  // second level (clustered sites): a cell holding more than kHeavy sites carries its own K^3 sub-grid;
  // its sites are sorted by sub-cell, subStart holds absolute first-site indices (K^3 + 1 entries)
  const int* __restrict__ heavyPrefix;    // [G0*G1*G2 + 1] number of refined cells below a cell index (null: no second level)
  const int* __restrict__ subOff;         // [G0*G1*G2] (K << 26) | offset into subStart, or -1
  const int* __restrict__ subStart;
  int countAlg;                           // vd_options.count_alg: queries also count D_alg (measurement runs)
  // S1b: delta_i = half the distance from v_i to its nearest other site, for the step-out of section VI-A
  const double* __restrict__ delta;       // [n] by original site id, or null (vd_options.step_out = 0)
  int stepMode;                           // 1: lambda = 2, 3, 4, ...; 2: lambda doubles
  // Power diagrams of 3-D sites (vd_create_weighted): the lifted sites p_i = (v_i, sqrt(eta - w_i)) in R^4 are
  // seen from the domain at height 0, so every squared distance to site i is |x - v_i|^2 + (eta - w_i).  The additive
  // terms, by sorted position and by original site id; null for ordinary (and for lifted 2-D) sites.  They are >= 0, so the
  // grid's plain box distances stay lower bounds.
  const double* __restrict__ sitesW;
  const double* __restrict__ siteWid;
  // fp32 filter (vd_options.fp32_filter; the paper's GPU runs are fp32): the sorted sites once more as 16-byte
  // float4 records (x, y, z, id bits), and the largest coordinate magnitude of the grid box (for the error bound)
  const float4* __restrict__ sites32;
  double f32M;
};

// The optional features of a query (weighted sites, step-out, D_alg counting) behind three predicates: the kernels exist in
// a lean form (EXT = false: the predicates are compile-time false, the code behind them is gone) and a full form -- the
// clip kernels are bound by instruction fetch, and every resident-but-unused code path costs them.
#ifndef VD_EXT
#define VD_EXT 1
#endif
__device__ __forceinline__ bool has_weights(const GridIndex& g) { return VD_EXT && g.sitesW != nullptr; }
__device__ __forceinline__ bool has_step_out(const GridIndex& g) { return VD_EXT && g.stepMode != 0; }
__device__ __forceinline__ bool counts_alg(const GridIndex& g) { return VD_EXT && g.countAlg != 0; }
__device__ __forceinline__ bool has_f32(const GridIndex& g) { return VD_EXT && g.sites32 != nullptr; }

// fp32 filter: a candidate whose squared distance to q, evaluated in fp32 from the float-rounded operands, exceeds this
// threshold cannot be closer than `best` in exact arithmetic, so its fp64 record is never loaded.  Error budget: q and the
// site are rounded to float (2^-24 relative each, coordinates up to M), the difference is rounded once more:
// |dx_f - dx| <= delta = 2.5e-7 M per coordinate; then |d2_f - d2| <= 2 sqrt(3) delta |d| + 3 delta^2 plus the rounding of
// three products and two sums (< 4e-6 relative).  With |d| <= sqrt(best) for every candidate that matters:
__device__ __forceinline__ float f32_threshold(double best, double M) {
  if (!(best < 1e300)) return __int_as_float(0x7f800000);
  const double delta = 2.5e-7 * M;
  return __double2float_ru((best + 3.5 * sqrt(best) * delta + 3.0 * delta * delta) * (1.0 + 4e-6));
}
__device__ __forceinline__ double f32_magnitude(const GridIndex& g, double qx, double qy, double qz) {
  return fmax(fmax(g.f32M, fabs(qx)), fmax(fabs(qy), fabs(qz)));
}
__device__ __forceinline__ double site_w(const GridIndex& g, int id) { return has_weights(g) ? __ldg(&g.siteWid[id]) : 0.0; }

#ifndef VD_HEAVY
#define VD_HEAVY 128   // measured on C3 (round 2): 32 sites 316 ms, 64: 302, 128: 294, 256: 301, 512: 333
#endif
constexpr int kHeavy = VD_HEAVY;                // sites per cell above which the cell is refined (one warp round)

// One unit of work: simplex a, site i, and a witness point w in T_a ∩ Ω_i
// (DESIGN.md "witness"): the start p_s of virtual edges instead of v_i (Alg. 3 line 3).
constexpr int kPairW = 7;

struct Pair {
  int a, i;
  double wx, wy, wz;
  // The tuple (u, f) of P:L211 in the form the clip needs: u = the site whose piece P_{a,u} discovered this pair
  // through its face f on B_ui, w[] = the positive flags of the faces of P_{a,u} adjacent to f.  -1: none (a seed).
  int u;
  int w[kPairW];
};
static_assert(sizeof(Pair) == 64, "one pair per 64 bytes");

// Per-pair output record.
struct Piece {
  int site, simplex;
  int nverts, nnbr;
  int64_t vbase;   // first corner in the corner pool
  int64_t nbase;   // first entry in the face-flag pool
  double measure;
  double mx, my, mz;  // first moment (measure * centroid)
};

struct Counters {
  unsigned long long pairs, pieces, queries, dist_evals, search_iters, clips, overflow_pairs, rows;
  unsigned long long search_evals, pre_clips;   // distance evaluations inside bisector searches; clips by nearest-site bisectors (U19)
  unsigned long long clip_corners, new_corners, fan_simplices, alg_evals, step_probes, f32_survivors;
};

// which kernel a counter block belongs to (vd_get_phase_counters): the step kernels of the phased schedule, the rest
enum { CNT_INIT = 0, CNT_VERIFY = 1, CNT_FIX = 2, CNT_FINISH = 3, CNT_TAIL = 4, CNT_OTHER = 5, kCntKinds = 6 };

__device__ __forceinline__ int lane_id() { return (int)(threadIdx.x % kLanes); }

template <typename T>
__device__ __forceinline__ T shfl(T v, int src) { return __shfl_sync(kFull, v, src); }

__device__ __forceinline__ bool closer(double d2, int id, double best, int bestId) {
  return d2 < best || (d2 == best && id < bestId);
}

// Warp argmin of (d2, id) with the tie rule "lowest id" (reading U5); result uniform.
__device__ __forceinline__ void warp_argmin(double& d2, int& id) {
  // (three __reduce_min_sync over the words of the bit pattern were measured slower than this butterfly)
#pragma unroll
  for (int off = kLanes / 2; off > 0; off >>= 1) {
    const double od = __shfl_xor_sync(kFull, d2, off);
    const int oi = __shfl_xor_sync(kFull, id, off);
    if (closer(od, oi, d2, id)) { d2 = od; id = oi; }
  }
}

__device__ __forceinline__ int warp_sum(int v) {
#pragma unroll
  for (int off = kLanes / 2; off > 0; off >>= 1) v += __shfl_xor_sync(kFull, v, off);
  return v;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int off = kLanes / 2; off > 0; off >>= 1) v += __shfl_xor_sync(kFull, v, off);
  return v;
}

// inclusive prefix sum over the lanes
__device__ __forceinline__ int warp_incl_scan(int v) {
  const int lane = lane_id();
#pragma unroll
  for (int off = 1; off < kLanes; off <<= 1) {
    const int o = __shfl_up_sync(kFull, v, off);
    if (lane >= off) v += o;
  }
  return v;
}

// exclusive prefix of a per-lane flag, and the total
__device__ __forceinline__ int warp_rank(bool flag, int& total) {
  const unsigned m = __ballot_sync(kFull, flag);
  total = __popc(m);
  return __popc(m & ((1u << lane_id()) - 1u));
}

__device__ __forceinline__ uint64_t pair_key(int a, int i) {
  return (((uint64_t)(uint32_t)a) << 32 | (uint32_t)i) + 1ull;   // 0 = empty slot
}

__device__ __forceinline__ uint64_t hash64(uint64_t x) {
  x ^= x >> 33; x *= 0xff51afd7ed558ccdull; x ^= x >> 33; x *= 0xc4ceb9fe1a85ec53ull; x ^= x >> 33;
  return x;
}

// "label it in atomic" (Alg. 4 line 5/13): true iff (a, i) was not yet labelled.
__device__ __forceinline__ bool visit(unsigned long long* table, uint64_t mask, int a, int i) {
  const unsigned long long key = pair_key(a, i);
  uint64_t h = hash64(key) & mask;
  for (uint64_t probe = 0; probe <= mask; ++probe) {
    const unsigned long long cur = atomicCAS(&table[h], 0ull, key);
    if (cur == 0ull) return true;
    if (cur == key) return false;
    h = (h + 1) & mask;
  }
  return false;
}

}  // namespace vd
