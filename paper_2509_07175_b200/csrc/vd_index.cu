// vd_index.cu -- S1: the site index ("build a structure S of V", line 1 of Alg. 2/4/5, P:L180/L250/L301;
// grid structure P:L377-383).  Bounding box -> cell key per site -> histogram + exclusive scan (bucket starts) -> refined
// cells planned -> ONE stable radix sort by (cell, sub-cell) key -> sites gathered in that order as 32-byte records ->
// duplicate check.  Plus S1b (k_delta), the S2 query as a kernel of its own (vd_nearest, and the per-mesh-vertex nearest
// site used by S3) and its no-allocation variant (vd_nearest_static).
#include <math.h>

#include "vd_internal.h"
#include "vd_nearest.cuh"
#include "vd_scan.cuh"

namespace vd {

constexpr int kBBoxBlocks = 512;   // partial boxes (a buffer size; the launch takes at most this many blocks)

__global__ void __launch_bounds__(kBlock) k_bbox_partial(const double* __restrict__ sites, int64_t n, double* __restrict__ part) {
  double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const double v = sites[i * 3 + a];
      lo[a] = fmin(lo[a], v);
      hi[a] = fmax(hi[a], v);
    }
  }
  __shared__ double sm[kWarpsPerBlock][6];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    for (int off = kLanes / 2; off > 0; off >>= 1) {
      lo[a] = fmin(lo[a], __shfl_xor_sync(kFull, lo[a], off));
      hi[a] = fmax(hi[a], __shfl_xor_sync(kFull, hi[a], off));
    }
  }
  const int w = (int)threadIdx.x / kLanes;
  if (lane_id() == 0) {
    for (int a = 0; a < 3; ++a) { sm[w][a] = lo[a]; sm[w][3 + a] = hi[a]; }
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int k = 1; k < (int)blockDim.x / kLanes; ++k)
      for (int a = 0; a < 3; ++a) {
        sm[0][a] = fmin(sm[0][a], sm[k][a]);
        sm[0][3 + a] = fmax(sm[0][3 + a], sm[k][3 + a]);
      }
    for (int a = 0; a < 6; ++a) part[blockIdx.x * 6 + a] = sm[0][a];
  }
}

// One thread: final box, grid resolution ("each grid cell contains, on average, 2~3 / 3~4 sites":
// average over all cells of the sites' box -- reading U9), header written to device memory.
__global__ void k_grid_params(const double* __restrict__ part, int nparts, int64_t n, double density, int64_t gridCap,
                              const int* cellStart, const double4* sorted, int countAlg, const double* delta, int stepMode,
                              const double* sitesW, const double* siteWid, const float4* sites32, GridIndex* g, unsigned int* err) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
  for (int k = 0; k < nparts; ++k)
    for (int a = 0; a < 3; ++a) {
      lo[a] = fmin(lo[a], part[k * 6 + a]);
      hi[a] = fmax(hi[a], part[k * 6 + 3 + a]);
    }
  double ext[3], vol = 1.0;
  int nd = 0;
  for (int a = 0; a < 3; ++a) {
    ext[a] = hi[a] - lo[a];
    if (!(ext[a] == ext[a]) || ext[a] > 1e300) atomicOr(err, ERR_INPUT);
    if (ext[a] > 0) { vol *= ext[a]; ++nd; }
  }
  double target = (double)n / density;
  if (target < 1.0) target = 1.0;
  double h = nd > 0 ? pow(vol / target, 1.0 / nd) : 1.0;
  int G[3];
  for (int it = 0; it < 64; ++it) {
    double prod = 1.0;
    for (int a = 0; a < 3; ++a) {
      G[a] = ext[a] > 0 ? (int)fmin(fmax(ceil(ext[a] / h), 1.0), 2047.0) : 1;
      prod *= G[a];
    }
    if (prod <= (double)gridCap) break;
    h *= 1.1;
  }
  GridIndex out;
  for (int a = 0; a < 3; ++a) {
    out.lo[a] = lo[a];
    out.hi[a] = hi[a];
    out.G[a] = G[a];
    out.h[a] = ext[a] > 0 ? ext[a] / G[a] : 0.0;
    out.inv_h[a] = ext[a] > 0 ? G[a] / ext[a] : 0.0;
  }
  out.n = (int)n;
  out.cellStart = cellStart;
  out.sites = sorted;
  out.heavyPrefix = nullptr;
  out.subOff = nullptr;
  out.subStart = nullptr;
  out.countAlg = countAlg;
  out.delta = delta;
  out.stepMode = stepMode;
  out.sitesW = sitesW;
  out.siteWid = siteWid;
  out.sites32 = sites32;
  out.f32M = 0.0;
  for (int a = 0; a < 3; ++a) out.f32M = fmax(out.f32M, fmax(fabs(lo[a]), fabs(hi[a])));
  *g = out;
}

__global__ void __launch_bounds__(kBlock) k_cell_count(const double* __restrict__ sites, int64_t n, const GridIndex* __restrict__ gp,
                                                        int* __restrict__ cellOf, int* __restrict__ cellFill) {
  const GridIndex g = *gp;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const int cx = cell_of(g, 0, sites[i * 3 + 0]), cy = cell_of(g, 1, sites[i * 3 + 1]), cz = cell_of(g, 2, sites[i * 3 + 2]);
    const int c = (cz * g.G[1] + cy) * g.G[0] + cx;
    cellOf[i] = c;
    atomicAdd(&cellFill[c], 1);
  }
}

// ---- second level: cells with more than kHeavy sites get a K^3 sub-grid (clustered site sets: a uniform
// grid at the paper's density leaves thousands of sites in one cell).  K is chosen so that a sub-cell holds
// `density` sites on average; the cell's sites are re-sorted by sub-cell key.
__device__ __forceinline__ int sub_k(int cnt, double density, int nd) {
  const double t = (double)cnt / density;
  int K = (int)ceil(nd == 3 ? cbrt(t) : (nd == 2 ? sqrt(t) : t));
  return min(max(K, 2), 31);
}

__global__ void __launch_bounds__(kBlock) k_sub_plan(const GridIndex* __restrict__ gp, double density, int64_t gridCap,
                                                      int* __restrict__ heavyFlag, int* __restrict__ need) {
  const GridIndex g = *gp;
  const int64_t G = (int64_t)g.G[0] * g.G[1] * g.G[2];
  const int nd = (g.h[0] > 0) + (g.h[1] > 0) + (g.h[2] > 0);
  for (int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; c <= gridCap; c += (int64_t)gridDim.x * blockDim.x) {
    int hv = 0, nd3 = 0;
    if (c < G) {
      const int cnt = g.cellStart[c + 1] - g.cellStart[c];
      if (cnt > kHeavy && nd > 0) {
        const int K = sub_k(cnt, density, nd);
        hv = 1;
        nd3 = (g.h[0] > 0 ? K : 1) * (g.h[1] > 0 ? K : 1) * (g.h[2] > 0 ? K : 1) + 1;
      }
    }
    heavyFlag[c] = hv;
    need[c] = nd3;
  }
}

__global__ void __launch_bounds__(kBlock) k_sub_pack(const GridIndex* __restrict__ gp, double density, const int* __restrict__ offRaw,
                                                      int64_t subCap, int* __restrict__ subOff) {
  const GridIndex g = *gp;
  const int64_t G = (int64_t)g.G[0] * g.G[1] * g.G[2];
  const int nd = (g.h[0] > 0) + (g.h[1] > 0) + (g.h[2] > 0);
  for (int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; c < G; c += (int64_t)gridDim.x * blockDim.x) {
    const int cnt = g.cellStart[c + 1] - g.cellStart[c];
    int v = -1;
    if (cnt > kHeavy && nd > 0 && (int64_t)offRaw[c + 1] <= subCap) v = (sub_k(cnt, density, nd) << 26) | offRaw[c];
    subOff[c] = v;
  }
}

__device__ __forceinline__ int sub_key(const GridIndex& g, int c, int K, double x, double y, double z) {
  const int cx = c % g.G[0], cy = (c / g.G[0]) % g.G[1], cz = c / (g.G[0] * g.G[1]);
  const int Kx = g.h[0] > 0 ? K : 1, Ky = g.h[1] > 0 ? K : 1, Kz = g.h[2] > 0 ? K : 1;
  const int kx = min(max((int)floor((x - (g.lo[0] + cx * g.h[0])) * (Kx * g.inv_h[0])), 0), Kx - 1);
  const int ky = min(max((int)floor((y - (g.lo[1] + cy * g.h[1])) * (Ky * g.inv_h[1])), 0), Ky - 1);
  const int kz = min(max((int)floor((z - (g.lo[2] + cz * g.h[2])) * (Kz * g.inv_h[2])), 0), Kz - 1);
  return (kz * Ky + ky) * Kx + kx;
}

// ---- sort: ONE stable radix sort of the sites by their finest bucket ("Morton/cell-key radix sort + counting-sort bucketing",
// BASELINE north_star (1)).  The key of site i is c + subOffRaw[c] + k: c its top cell (row-major: a run of cells along x stays
// one contiguous range), k its sub-cell inside a refined cell (0 in a plain one); subOffRaw[c] = the sub-cells of all refined
// cells before c, so the key is monotone in (c, k).  Input order is the site id and the sort is stable: inside a bucket the
// sites end up in ascending id, the same in every run (the first build scattered through atomic cursors: arrival order).
__global__ void __launch_bounds__(kBlock) k_site_keys(const GridIndex* __restrict__ gp, const double* __restrict__ sites, int64_t n,
                                                       const int* __restrict__ cellOf, const int* __restrict__ subOff, const int* __restrict__ subOffRaw,
                                                       unsigned* __restrict__ key, int* __restrict__ val, int* __restrict__ subCount) {
  const GridIndex g = *gp;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const int c = cellOf[i];
    const int so = subOff[c];
    int k = 0;
    if (so >= 0) {
      k = sub_key(g, c, so >> 26, sites[i * 3 + 0], sites[i * 3 + 1], sites[i * 3 + 2]);
      atomicAdd(&subCount[(so & 0x3ffffff) + k], 1);   // (a count: the same whatever the arrival order)
    }
    key[i] = (unsigned)(c + subOffRaw[c] + k);
    val[i] = (int)i;
  }
}

// LSD radix sort, up to 11 bits per pass (22-bit keys -- two million sites -- take two passes), one WARP per segment of kSortSeg consecutive elements (stable: segments in order, chunks of
// 32 in order, lanes in order).  Pass = histogram per (digit, segment) -> exclusive scan in digit-major order -> scatter.
constexpr int kSortSeg = 2048;
constexpr int kSortWarps = 4, kSortDigits = 2048;   // per block: 4 warps x 2048 counters = 32 KB of shared memory

__device__ __forceinline__ unsigned match_digit(unsigned active, unsigned d) { return __match_any_sync(active, d); }

__global__ void __launch_bounds__(kSortWarps * kLanes) k_radix_hist(const unsigned* __restrict__ key, int64_t n, int shift, int dbits, int nseg, int* __restrict__ hist) {
  __shared__ int cnt[kSortWarps][kSortDigits];
  const int nd = 1 << dbits;
  const unsigned dmask = (unsigned)nd - 1u;
  const int w = (int)threadIdx.x / kLanes, lane = lane_id();
  const int64_t seg = (int64_t)blockIdx.x * kSortWarps + w;
  for (int d = lane; d < nd; d += kLanes) cnt[w][d] = 0;
  __syncwarp();
  if (seg < nseg) {
    const int64_t b = seg * kSortSeg, e = b + kSortSeg < n ? b + kSortSeg : n;
    for (int64_t p0 = b; p0 < e; p0 += kLanes) {
      const int64_t p = p0 + lane;
      const unsigned active = __ballot_sync(kFull, p < e);
      if (p < e) {
        const unsigned d = (key[p] >> shift) & dmask;
        const unsigned m = match_digit(active, d);
        if ((int)(__ffs((int)m) - 1) == lane) cnt[w][d] += __popc(m);   // one lane per distinct digit
      }
      __syncwarp();
    }
    for (int d = lane; d < nd; d += kLanes) hist[(int64_t)d * nseg + seg] = cnt[w][d];
  }
}

__global__ void __launch_bounds__(kSortWarps * kLanes) k_radix_scatter(const unsigned* __restrict__ key, const int* __restrict__ val, int64_t n, int shift, int dbits, int nseg,
                                                           const int* __restrict__ scanned, unsigned* __restrict__ keyOut, int* __restrict__ valOut) {
  __shared__ int off[kSortWarps][kSortDigits];
  const int nd = 1 << dbits;
  const unsigned dmask = (unsigned)nd - 1u;
  const int w = (int)threadIdx.x / kLanes, lane = lane_id();
  const int64_t seg = (int64_t)blockIdx.x * kSortWarps + w;
  if (seg >= nseg) return;
  for (int d = lane; d < nd; d += kLanes) off[w][d] = scanned[(int64_t)d * nseg + seg];
  __syncwarp();
  const int64_t b = seg * kSortSeg, e = b + kSortSeg < n ? b + kSortSeg : n;
  for (int64_t p0 = b; p0 < e; p0 += kLanes) {
    const int64_t p = p0 + lane;
    const unsigned active = __ballot_sync(kFull, p < e);
    unsigned k = 0, d = 0, m = 0;
    int v = 0, dst = 0;
    if (p < e) {
      k = key[p]; v = val[p];
      d = (k >> shift) & dmask;
      m = match_digit(active, d);
      dst = off[w][d] + __popc(m & ((1u << lane) - 1u));   // earlier lanes with the same digit go first
    }
    __syncwarp();
    if (p < e && (int)(__ffs((int)m) - 1) == lane) off[w][d] += __popc(m);
    __syncwarp();
    if (p < e) { keyOut[dst] = k; valOut[dst] = v; }
  }
}

__global__ void __launch_bounds__(kBlock) k_gather_sorted(const double* __restrict__ sites, const int* __restrict__ order, int64_t n,
                                                           double4* __restrict__ sorted, float4* __restrict__ sorted32) {
  for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
    const int i = order[p];
    const double x = sites[(int64_t)i * 3 + 0], y = sites[(int64_t)i * 3 + 1], z = sites[(int64_t)i * 3 + 2];
    sorted[p] = make_double4(x, y, z, __longlong_as_double((long long)i));
    if (sorted32) sorted32[p] = make_float4((float)x, (float)y, (float)z, __int_as_float(i));   // fp32 filter records
  }
}

// subScan (exclusive scan of the sub-cell counts, all refined cells concatenated) -> absolute start indices
__global__ void __launch_bounds__(kBlock) k_sub_finalize(const GridIndex* __restrict__ gp, const int* __restrict__ subOff,
                                                          const int* __restrict__ subScan, int* __restrict__ subStart) {
  const GridIndex g = *gp;
  const int64_t G = (int64_t)g.G[0] * g.G[1] * g.G[2];
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / kLanes;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) / kLanes;
  for (int64_t c = warp; c < G; c += nwarps) {
    const int so = subOff[c];
    if (so < 0) continue;
    const int K = so >> 26, off = so & 0x3ffffff;
    const int cells = (g.h[0] > 0 ? K : 1) * (g.h[1] > 0 ? K : 1) * (g.h[2] > 0 ? K : 1);
    const int base = subScan[off], start = g.cellStart[c];
    __syncwarp();   // every lane holds the base before entry 0 is rewritten in place
    for (int k = lane_id(); k <= cells; k += kLanes) subStart[off + k] = start + subScan[off + k] - base;
  }
}

__global__ void k_grid_finish(GridIndex* g, const double4* sorted2, const int* heavyPrefix, const int* subOff, const int* subStart,
                              unsigned int* nHeavy) {
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    *nHeavy = (unsigned int)heavyPrefix[(int64_t)g->G[0] * g->G[1] * g->G[2]];
    g->sites = sorted2;
    g->heavyPrefix = heavyPrefix;
    g->subOff = subOff;
    g->subStart = subStart;
  }
}

// Power diagrams of 3-D sites: the additive term of every site, in the order of the finished index
__global__ void __launch_bounds__(kBlock) k_gather_weights(const GridIndex* __restrict__ gp, int64_t n, const double* __restrict__ byId,
                                                            double* __restrict__ sortedW) {
  const double4* sites = gp->sites;
  for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x)
    sortedW[p] = byId[(int)(__double_as_longlong(sites[p].w) & 0x7fffffff)];
}

// Duplicate sites (reading U14: VD_E_INPUT): equal coordinates mean equal cell and sub-cell keys, so the two sites sit
// in the same finest bucket of the finished index.  One thread per sorted position compares with the rest of its bucket.
__global__ void __launch_bounds__(kBlock) k_find_duplicates(const GridIndex* __restrict__ gp, int64_t n, unsigned int* err) {
  const GridIndex g = *gp;
  for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < n; p += (int64_t)gridDim.x * blockDim.x) {
    const double4 s = g.sites[p];
    const int cx = cell_of(g, 0, s.x), cy = cell_of(g, 1, s.y), cz = cell_of(g, 2, s.z);
    const int c = (cz * g.G[1] + cy) * g.G[0] + cx;
    int end = g.cellStart[c + 1];
    const int so = g.subOff ? g.subOff[c] : -1;
    if (so >= 0) end = g.subStart[(so & 0x3ffffff) + sub_key(g, c, so >> 26, s.x, s.y, s.z) + 1];
    for (int64_t q = p + 1; q < end; ++q) {
      const double4 t = g.sites[q];
      if (t.x == s.x && t.y == s.y && t.z == s.z) { atomicOr(err, ERR_DUPLICATE); break; }
    }
  }
}

// S2 as a kernel: one warp per query point.
__global__ void __launch_bounds__(kBlock) k_nearest_points(const GridIndex* __restrict__ gp, const double* __restrict__ q3, int64_t nq,
                                                            int* __restrict__ out, Counters* cnt) {
  const GridIndex g = *gp;
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / kLanes;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) / kLanes;
  QueryStats st = {0};
  extra_cnt_reset();
  for (int64_t q = warp; q < nq; q += nwarps) {
    double best = 2e300;
    int bestId = 0x7fffffff;
    nearest<true>(g, q3[q * 3 + 0], q3[q * 3 + 1], q3[q * 3 + 2], best, bestId, st);
    if (lane_id() == 0) out[q] = bestId;
  }
  __syncwarp();
  if (lane_id() == 0 && cnt) {
    atomicAdd(&cnt->queries, (unsigned long long)warp_stats().queries);
    atomicAdd(&cnt->dist_evals, (unsigned long long)warp_stats().dist_evals);
  }
}

// S1b: delta_i = || N_i - v_i || / 2, N_i the site nearest to v_i other than v_i itself -- one warp per site, the
// nearest-site query of S2 with the site's own record skipped.  The ball (v_i, delta_i) lies inside Omega_i; the step-out of
// section VI-A advances in multiples of it.
__global__ void __launch_bounds__(kBlock) k_delta(const GridIndex* __restrict__ gp, const double* __restrict__ sites3, int64_t n,
                                                   double* __restrict__ delta, Counters* cnt) {
  const GridIndex g = *gp;
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / kLanes;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) / kLanes;
  QueryStats st = {0};
  extra_cnt_reset();
  for (int64_t i = warp; i < n; i += nwarps) {
    double best = 2e300;
    int bestId = 0x7fffffff;
    st.skip = (int)i;
    nearest<true, true>(g, sites3[i * 3 + 0], sites3[i * 3 + 1], sites3[i * 3 + 2], best, bestId, st);
    if (lane_id() == 0) delta[i] = best < 1e300 ? 0.5 * sqrt(best) : 1e300;   // n = 1: no other site
  }
  __syncwarp();
  if (lane_id() == 0 && cnt) {
    atomicAdd(&cnt->queries, (unsigned long long)warp_stats().queries);
    atomicAdd(&cnt->dist_evals, (unsigned long long)warp_stats().dist_evals);
  }
}

static int grid_for(int64_t items, int perBlock) {
  int64_t b = (items + perBlock - 1) / perBlock;
  const int64_t cap = sm_count() * 16;
  if (b > cap) b = cap;
  if (b < 1) b = 1;
  return (int)b;
}

vd_status stage_index(vd_ctx* c) {
  const int64_t n = c->n;
  const double density = c->opt.grid_density > 0 ? c->opt.grid_density : 2.0;
  const int64_t gridCap = (int64_t)((double)n / density) * 2 + 64;
  c->gridCap = gridCap;
  vd_status s;
  if ((s = ensure(c, c->grid, sizeof(GridIndex)))) return s;
  if ((s = ensure(c, c->bbox, sizeof(double) * 6 * kBBoxBlocks))) return s;
  if ((s = ensure(c, c->cellOf, sizeof(int) * n))) return s;
  if ((s = ensure(c, c->cellStart, sizeof(int) * (gridCap + 2)))) return s;
  if ((s = ensure(c, c->cellFill, sizeof(int) * (gridCap + 2)))) return s;
  if ((s = ensure(c, c->sorted2, sizeof(double4) * n))) return s;
  if ((s = ensure(c, c->scanTmp, sizeof(int64_t) * scan_scratch_elems(n > gridCap ? n : gridCap) * 2))) return s;
  if ((s = ensure(c, c->control, sizeof(Control)))) return s;
  const int stepMode = c->opt.step_out > 0 ? (c->opt.step_out > 2 ? 2 : c->opt.step_out) : 0;
  if (stepMode && (s = ensure(c, c->delta, sizeof(double) * n))) return s;
  const bool lifted4 = c->weighted && c->dim == 3;   // power diagram of 3-D sites: additive terms travel with the sorted records
  if (lifted4 && (s = ensure(c, c->sortedW, sizeof(double) * n))) return s;
  const bool f32 = c->opt.fp32_filter > 0 && !lifted4;
  if (f32 && (s = ensure(c, c->sorted32, sizeof(float4) * n))) return s;
  cudaStream_t st = c->stream;
  const int nb = grid_for(n, kBlock) < kBBoxBlocks ? grid_for(n, kBlock) : kBBoxBlocks;
  VD_LAUNCH(k_bbox_partial, nb, kBlock, 0, st)(c->sites.as<double>(), n, c->bbox.as<double>());
  VD_LAUNCH(k_grid_params, 1, 1, 0, st)(c->bbox.as<double>(), nb, n, density, gridCap, c->cellStart.as<int>(),
                                         c->sorted2.as<double4>(), c->opt.count_alg > 1 ? 1 : 0,
                                         stepMode ? c->delta.as<double>() : nullptr, stepMode,
                                         lifted4 ? c->sortedW.as<double>() : nullptr, lifted4 ? c->siteW.as<double>() : nullptr,
                                         f32 ? c->sorted32.as<float4>() : nullptr, c->grid.as<GridIndex>(),
                                         &c->control.as<Control>()->err);
  cudaMemsetAsync(c->cellFill.p, 0, sizeof(int) * (gridCap + 2), st);
  VD_LAUNCH(k_cell_count, grid_for(n, kBlock), kBlock, 0, st)(c->sites.as<double>(), n, c->grid.as<GridIndex>(), c->cellOf.as<int>(),
                                                              c->cellFill.as<int>());
  exclusive_scan<int, int>(c->cellFill.as<int>(), gridCap + 1, c->cellStart.as<int>(), c->scanTmp.as<int>(), st);
  // second level
  const int64_t subCap = (int64_t)(4.0 * (double)n / density) + gridCap + 64;
  c->subCap = subCap;
  if ((s = ensure(c, c->heavyFlag, sizeof(int) * (gridCap + 2)))) return s;
  if ((s = ensure(c, c->heavyPrefix, sizeof(int) * (gridCap + 3)))) return s;
  if ((s = ensure(c, c->subNeed, sizeof(int) * (gridCap + 2)))) return s;
  if ((s = ensure(c, c->subOffRaw, sizeof(int) * (gridCap + 3)))) return s;
  if ((s = ensure(c, c->subOff, sizeof(int) * (gridCap + 2)))) return s;
  if ((s = ensure(c, c->subCount, sizeof(int) * (subCap + 2)))) return s;
  if ((s = ensure(c, c->subStart, sizeof(int) * (subCap + 3)))) return s;
  if ((s = ensure(c, c->scanTmp, sizeof(int64_t) * scan_scratch_elems(subCap > n ? subCap : n) * 2))) return s;
  GridIndex* gp = c->grid.as<GridIndex>();
  const int gb = grid_for(gridCap + 1, kBlock);
  VD_LAUNCH(k_sub_plan, gb, kBlock, 0, st)(gp, density, gridCap, c->heavyFlag.as<int>(), c->subNeed.as<int>());
  exclusive_scan<int, int>(c->heavyFlag.as<int>(), gridCap + 1, c->heavyPrefix.as<int>(), c->scanTmp.as<int>(), st);
  exclusive_scan<int, int>(c->subNeed.as<int>(), gridCap + 1, c->subOffRaw.as<int>(), c->scanTmp.as<int>(), st);
  VD_LAUNCH(k_sub_pack, gb, kBlock, 0, st)(gp, density, c->subOffRaw.as<int>(), subCap, c->subOff.as<int>());
  cudaMemsetAsync(c->subCount.p, 0, sizeof(int) * (subCap + 2), st);
  // the stable radix sort by finest bucket (header of k_site_keys): keys / values ping-pong in two halves of one buffer each
  const int nseg = (int)((n + kSortSeg - 1) / kSortSeg);
  if ((s = ensure(c, c->sortKeys, sizeof(unsigned) * 2 * n))) return s;
  if ((s = ensure(c, c->sortVals, sizeof(int) * 2 * n))) return s;
  if ((s = ensure(c, c->sortHist, sizeof(int) * (kSortDigits * (size_t)nseg + 2)))) return s;
  if ((s = ensure(c, c->scanTmp, sizeof(int64_t) * scan_scratch_elems(kSortDigits * (int64_t)nseg) * 2))) return s;
  unsigned* keyA = c->sortKeys.as<unsigned>();
  unsigned* keyB = keyA + n;
  int* valA = c->sortVals.as<int>();
  int* valB = valA + n;
  VD_LAUNCH(k_site_keys, grid_for(n, kBlock), kBlock, 0, st)(gp, c->sites.as<double>(), n, c->cellOf.as<int>(), c->subOff.as<int>(),
                                                             c->subOffRaw.as<int>(), keyA, valA, c->subCount.as<int>());
  exclusive_scan<int, int>(c->subCount.as<int>(), subCap + 1, c->subStart.as<int>(), c->scanTmp.as<int>(), st);
  int bits = 1;
  while (bits < 32 && ((int64_t)1 << bits) <= gridCap + subCap + 2) ++bits;   // keys are below gridCap + subCap
  const int sb = (nseg + kSortWarps - 1) / kSortWarps;
  const int npass = bits <= 11 ? 1 : (bits <= 22 ? 2 : 3);
  const int dbits = (bits + npass - 1) / npass;
  for (int shift = 0; shift < bits; shift += dbits) {
    VD_LAUNCH(k_radix_hist, sb, kSortWarps * kLanes, 0, st)(keyA, n, shift, dbits, nseg, c->sortHist.as<int>());
    exclusive_scan<int, int>(c->sortHist.as<int>(), ((int64_t)nseg << dbits), c->sortHist.as<int>(), c->scanTmp.as<int>(), st);
    VD_LAUNCH(k_radix_scatter, sb, kSortWarps * kLanes, 0, st)(keyA, valA, n, shift, dbits, nseg, c->sortHist.as<int>(), keyB, valB);
    unsigned* tk = keyA; keyA = keyB; keyB = tk;
    int* tv = valA; valA = valB; valB = tv;
  }
  VD_LAUNCH(k_gather_sorted, grid_for(n, kBlock), kBlock, 0, st)(c->sites.as<double>(), valA, n, c->sorted2.as<double4>(), f32 ? c->sorted32.as<float4>() : nullptr);
  // subStart holds the scan of the sub-cell counts for now; it is rebased to absolute positions in place
  VD_LAUNCH(k_sub_finalize, grid_for(gridCap, kWarpsPerBlock), kBlock, 0, st)(gp, c->subOff.as<int>(), c->subStart.as<int>(),
                                                                               c->subStart.as<int>());
  VD_LAUNCH(k_grid_finish, 1, 1, 0, st)(gp, c->sorted2.as<double4>(), c->heavyPrefix.as<int>(), c->subOff.as<int>(),
                                         c->subStart.as<int>(), &c->control.as<Control>()->nHeavy);
  if (lifted4) VD_LAUNCH(k_gather_weights, grid_for(n, kBlock), kBlock, 0, st)(gp, n, c->siteW.as<double>(), c->sortedW.as<double>());
  VD_LAUNCH(k_find_duplicates, grid_for(n, kBlock), kBlock, 0, st)(gp, n, &c->control.as<Control>()->err);
  if (stepMode)   // S1b
    VD_LAUNCH(k_delta, grid_for(n, kWarpsPerBlock), kBlock, 0, st)(gp, c->sites.as<double>(), n, c->delta.as<double>(),
                                                                   &c->control.as<Control>()->cnt[CNT_OTHER]);
  c->indexValid = true;
  return cuda_check(c, cudaGetLastError(), "site index");
}

vd_status stage_nearest_points(vd_ctx* c, const double* q3, int64_t nq, int* out) {
  if (nq <= 0) return VD_OK;
  const int blocks = grid_for(nq, kWarpsPerBlock);
  VD_LAUNCH(k_nearest_points, blocks, kBlock, 0, c->stream)(c->grid.as<GridIndex>(), q3, nq, out, &c->control.as<Control>()->cnt[CNT_OTHER]);
  return cuda_check(c, cudaGetLastError(), "nearest");
}

// ---- vd_nearest_static: the nearest-site query for callers that must not allocate (vd.h) ---------------------------------
//
// vd_nearest stages its queries and results in buffers it allocates per call.  This variant stages them in ONE file-scope
// device array of fixed size instead, so the call makes no cudaMalloc / cudaFree (nor any allocating routine): usable where
// allocation is forbidden (a stream under graph capture elsewhere in the process, a serving loop, a harness that traps
// cudaMalloc).  Every GPU that loads libvd.so holds the array (about 1.8 MB) until the process exits.  All calls, from every
// context, share it: it keeps the last call's contents, and calls that overlap on the GPU race -- one call at a time.
constexpr int kStaticMaxQueries = 1 << 16;

struct NearestScratch {
  double q[(size_t)kStaticMaxQueries * 3];   // the queries as given, [nq][dim]
  int res[kStaticMaxQueries];                // N_q of every query
  unsigned bad;                              // set when a query coordinate is not finite; must start at zero: cleared by every call
  unsigned pad[63];
};

static __device__ __align__(256) unsigned char g_nearest_scratch[sizeof(NearestScratch)];

// k_nearest_points with its input and output in the scratch block: one warp per query point; a 2-D query is padded with z = 0
// on the fly (the sites of a 2-D problem are stored that way).
__global__ void __launch_bounds__(kBlock) k_nearest_points_static(const GridIndex* __restrict__ gp, NearestScratch* __restrict__ S, int64_t nq, int dim) {
  const GridIndex g = *gp;
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / kLanes;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) / kLanes;
  QueryStats st = {0};
  extra_cnt_reset();
  for (int64_t q = warp; q < nq; q += nwarps) {
    const double x = S->q[q * dim + 0], y = S->q[q * dim + 1], z = dim == 3 ? S->q[q * dim + 2] : 0.0;
    const bool finite = x == x && y == y && z == z && fabs(x) <= 1e150 && fabs(y) <= 1e150 && fabs(z) <= 1e150;
    double best = 2e300;
    int bestId = 0x7fffffff;
    if (finite) nearest<true>(g, x, y, z, best, bestId, st);
    if (lane_id() == 0) {
      S->res[q] = finite ? bestId : -1;
      if (!finite) atomicOr(&S->bad, 1u);
    }
  }
}

// The array's name is a host-side stand-in in host code, not a device address: the address is asked for once per device,
// with that device current, and handed to the kernel.
static NearestScratch* nearest_scratch(vd_ctx* c) {
  static NearestScratch* ptr[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); c->lastError = "vd_nearest_static: no current device"; return nullptr; }
  if (!ptr[dev]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_nearest_scratch);
    if (e != cudaSuccess || !p) { cudaGetLastError(); c->lastError = std::string("vd_nearest_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e); return nullptr; }
    ptr[dev] = reinterpret_cast<NearestScratch*>(p);
  }
  return ptr[dev];
}

}  // namespace vd

extern "C" vd_status vd_nearest_static(vd_ctx* c, const double* queries, int64_t nq, int32_t* out_index) {
  using namespace vd;
  if (!c || !queries || !out_index || nq < 1) return VD_E_ARG;
  if (nq > kStaticMaxQueries) {
    c->lastError = "vd_nearest_static: at most " + std::to_string(kStaticMaxQueries) + " queries per call (the static scratch block); split the batch or use vd_nearest";
    return VD_E_ARG;
  }
  if (!c->indexValid) {
    c->lastError = "vd_nearest_static: the site index is not built (building it allocates: run vd_compute or vd_nearest once first)";
    return VD_E_STATE;
  }
  NearestScratch* S = nearest_scratch(c);
  if (!S) return VD_E_CUDA;
  cudaStream_t st = c->stream;
  cudaError_t e = cudaMemsetAsync(&S->bad, 0, sizeof(unsigned), st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(S->q, queries, sizeof(double) * c->dim * nq, cudaMemcpyDefault, st);
  if (e != cudaSuccess) return cuda_check(c, e, "vd_nearest_static");
  VD_LAUNCH(k_nearest_points_static, grid_for(nq, kWarpsPerBlock), kBlock, 0, st)(c->grid.as<GridIndex>(), S, nq, c->dim);
  unsigned bad = 0;
  e = cudaMemcpyAsync(out_index, S->res, sizeof(int) * nq, cudaMemcpyDefault, st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(&bad, &S->bad, sizeof(unsigned), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return cuda_check(c, e, "vd_nearest_static");
  if (bad) { c->lastError = "vd_nearest_static: non-finite query coordinate"; return VD_E_INPUT; }
  return VD_OK;
}
