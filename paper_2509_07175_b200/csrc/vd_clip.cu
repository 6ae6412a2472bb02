// vd_clip.cu -- S3 seeds, S4 clip kernels (one warp per (simplex, site) pair), S5 propagation through
// the pair list.  Alg. 4 / Alg. 5 lines 15-27 as a wavefront over one growing
// list: wave k processes the pairs pushed by wave k-1.  The wavefront loop itself runs on the device (wave programs,
// below: k_wave_begin / k_wave_end around the kernels of a wave); the host enqueues programs in batches.
#include <string.h>

#include <type_traits>

#include "vd_clip2d.cuh"
#include "vd_clip3d.cuh"

// This file (and vd_phase.cu) is compiled TWICE (build.py): as namespace vd::lean with VD_EXT = 0 -- the kernels without the code
// of the optional query features (weighted 3-D sites, step-out, D_alg counting) -- and as vd::full with VD_EXT = 1.  The kernels
// are bound by instruction fetch: the lean ones are 4-7 % faster on the BASELINE configs.  vd_compute picks per call.
#ifndef VD_CLIP2D_BLOCKS
#define VD_CLIP2D_BLOCKS 3   // resident blocks per SM of the one-kernel form on the triangle kinds
#endif
namespace vd {
namespace VD_VARIANT {

// S3 (Alg. 2 line 4: the first corner; Alg. 4 lines 3-6: the centroid): the nearest site of a corner of
// T_a owns that corner, so (T_a, N_p) is a non-empty pair and p is its witness.  One corner per simplex by default
// (vd_options.seed_corners): a seed pair starts from the bare simplex, a pair discovered from it brings the tuple
// (u, f) of P:L211 -- first clips without a search, corners known inside (U21, U22) -- so fewer seeds mean
// cheaper pairs; the closure of any one seed under positive flags is still every cell meeting T_a.
__global__ void __launch_bounds__(kBlock) k_seed(ClipArgs A, int nc, int nseed) {
  for (int64_t a = A.aBegin + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; a < A.aEnd; a += (int64_t)gridDim.x * blockDim.x) {
    for (int k = 0; k < nseed; ++k) {
      const int v = A.simp[a * nc + k];
      const int j = A.vnn[v];
      if (j < 0 || j >= A.n) continue;
      push_pair(A, (int)a, j, A.verts[(int64_t)v * 3 + 0], A.verts[(int64_t)v * 3 + 1], A.verts[(int64_t)v * 3 + 2]);
    }
  }
}

// More seeds when a simplex holds very many cells (n >= 64 m: a square of two triangles, "rectangle m = 1"):
// the pairs of T_a are found by propagation from its seeds over positive flags, one generation of
// neighbours per wavefront, so with only the corners as seeds a simplex of k cells takes ~k^(1/d) dependent
// wavefronts.  S interior points per simplex (a fixed low-discrepancy lattice in barycentric coordinates), each with
// its nearest site, seed (a, N_p) with witness p just as the centroid does in Alg. 4.
__global__ void __launch_bounds__(kBlock) k_sample_points(ClipArgs A, int nc, int S, double* __restrict__ pts) {
  const int64_t total = (int64_t)(A.aEnd - A.aBegin) * S;
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
    const int64_t a = A.aBegin + idx / S;
    const int j = (int)(idx % S) + 1;
    const double alpha[4] = {0.7548776662466927, 0.5698402909980532, 0.8191725133961645, 0.6710436067037893};
    double w[4], sum = 0.0;
    for (int k = 0; k < nc; ++k) {
      const double r = j * alpha[k];
      w[k] = (r - floor(r)) + 0.02;   // strictly inside
      sum += w[k];
    }
    double x = 0, y = 0, z = 0;
    for (int k = 0; k < nc; ++k) {
      const int v = A.simp[a * nc + k];
      const double t = w[k] / sum;
      x += t * A.verts[(int64_t)v * 3 + 0]; y += t * A.verts[(int64_t)v * 3 + 1]; z += t * A.verts[(int64_t)v * 3 + 2];
    }
    pts[idx * 3 + 0] = x; pts[idx * 3 + 1] = y; pts[idx * 3 + 2] = z;
  }
}

__global__ void __launch_bounds__(kBlock) k_seed_points(ClipArgs A, int S, const double* __restrict__ pts, const int* __restrict__ nn) {
  const int64_t total = (int64_t)(A.aEnd - A.aBegin) * S;
  for (int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (int64_t)gridDim.x * blockDim.x) {
    const int j = nn[idx];
    if (j < 0 || j >= A.n) continue;
    push_pair(A, (int)(A.aBegin + idx / S), j, pts[idx * 3 + 0], pts[idx * 3 + 1], pts[idx * 3 + 2]);
  }
}

// Simple domains (section V-B): a site inside the box owns its own position, so (box, v_i) is a non-empty pair
// with witness v_i ("each site must be in its own Voronoi cell").
__global__ void __launch_bounds__(kBlock) k_seed_sites(ClipArgs A, int ncorner, const int* __restrict__ own) {
  // the box's corners are the "mesh vertices": corner 0 = lo, the last = hi
  const double lx = A.verts[0], ly = A.verts[1], lz = A.verts[2];
  const double hx = A.verts[3 * (ncorner - 1) + 0], hy = A.verts[3 * (ncorner - 1) + 1], hz = A.verts[3 * (ncorner - 1) + 2];
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < A.n; i += (int64_t)gridDim.x * blockDim.x) {
    const double x = A.sites[i * 3 + 0], y = A.sites[i * 3 + 1], z = A.sites[i * 3 + 2];
    // power diagram: a site need not lie in its own cell (own[] = the power-nearest site of every site's position)
    if (x >= lx && x <= hx && y >= ly && y <= hy && z >= lz && z <= hz && (!own || own[i] == (int)i)) push_pair(A, 0, (int)i, x, y, z);
  }
}

// Alg. 5 lines 4-14 in one pass over the sites, after the restricted diagram on the boundary triangles (child
// context) is known: a site with a non-empty restricted cell is a BOUNDARY site -- every restricted polygon H of its cell seeds
// (incident tet of H's triangle, site), witness = H's corner average (lines 8-14); a site with an empty one whose position lies
// in the convex domain is INTERIOR -- its cell is its whole Voronoi cell, one pair (m, site) against the bounding
// box (line 6); a site outside the domain with an empty restricted cell owns nothing (reading U13).
__global__ void __launch_bounds__(kBlock) k_dissolve_seeds(ClipArgs A, const double* __restrict__ bMeasure, const int64_t* __restrict__ bPieceOff,
                                                            const int* __restrict__ bPieceTri, const int64_t* __restrict__ bVertOff,
                                                            const double* __restrict__ bXYZ, const int* __restrict__ bTet,
                                                            const double4* __restrict__ planes, int np, double tol) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < A.n; i += (int64_t)gridDim.x * blockDim.x) {
    if (bMeasure[i] > 0.0) {
      for (int64_t p = bPieceOff[i]; p < bPieceOff[i + 1]; ++p) {
        double x = 0, y = 0, z = 0;
        const int64_t v0 = bVertOff[p], v1 = bVertOff[p + 1];
        for (int64_t v = v0; v < v1; ++v) { x += bXYZ[v * 3 + 0]; y += bXYZ[v * 3 + 1]; z += bXYZ[v * 3 + 2]; }
        const double inv = 1.0 / (double)(v1 - v0);
        push_pair(A, bTet[bPieceTri[p]], (int)i, x * inv, y * inv, z * inv);
      }
    } else {
      const double x = A.sites[i * 3 + 0], y = A.sites[i * 3 + 1], z = A.sites[i * 3 + 2];
      bool inside = true;
      for (int k = 0; k < np && inside; ++k) {
        const double4 q = planes[k];
        inside = q.x * x + q.y * y + q.z * z - q.w <= tol * fmax(1.0, fmax(fabs(q.w), fabs(x) + fabs(y) + fabs(z)));
      }
      if (inside) push_pair(A, A.m, (int)i, x, y, z);
    }
  }
}

// Tet meshes: U19 pays when the cells are about as large as the simplices or smaller and most sites own one -- every pair then
// faces several of its site's nearest bisectors (C2: 17.0 -> 14.8 ms).  With far sites (C5) or cells that span many simplices
// nearly all those planes miss the pair's simplex and the list is wasted work.  Decided on the device from two counts: the
// sites inside the domain's bounding box against n and against m.  auto[0..2] / [3..5]: the box as sortable keys, [6]: the count.
__device__ __forceinline__ unsigned long long dkey(double v) {
  const unsigned long long b = (unsigned long long)__double_as_longlong(v);
  return (b >> 63) ? ~b : (b | 0x8000000000000000ull);
}
__device__ __forceinline__ double dkey_inv(unsigned long long k) {
  return __longlong_as_double((long long)((k >> 63) ? (k & 0x7fffffffffffffffull) : ~k));
}
__global__ void __launch_bounds__(kBlock) k_near_box(const double* __restrict__ verts, int64_t nv, unsigned long long* __restrict__ au) {
  double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nv; i += (int64_t)gridDim.x * blockDim.x)
    for (int a = 0; a < 3; ++a) { const double v = verts[i * 3 + a]; lo[a] = fmin(lo[a], v); hi[a] = fmax(hi[a], v); }
  for (int a = 0; a < 3; ++a) {
    for (int off = kLanes / 2; off > 0; off >>= 1) {
      lo[a] = fmin(lo[a], __shfl_xor_sync(kFull, lo[a], off));
      hi[a] = fmax(hi[a], __shfl_xor_sync(kFull, hi[a], off));
    }
    if (lane_id() == 0) { atomicMin(&au[a], dkey(lo[a])); atomicMax(&au[3 + a], dkey(hi[a])); }
  }
}
__global__ void __launch_bounds__(kBlock) k_near_count(const double* __restrict__ sites, int64_t n, unsigned long long* __restrict__ au) {
  double lo[3], hi[3];
  for (int a = 0; a < 3; ++a) { lo[a] = dkey_inv(au[a]); hi[a] = dkey_inv(au[3 + a]); }
  int cnt = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    bool in = true;
    for (int a = 0; a < 3; ++a) { const double v = sites[i * 3 + a]; in = in && v >= lo[a] && v <= hi[a]; }
    cnt += in ? 1 : 0;
  }
  cnt = warp_sum(cnt);
  if (lane_id() == 0 && cnt) atomicAdd(&au[6], (unsigned long long)cnt);
}

// Reading U19: the sites nearest to every site (approximately, from the 3 x 3 x 3 grid cells around it), nearest
// first; one warp per site.  Their bisectors are the first clips of every piece of that site's cell.
// au (tet meshes, no explicit vd_options.near_clips): the counts above decide; "no" leaves every list empty.
__global__ void __launch_bounds__(kBlock) k_near(ClipArgs A, int* __restrict__ list, int K, const unsigned long long* __restrict__ au, long long m) {
  if (au) {
    const long long inside = (long long)au[6];
    if (!(2 * inside >= (long long)A.n && m <= 4 * inside)) {
      for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < A.n; i += (int64_t)gridDim.x * blockDim.x) list[i * K] = -1;
      return;
    }
  }
  __shared__ GridIndex g;
  __shared__ int ids[kWarpsPerBlock][kLanes];
  if (threadIdx.x == 0) g = *A.grid;
  __syncthreads();
  const int w = (int)threadIdx.x / kLanes, lane = lane_id();
  QueryStats st = {0};
  for (int64_t i = (int64_t)blockIdx.x * kWarpsPerBlock + w; i < A.n; i += (int64_t)gridDim.x * kWarpsPerBlock) {
    const int k = near_sites(g, A.sites[i * 3 + 0], A.sites[i * 3 + 1], A.sites[i * 3 + 2], (int)i, K, ids[w], st);
    if (lane < K) list[i * K + lane] = lane < k ? ids[w][lane] : -1;
    __syncwarp();
  }
}

// vd_phase.cu
vd_status phase_buffers(vd_ctx* c, int64_t cap);
void enqueue_phased(vd_ctx* c, const ClipArgs& A, bool hv, int64_t cap, int rounds, int tailPairs);
PhaseCtl* phase_ctl(vd_ctx* c, int64_t cap);

constexpr int kSmallWave = 8192;       // phased schedule: a wavefront smaller than this runs as one launch of the one-kernel form
constexpr int P3 = 32, C3 = 64;        // fast tier: planes / corners per piece held per warp
constexpr int P3B = 256, C3B = 512;    // large tier (one warp per block)
constexpr int K2B = 256;                // large 2D tier: corners per polygon

// The one-kernel form: a warp takes a pair through all of Alg. 3.  What it works on comes from the wave program's state
// (k_wave_begin): fast tier -- the wave [pc->begin, + pc->count) (WAVE_SINGLE), or the whole list from the wave's first pair
// on as a device-side queue (WAVE_QUEUE); large tier (BIG) -- the deferred pairs ovf[ovfBegin .. ovfEnd).
template <int KIND, bool BIG, bool HV>
__global__ void __launch_bounds__(BIG ? kLanes : kBlock, BIG ? 1 : ((KIND == KIND_TRI_2D || KIND == KIND_BOX_2D) ? VD_CLIP2D_BLOCKS : 3)) k_clip(ClipArgs A, const int* __restrict__ list, const PhaseCtl* __restrict__ pc) {
  constexpr int W = BIG ? 1 : kWarpsPerBlock;
  int64_t begin, end;
  bool persist = false;
  if (BIG) {
    begin = (int64_t)A.ctl->ovfBegin; end = (int64_t)A.ctl->ovfEnd;
    if (begin >= end) return;
  } else {
    const unsigned mode = pc->mode;
    if (mode != WAVE_QUEUE && mode != WAVE_SINGLE) return;
    persist = mode == WAVE_QUEUE;
    begin = persist ? 0 : (int64_t)pc->begin;     // queue: tickets are absolute list positions (the cursor starts at the wave)
    end = (int64_t)pc->begin + (int64_t)pc->count;
  }
  __shared__ GridIndex g;
  if (threadIdx.x == 0) g = *A.grid;
  __syncthreads();
  const int w = (int)threadIdx.x / kLanes;
  QueryStats st = {0};
  LocalCnt lc = {0u, 0u, 0u, 0u, 0u, 0u};
  extra_cnt_reset();
  constexpr bool BOX = KIND == KIND_BOX_2D || KIND == KIND_BOX_3D;
  if constexpr (KIND == KIND_TET_3D || KIND == KIND_BOX_3D) {
    __shared__ Poly3<BIG ? P3B : P3, BIG ? C3B : C3> S[W];
    for (;;) {
      // dynamic work distribution: pieces range from 4 to hundreds of corners
      const int64_t k = next_ticket<BIG>(A, begin, end, persist);
      if (k < 0) break;
      const int64_t idx = list ? (int64_t)list[k] : k;
      const int rc = clip_pair_3d<BIG ? P3B : P3, BIG ? C3B : C3, HV, BOX>(S[w], g, A, idx, st, lc);
      if (rc == 1) {
        if (BIG) {
          if (lane_id() == 0) {
            atomicOr(&A.ctl->err, ERR_PIECE_CAP);
            Piece pc = {};
            pc.site = A.pairs[idx].i; pc.simplex = A.pairs[idx].a;
            A.pieces[idx] = pc;
          }
        } else if (lane_id() == 0) {
          const unsigned long long slot = atomicAdd(&A.ctl->ovfTail, 1ull);
          if ((int64_t)slot < A.ovfCap) A.ovf[slot] = (int)idx; else atomicOr(&A.ctl->err, ERR_PAIR_CAP);
        }
      }
      if (!BIG) pair_done(A);
      __syncwarp();
    }
  } else {
    // fast tier: one lane per corner (at most 32 corners); large tier: the serial loop surgery on up to 256 corners
    __shared__ typename std::conditional<BIG, Poly2<K2B>, Poly2P>::type S[W];
    for (;;) {
      const int64_t k = next_ticket<BIG>(A, begin, end, persist);
      if (k < 0) break;
      const int64_t idx = list ? (int64_t)list[k] : k;
      int rc;
      if constexpr (BIG) rc = clip_pair_2d<K2B, HV, BOX>(S[w], g, A, idx, st, lc);
      else rc = clip_pair_2d_par<HV, BOX>(S[w], g, A, idx, st, lc);
      if (rc == 1) {
        if (BIG) {
          if (lane_id() == 0) {
            atomicOr(&A.ctl->err, ERR_PIECE_CAP);
            Piece pc = {};
            pc.site = A.pairs[idx].i; pc.simplex = A.pairs[idx].a;
            A.pieces[idx] = pc;
          }
        } else if (lane_id() == 0) {
          const unsigned long long slot = atomicAdd(&A.ctl->ovfTail, 1ull);
          if ((int64_t)slot < A.ovfCap) A.ovf[slot] = (int)idx; else atomicOr(&A.ctl->err, ERR_PAIR_CAP);
        }
      }
      if (!BIG) pair_done(A);
      __syncwarp();
    }
  }
  flush_counters(A.ctl, st, lc);
}

// reading U19: the whole-cell kinds start every cell from the bisectors of its site's 24 nearest sites; tet meshes from 16, where
// the device-side counts of k_near say it pays (near_auto)
static int near_clips_of(const vd_ctx* c) {
  const int k = c->opt.near_clips;
  if (k == 0) return (c->kind == KIND_BOX_3D || (c->kind == KIND_TET_3D && c->opt.dissolve > 0)) ? 24 : (c->kind == KIND_TET_3D ? 16 : 0);
  return k > kLanes ? kLanes : (k < 0 ? 0 : k);
}
static bool near_auto(const vd_ctx* c) { return c->opt.near_clips == 0 && c->kind == KIND_TET_3D && !(c->opt.dissolve > 0); }

static ClipArgs make_args(vd_ctx* c) {
  ClipArgs A;
  A.grid = c->grid.as<GridIndex>();
  A.sites = c->sites.as<double>();
  A.siteW = (c->weighted && c->dim == 3) ? c->siteW.as<double>() : nullptr;
  A.verts = c->verts.as<double>();
  A.simp = c->simp.as<int>();
  A.adj = c->adj.as<int>();
  A.vnn = c->vnn.as<int>();
  A.nearList = nullptr;
  A.queue = 0;
  A.wholeA = -1; A.dissolve = 0; A.boxVerts = c->verts.as<double>(); A.boxVnn = c->vnn.as<int>();
  if (c->kind == KIND_BOX_3D) A.wholeA = 0;
  if (c->kind == KIND_TET_3D && c->opt.dissolve > 0) {
    A.wholeA = (int)c->m; A.dissolve = 1;
    A.boxVerts = c->boxVerts.as<double>(); A.boxVnn = c->boxVnn.as<int>();
  }
  A.n = (int)c->n; A.m = (int)c->m; A.kind = c->kind;
  A.realEdges = c->opt.real_edges;
  A.ballCells = c->opt.ball_cells == 0 ? 64 : c->opt.ball_cells;
  A.nearClips = near_clips_of(c);
  A.firstClip = c->opt.first_clip >= 0 ? 1 : 0;
  A.aBegin = 0; A.aEnd = (int)c->m;
  if (c->opt.simplex_end > 0 && c->kind != KIND_BOX_2D && c->kind != KIND_BOX_3D) {
    A.aBegin = c->opt.simplex_begin < 0 ? 0 : c->opt.simplex_begin;
    A.aEnd = c->opt.simplex_end > (int)c->m ? (int)c->m : c->opt.simplex_end;
    if (A.aBegin > A.aEnd) A.aBegin = A.aEnd;
  }
  if (A.nearClips > 0 && c->nearList.p) A.nearList = c->nearList.as<int>();
  A.ctl = c->control.as<Control>();
  A.pairs = c->pairs.as<Pair>();
  A.pieces = c->pieces.as<Piece>();
  A.visited = c->visited.as<unsigned long long>();
  A.hashMask = (uint64_t)c->hashCap - 1;
  A.pairCap = c->pairCap; A.vertCap = c->vertCap; A.nbrCap = c->nbrCap; A.ovfCap = c->ovfCap;
  A.ovf = c->ovf.as<int>();
  A.poolXYZ = c->poolXYZ.as<double>();
  A.poolFlags = c->poolFlags.as<int>();
  A.poolNbr = c->poolNbr.as<int>();
  A.sitePieces = c->sitePieces.as<int>();
  A.siteNbrRaw = c->siteNbrRaw.as<int>();
  return A;
}

static int blocks_for(int64_t items, int perBlock, int cap) {
  int64_t b = (items + perBlock - 1) / perBlock;
  if (b > cap) b = cap;
  if (b < 1) b = 1;
  return (int)b;
}

vd_status stage_seed(vd_ctx* c) {
  vd_status s;
  cudaStream_t st = c->stream;
  if ((s = ensure(c, c->vnn, sizeof(int) * c->nv))) return s;
  // nearest site of every mesh vertex: classifies the corners of every T_a and seeds the pair list
  if ((s = stage_nearest_points(c, c->verts.as<double>(), c->nv, c->vnn.as<int>()))) return s;
  cudaMemsetAsync(c->visited.p, 0, sizeof(unsigned long long) * c->hashCap, st);
  cudaMemsetAsync(c->pairs.p, 0xff, sizeof(Pair) * c->pairCap, st);   // simplex id < 0: slot not yet pushed
  cudaMemsetAsync(c->sitePieces.p, 0, sizeof(int) * c->n, st);
  cudaMemsetAsync(c->siteNbrRaw.p, 0, sizeof(int) * c->n, st);
  const int K = near_clips_of(c);
  if (K != c->nearK) c->nearReady = false;   // (a list of another width is of no use)
  c->nearK = K;
  if (K > 0) {
    if ((s = ensure(c, c->nearList, sizeof(int) * c->n * K))) return s;
  } else {
    release(c, c->nearList);
  }
  const ClipArgs A = make_args(c);
  const bool boxKind0 = c->kind == KIND_BOX_2D || c->kind == KIND_BOX_3D;
  if (A.dissolve) {
    // Alg. 5 lines 2-14: classify the sites through the restricted diagram on the boundary, seed boundary sites tet by tet and
    // interior sites as whole cells
    if ((s = stage_nearest_points(c, c->boxVerts.as<double>(), 8, c->boxVnn.as<int>()))) return s;
    if (K > 0) VD_LAUNCH(k_near, blocks_for(c->n, kWarpsPerBlock, sm_count() * 8), kBlock, 0, st)(A, c->nearList.as<int>(), K, nullptr, 0);
    if ((s = stage_dissolve_classify(c))) return s;
    const vd_cells& b = c->boundary->cells;
    VD_LAUNCH(k_dissolve_seeds, blocks_for(c->n, kBlock, sm_count() * 8), kBlock, 0, st)(
        A, b.measure, b.piece_off, b.piece_simplex, b.vert_off, b.vert_xyz, c->bTet.as<int>(), c->bPlanes.as<double4>(), c->nBPlanes, 1e-12);
    return cuda_check(c, cudaGetLastError(), "seed (dissolve)");
  }
  const unsigned long long* au = nullptr;
  if (K > 0 && near_auto(c)) {
    if ((s = ensure(c, c->nearAuto, sizeof(unsigned long long) * 8))) return s;
    cudaMemsetAsync(c->nearAuto.p, 0xff, sizeof(unsigned long long) * 3, st);
    cudaMemsetAsync(c->nearAuto.as<unsigned long long>() + 3, 0, sizeof(unsigned long long) * 5, st);
    VD_LAUNCH(k_near_box, blocks_for(c->nv, kBlock, sm_count() * 4), kBlock, 0, st)(c->verts.as<double>(), c->nv, c->nearAuto.as<unsigned long long>());
    VD_LAUNCH(k_near_count, blocks_for(c->n, kBlock, sm_count() * 8), kBlock, 0, st)(c->sites.as<double>(), c->n, c->nearAuto.as<unsigned long long>());
    au = c->nearAuto.as<unsigned long long>();
  }
  if (K > 0 && !c->nearReady) VD_LAUNCH(k_near, blocks_for(c->n, kWarpsPerBlock, sm_count() * 8), kBlock, 0, st)(A, c->nearList.as<int>(), K, au, (long long)c->m);
  c->nearReady = false;   // (set by vd_lloyd: the list holds the previous iteration's neighbours)
  VD_LAUNCH(k_seed, blocks_for(A.aEnd - A.aBegin + 1, kBlock, sm_count() * 8), kBlock, 0, st)(A, c->nc, (boxKind0 || c->opt.seed_corners >= c->nc) ? c->nc : (c->opt.seed_corners > 0 ? c->opt.seed_corners : 1));
  const bool boxKind = c->kind == KIND_BOX_2D || c->kind == KIND_BOX_3D;
  const int64_t mLocal = A.aEnd - A.aBegin;
  if (!boxKind && mLocal > 0 && c->n >= 64 * mLocal) {
    // about one seed point per expected cell of the simplex, at most 1024 (measured on C1: n / 4m seeds 1.25 ms and 10
    // wavefronts, n / m seeds 0.88 ms and 5 -- a seed pair costs more queries than a discovered one, but here latency rules)
    const int64_t want = c->n / mLocal;
    const int S = (int)(want > 1024 ? 1024 : want);
    const int64_t total = mLocal * S;
    if ((s = ensure(c, c->seedPts, sizeof(double) * 3 * total))) return s;
    if ((s = ensure(c, c->seedNN, sizeof(int) * total))) return s;
    VD_LAUNCH(k_sample_points, blocks_for(total, kBlock, sm_count() * 8), kBlock, 0, st)(A, c->nc, S, c->seedPts.as<double>());
    if ((s = stage_nearest_points(c, c->seedPts.as<double>(), total, c->seedNN.as<int>()))) return s;
    VD_LAUNCH(k_seed_points, blocks_for(total, kBlock, sm_count() * 8), kBlock, 0, st)(A, S, c->seedPts.as<double>(), c->seedNN.as<int>());
  }
  if (boxKind) {
    const int* own = nullptr;
    if (A.siteW) {
      if ((s = ensure(c, c->seedNN, sizeof(int) * c->n))) return s;
      if ((s = stage_nearest_points(c, c->sites.as<double>(), c->n, c->seedNN.as<int>()))) return s;
      own = c->seedNN.as<int>();
    }
    VD_LAUNCH(k_seed_sites, blocks_for(c->n, kBlock, sm_count() * 8), kBlock, 0, st)(A, c->nc, own);
  }
  return cuda_check(c, cudaGetLastError(), "seed");
}

// ---- wave programs: the wavefront loop of Alg. 4 / 5 ("while L1 is not empty") without the host -----------
//
// A wave program is a fixed sequence of launches: k_wave_begin looks at the pair list and decides what this wave is (nothing
// / phased / queue drain / one launch of the one-kernel form), the kernels that follow read that decision and their counts
// from device memory (PhaseCtl) and return at once when they have no work, k_wave_end closes the wave and hands the deferred
// pairs to the large tier.  The host enqueues programs a batch at a time and looks at the device once per batch.

// allowPhased: 3D kinds under the phased schedule; smallMode: what a wave below smallWave pairs (or any wave when
// !allowPhased) runs as -- WAVE_QUEUE or WAVE_SINGLE.
__global__ void k_wave_begin(ClipArgs A, PhaseCtl* pc, int allowPhased, int smallWave, int smallMode, long long chunkCap) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  Control* ctl = A.ctl;
  pc->mode = WAVE_NONE; pc->count = 0; pc->nDone = 0;
  for (int k = 0; k < kMaxRounds + 2; ++k) { pc->nClip[k] = 0; pc->nLoose[k] = 0; pc->nLooseFix[k] = 0; }
  for (int k = 0; k < 4 * kMaxRounds + 4; ++k) pc->ticket[k] = 0;
  if (ctl->err & (ERR_PAIR_CAP | ERR_VERT_CAP | ERR_NBR_CAP | ERR_DUPLICATE | ERR_INPUT)) return;   // the host reruns / reports
  const unsigned long long begin = ctl->waveEnd;
  unsigned long long tail = ctl->pairTail;
  if (tail > (unsigned long long)A.pairCap) tail = (unsigned long long)A.pairCap;
  if (tail <= begin) return;
  unsigned long long n = tail - begin;
  ctl->nWaves += 1;
  pc->begin = begin;
  if (allowPhased && n >= (unsigned long long)smallWave) {
    if (n > (unsigned long long)chunkCap) n = (unsigned long long)chunkCap;   // a wave larger than the parking area runs in chunks
    pc->mode = WAVE_PHASED;
    ctl->waveEnd = begin + n;
  } else if (smallMode == WAVE_QUEUE) {
    pc->mode = WAVE_QUEUE;
    ctl->fetch[0] = begin;       // next ticket = next list position
    ctl->finished = begin;       // the queue is drained when every dispatched pair has finished and none is left
    ctl->waveEnd = tail;         // (k_wave_end moves it to the final tail)
  } else {
    pc->mode = WAVE_SINGLE;
    ctl->fetch[0] = 0;
    ctl->waveEnd = tail;
  }
  pc->count = (unsigned)n;
}

__global__ void k_wave_end(ClipArgs A, PhaseCtl* pc) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  Control* ctl = A.ctl;
  if (pc->mode == WAVE_QUEUE) {
    unsigned long long tail = ctl->pairTail;
    if (tail > (unsigned long long)A.pairCap) tail = (unsigned long long)A.pairCap;
    ctl->waveEnd = tail;         // the queue kernel ended: every pair pushed so far has been processed
  }
  unsigned long long ot = ctl->ovfTail;
  if (ot > (unsigned long long)A.ovfCap) ot = (unsigned long long)A.ovfCap;
  ctl->ovfBegin = ctl->ovfDone;
  ctl->ovfEnd = ot;
  ctl->ovfDone = ot;
  ctl->fetch[1] = 0;
}

template <int KIND>
static void launch_kind(vd_ctx* c, const ClipArgs& A, bool hv, bool big, const PhaseCtl* pc) {
  cudaStream_t st = c->stream;
  if (!big) {
    const int blocks = sm_count() * ((KIND == KIND_TRI_2D || KIND == KIND_BOX_2D) ? VD_CLIP2D_BLOCKS : 3);
    if (hv) VD_LAUNCH((k_clip<KIND, false, true>), blocks, kBlock, 0, st)(A, nullptr, pc);
    else VD_LAUNCH((k_clip<KIND, false, false>), blocks, kBlock, 0, st)(A, nullptr, pc);
  } else {
    const int blocks = sm_count() * 8;
    if (hv) VD_LAUNCH((k_clip<KIND, true, true>), blocks, kLanes, 0, st)(A, A.ovf, pc);
    else VD_LAUNCH((k_clip<KIND, true, false>), blocks, kLanes, 0, st)(A, A.ovf, pc);
  }
}

// one kernel per piece structure: triangles (both triangle kinds share the loop code), tets, rectangle, box
static void launch(vd_ctx* c, const ClipArgs& A, bool hv, bool big, const PhaseCtl* pc) {
  switch (c->kind) {
    case KIND_TET_3D: launch_kind<KIND_TET_3D>(c, A, hv, big, pc); break;
    case KIND_BOX_3D: launch_kind<KIND_BOX_3D>(c, A, hv, big, pc); break;
    case KIND_BOX_2D: launch_kind<KIND_BOX_2D>(c, A, hv, big, pc); break;
    default:          launch_kind<KIND_TRI_2D>(c, A, hv, big, pc); break;
  }
}

static cudaError_t read_control(vd_ctx* c, Control& h) {
  static_assert(sizeof(Control) <= 1024, "fits the page-locked staging block");
  Control* dst = c->pinned ? reinterpret_cast<Control*>(c->pinned) : &h;
  cudaError_t e = cudaMemcpyAsync(dst, c->control.p, sizeof(Control), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = sync_stream(c, "wave batch");
  if (e == cudaSuccess && dst != &h) h = *dst;
  return e;
}

vd_status stage_clip(vd_ctx* c) {
  ClipArgs A = make_args(c);
  A.queue = 1;   // a program may run the device-side queue: pushed pairs are published with a fence
  const int mode = c->opt.persistent;
  const bool solid = c->kind == KIND_TET_3D || c->kind == KIND_BOX_3D;
  const bool phased = solid && (mode == 1 || mode == 2);   // 3D kinds: one small kernel per step (vd_phase.cu)
  // waves that do not run phased: a device-side queue that drains everything (3; the short last wavefronts of the 3D
  // kinds; 2 for the triangle kinds), or one launch of the one-kernel form per wavefront (0; the triangle kinds' default:
  // with the discovery tuples and interior seeds their wavefronts are few, and the queue's polling costs more)
  const int smallMode = (mode == 3 || (mode == 2 && !solid) || (phased && mode == 1 && c->opt.small_wave >= 0)) ? WAVE_QUEUE : WAVE_SINGLE;
  const int smallWave = !phased ? 0 : (c->opt.small_wave == 0 ? kSmallWave : (c->opt.small_wave < 0 ? 1 : c->opt.small_wave));
  const int tailPairs = c->opt.tail_pairs == 0 ? 65536 : (c->opt.tail_pairs < 0 ? 0 : c->opt.tail_pairs);
  const int64_t chunk = (int64_t)1 << 20;
  const int64_t cap = phased ? (c->pairCap < chunk ? c->pairCap : chunk) : 1;
  vd_status s;
  if ((s = phase_buffers(c, cap))) return s;
  PhaseCtl* pc = phase_ctl(c, cap);
  // refined cells of the index decide which kernels run (those that know the second level), and bad sites end the step
  // here: one look at the device -- unless this context already built the index of these very sites
  Control h;
  cudaError_t e = cudaSuccess;
  if (c->heavyKnown >= 0) {
    memset(&h, 0, sizeof(h));
    h.nHeavy = (unsigned)c->heavyKnown;
    h.pairTail = 1;   // (unknown yet: the seeds)
  } else {
    if ((e = read_control(c, h)) != cudaSuccess) return cuda_check(c, e, "clip");
    if (!(h.err & (ERR_DUPLICATE | ERR_INPUT))) c->heavyKnown = (int)h.nHeavy;
  }
  const bool hv = h.nHeavy > 0;
  // rounds of {tests, clips} per wave program before k_ph_tail finishes what they leave.  Measured: on tet meshes with
  // the plain index the finishing kernel's loop alone (no parking between a pair's clips) beats any number of rounds; whole cells (more
  // clips per pair) and the refined index (long searches, better in kernels of their own) want rounds.
  int rounds = c->opt.rounds > 0 ? c->opt.rounds : (c->opt.rounds < 0 ? 0 : (hv ? 5 : (c->kind == KIND_BOX_3D ? 3 : 0)));
  if (rounds > kMaxRounds) rounds = kMaxRounds;
  int batch = (!phased && smallMode == WAVE_SINGLE) ? 8 : 6;   // the seeds' wave and the large ones it sets off
  for (int guard = 0; guard < 4096; ++guard) {
    if (h.err & (ERR_PAIR_CAP | ERR_VERT_CAP | ERR_NBR_CAP)) break;   // caller grows the pools and reruns
    if (h.err & (ERR_DUPLICATE | ERR_INPUT)) break;                   // bad sites (S1): nothing to clip
    unsigned long long tail = h.pairTail, otail = h.ovfTail;
    if (tail > (unsigned long long)c->pairCap) tail = (unsigned long long)c->pairCap;
    if (otail > (unsigned long long)c->ovfCap) otail = (unsigned long long)c->ovfCap;
    if (h.waveEnd >= tail && h.ovfDone >= otail) break;               // "while L1 is not empty"
    for (int k = 0; k < batch; ++k) {
      VD_LAUNCH(k_wave_begin, 1, 32, 0, c->stream)(A, pc, phased ? 1 : 0, smallWave, smallMode, (long long)cap);
      if (phased) enqueue_phased(c, A, hv, cap, rounds, tailPairs);
      launch(c, A, hv, false, pc);
      VD_LAUNCH(k_wave_end, 1, 32, 0, c->stream)(A, pc);
      launch(c, A, hv, true, pc);
    }
    if ((e = read_control(c, h)) != cudaSuccess) return cuda_check(c, e, "clip wave");
    phase_marks_collect(c);
    // what is waiting now is the next wave, exactly: a large one will set off another, a short one is drained -- with all
    // that follows from it -- by the queue kernel of a single program
    const unsigned long long waiting = (h.pairTail < (unsigned long long)c->pairCap ? h.pairTail : (unsigned long long)c->pairCap) - h.waveEnd;
    batch = (!phased && smallMode == WAVE_SINGLE) ? 8 : ((phased && waiting >= (unsigned long long)smallWave) ? 2 : 1);   // (a program of the triangle kinds is four launches)
  }
  c->hostControl = h;
  c->counters.waves = (int64_t)h.nWaves;
  return cuda_check(c, cudaGetLastError(), "clip");
}

}  // namespace VD_VARIANT
}  // namespace vd
