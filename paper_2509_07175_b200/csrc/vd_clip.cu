// vd_clip.cu -- S3 seeds, S4 clip kernels (one warp per (simplex, site) pair), S5 propagation through
// the pair list.  Alg. 4 / Alg. 5 lines 15-27 as a wavefront over one growing
// list: wave k processes the pairs pushed by wave k-1.
#include "vd_clip2d.cuh"
#include "vd_clip3d.cuh"

namespace vd {

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
__global__ void __launch_bounds__(kBlock) k_seed_sites(ClipArgs A, double lx, double ly, double lz, double hx, double hy, double hz) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < A.n; i += (int64_t)gridDim.x * blockDim.x) {
    const double x = A.sites[i * 3 + 0], y = A.sites[i * 3 + 1], z = A.sites[i * 3 + 2];
    if (x >= lx && x <= hx && y >= ly && y <= hy && z >= lz && z <= hz) push_pair(A, 0, (int)i, x, y, z);
  }
}

// Reading U19: the sites nearest to every site (approximately, from the 3 x 3 x 3 grid cells around it), nearest
// first; one warp per site.  Their bisectors are the first clips of every piece of that site's cell.
__global__ void __launch_bounds__(kBlock) k_near(ClipArgs A, int* __restrict__ list, int K) {
  __shared__ GridIndex g;
  __shared__ int ids[kWarpsPerBlock][kLanes];
  if (threadIdx.x == 0) g = *A.grid;
  __syncthreads();
  const int w = (int)threadIdx.x / kLanes, lane = lane_id();
  QueryStats st = {0u, 0u, 0u};
  for (int64_t i = (int64_t)blockIdx.x * kWarpsPerBlock + w; i < A.n; i += (int64_t)gridDim.x * kWarpsPerBlock) {
    const int k = near_sites(g, A.sites[i * 3 + 0], A.sites[i * 3 + 1], A.sites[i * 3 + 2], (int)i, K, ids[w], st);
    if (lane < K) list[i * K + lane] = lane < k ? ids[w][lane] : -1;
    __syncwarp();
  }
}

vd_status run_phases(vd_ctx* c, const ClipArgs& A, bool hv, int64_t begin, int64_t end);   // vd_phase.cu

constexpr int kSmallWave = 8192;       // phased schedule: a wavefront smaller than this runs as one launch of the one-kernel form
constexpr int P3 = 32, C3 = 64;        // fast tier: planes / corners per piece held per warp
constexpr int P3B = 256, C3B = 512;    // large tier (one warp per block)
constexpr int K2 = 32, K2B = 256;

// items: pairs[begin .. end) when list == nullptr, else pairs[list[begin .. end)]
template <int KIND, bool BIG, bool HV>
__global__ void __launch_bounds__(BIG ? kLanes : kBlock, BIG ? 1 : 3) k_clip(ClipArgs A, const int* __restrict__ list, int64_t begin, int64_t end, bool persist) {
  constexpr int W = BIG ? 1 : kWarpsPerBlock;
  __shared__ GridIndex g;
  if (threadIdx.x == 0) g = *A.grid;
  __syncthreads();
  const int w = (int)threadIdx.x / kLanes;
  QueryStats st = {0u, 0u, 0u};
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
    __shared__ Poly2<BIG ? K2B : K2> S[W];
    for (;;) {
      const int64_t k = next_ticket<BIG>(A, begin, end, persist);
      if (k < 0) break;
      const int64_t idx = list ? (int64_t)list[k] : k;
      const int rc = clip_pair_2d<BIG ? K2B : K2, HV, BOX>(S[w], g, A, idx, st, lc);
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

// reading U19: by default only the whole-cell kinds start from the bisectors of the nearest sites (measured: on
// tet meshes the extra plane tests and redundant clips cost more than the searches they save)
static int near_clips_of(const vd_ctx* c) {
  const int k = c->opt.near_clips;
  if (k == 0) return (c->kind == KIND_BOX_3D) ? 20 : 0;
  return k > kLanes ? kLanes : k;
}

static ClipArgs make_args(vd_ctx* c) {
  ClipArgs A;
  A.grid = c->grid.as<GridIndex>();
  A.sites = c->sites.as<double>();
  A.verts = c->verts.as<double>();
  A.simp = c->simp.as<int>();
  A.adj = c->adj.as<int>();
  A.vnn = c->vnn.as<int>();
  A.nearList = nullptr;
  A.queue = 0;
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
  if (K > 0) {
    if ((s = ensure(c, c->nearList, sizeof(int) * c->n * K))) return s;
  } else {
    release(c, c->nearList);
  }
  const ClipArgs A = make_args(c);
  const bool boxKind0 = c->kind == KIND_BOX_2D || c->kind == KIND_BOX_3D;
  if (K > 0) VD_LAUNCH(k_near, blocks_for(c->n, kWarpsPerBlock, sm_count() * 8), kBlock, 0, st)(A, c->nearList.as<int>(), K);
  VD_LAUNCH(k_seed, blocks_for(A.aEnd - A.aBegin + 1, kBlock, sm_count() * 8), kBlock, 0, st)(A, c->nc, (boxKind0 || c->opt.seed_corners >= c->nc) ? c->nc : (c->opt.seed_corners > 0 ? c->opt.seed_corners : 1));
  const bool boxKind = c->kind == KIND_BOX_2D || c->kind == KIND_BOX_3D;
  const int64_t mLocal = A.aEnd - A.aBegin;
  if (!boxKind && mLocal > 0 && c->n >= 64 * mLocal) {
    const int64_t want = c->n / (4 * mLocal);
    const int S = (int)(want > 256 ? 256 : want);
    const int64_t total = mLocal * S;
    if ((s = ensure(c, c->seedPts, sizeof(double) * 3 * total))) return s;
    if ((s = ensure(c, c->seedNN, sizeof(int) * total))) return s;
    VD_LAUNCH(k_sample_points, blocks_for(total, kBlock, sm_count() * 8), kBlock, 0, st)(A, c->nc, S, c->seedPts.as<double>());
    if ((s = stage_nearest_points(c, c->seedPts.as<double>(), total, c->seedNN.as<int>()))) return s;
    VD_LAUNCH(k_seed_points, blocks_for(total, kBlock, sm_count() * 8), kBlock, 0, st)(A, S, c->seedPts.as<double>(), c->seedNN.as<int>());
  }
  if (boxKind) {
    double cv[8 * 3];
    cudaMemcpyAsync(cv, c->verts.p, sizeof(double) * 3 * c->nc, cudaMemcpyDeviceToHost, st);
    sync_stream(c);
    const double* lo = cv;
    const double* hi = cv + 3 * (c->nc - 1);
    VD_LAUNCH(k_seed_sites, blocks_for(c->n, kBlock, sm_count() * 8), kBlock, 0, st)(A, lo[0], lo[1], lo[2], hi[0], hi[1], hi[2]);
  }
  return cuda_check(c, cudaGetLastError(), "seed");
}

template <int KIND, bool HV>
static void launch_fast(vd_ctx* c, const ClipArgs& A, int64_t b, int64_t e, bool persist) {
  const int blocks = persist ? sm_count() * 3 : blocks_for(e - b, kWarpsPerBlock, sm_count() * 6);
  VD_LAUNCH((k_clip<KIND, false, HV>), blocks, kBlock, 0, c->stream)(A, nullptr, b, e, persist);
}

template <int KIND, bool HV>
static void launch_big(vd_ctx* c, const ClipArgs& A, int64_t ob, int64_t oe) {
  VD_LAUNCH((k_clip<KIND, true, HV>), blocks_for(oe - ob, 1, sm_count() * 8), kLanes, 0, c->stream)(A, A.ovf, ob, oe, false);
}

template <int KIND>
static void launch_kind(vd_ctx* c, const ClipArgs& A, bool hv, bool big, int64_t b, int64_t e, bool persist) {
  if (!big) { if (hv) launch_fast<KIND, true>(c, A, b, e, persist); else launch_fast<KIND, false>(c, A, b, e, persist); }
  else      { if (hv) launch_big<KIND, true>(c, A, b, e); else launch_big<KIND, false>(c, A, b, e); }
}

// one kernel per piece structure: triangles (both triangle kinds share the loop code), tets, rectangle, box
static void launch(vd_ctx* c, const ClipArgs& A, bool hv, bool big, int64_t b, int64_t e, bool persist) {
  switch (c->kind) {
    case KIND_TET_3D: launch_kind<KIND_TET_3D>(c, A, hv, big, b, e, persist); break;
    case KIND_BOX_3D: launch_kind<KIND_BOX_3D>(c, A, hv, big, b, e, persist); break;
    case KIND_BOX_2D: launch_kind<KIND_BOX_2D>(c, A, hv, big, b, e, persist); break;
    default:          launch_kind<KIND_TRI_2D>(c, A, hv, big, b, e, persist); break;
  }
}

static cudaError_t read_control(vd_ctx* c, Control& h) {
  static_assert(sizeof(Control) <= 1024, "fits the page-locked staging block");
  Control* dst = c->pinned ? reinterpret_cast<Control*>(c->pinned) : &h;
  cudaError_t e = cudaMemcpyAsync(dst, c->control.p, sizeof(Control), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = sync_stream(c);
  if (e == cudaSuccess && dst != &h) h = *dst;
  return e;
}

static void set_cursor(vd_ctx* c, int which, unsigned long long v) {
  cudaMemcpyAsync(&c->control.as<Control>()->fetch[which], &v, sizeof(v), cudaMemcpyHostToDevice, c->stream);
  sync_stream(c);   // v lives on the host stack
}

vd_status stage_clip(vd_ctx* c) {
  ClipArgs A = make_args(c);
  const int mode = c->opt.persistent;
  const bool solid = c->kind == KIND_TET_3D || c->kind == KIND_BOX_3D;
  const bool phased = solid && (mode == 1 || mode == 2);   // 3D kinds: one small kernel per step (vd_phase.cu)
  // otherwise the one-kernel form: a device-side queue (3), or one launch per wave (0; and the default of the triangle
  // kinds: with the discovery tuples and interior seeds their wavefronts are few, and the queue's polling costs more)
  const bool persist = !phased && (mode == 3 || (mode == 2 && !solid));
  A.queue = persist ? 1 : 0;
  int64_t begin = 0, obegin = 0, waves = 0;
  Control h;
  cudaError_t e = read_control(c, h);   // seeds pushed so far, refined cells of the index
  if (e != cudaSuccess) return cuda_check(c, e, "clip");
  const bool hv = h.nHeavy > 0;         // refined cells exist: the kernels that know the second index level
  for (;;) {
    if (h.err & (ERR_PAIR_CAP | ERR_VERT_CAP | ERR_NBR_CAP)) break;   // caller grows the pools and reruns
    if (h.err & (ERR_DUPLICATE | ERR_INPUT)) break;                   // bad sites (S1): nothing to clip
    int64_t end = (int64_t)h.pairTail, oend = (int64_t)h.ovfTail;
    if (end > c->pairCap) end = c->pairCap;
    if (oend > c->ovfCap) oend = c->ovfCap;
    if (end == begin && oend == obegin) break;   // "while L1 is not empty"
    if (end > begin && phased && end - begin >= (c->opt.small_wave == 0 ? kSmallWave : c->opt.small_wave)) {
      // phased mode: one small kernel per step of Alg. 3 over the whole wave (vd_phase.cu); a wave of a few thousand
      // pairs (the last wavefronts) takes the branch below instead: one launch and one counter read, not a dozen
      const vd_status s = run_phases(c, A, hv, begin, end);
      if (s != VD_OK) return s;
      ++waves;
    } else if (end > begin) {
      // wave mode: one launch per wavefront.  persistent mode: the kernel drains the queue as it grows
      set_cursor(c, 0, persist ? (unsigned long long)begin : 0ull);
      launch(c, A, hv, false, persist ? 0 : begin, end, persist);
      ++waves;
    } else if (oend > obegin) {
      set_cursor(c, 1, 0ull);
      launch(c, A, hv, true, obegin, oend, false);
      obegin = oend;
    }
    if ((e = read_control(c, h)) != cudaSuccess) return cuda_check(c, e, "clip wave");
    if (end > begin) begin = persist ? (int64_t)h.finished : end;
  }
  c->hostControl = h;
  c->counters.waves = waves;
  return cuda_check(c, cudaGetLastError(), "clip");
}

}  // namespace vd
