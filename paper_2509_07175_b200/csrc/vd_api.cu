// vd_api.cu -- the C ABI of include/vd.h: argument marshalling, memory, the stage sequence of
// vd_compute and the pool-growth / rerun policy.  No geometry happens on the host.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include <nvtx3/nvToolsExt.h>   // header-only: ranges cost nothing unless a profiler is attached

#include "vd_internal.h"

namespace vd {

unsigned long long g_launches = 0;

int sm_count() {
  static int cached[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { cudaGetLastError(); return 148; }
  if (cached[dev] == 0) {
    int v = 0;
    if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || v < 1) { cudaGetLastError(); v = 148; }
    cached[dev] = v;
  }
  return cached[dev];
}

cudaError_t sync_stream(vd_ctx* c, const char* why) {
  c->syncs += 1;
  static const bool trace = getenv("VD_TRACE_SYNC") != nullptr;
  if (trace) fprintf(stderr, "vd sync %lld: %s\n", (long long)c->syncs, why ? why : "?");
  return cudaStreamSynchronize(c->stream);
}

void phase_mark(vd_ctx* c, int kind) {
  if (c->evUsed == (int)c->evPool.size()) {
    cudaEvent_t e = nullptr;
    if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); return; }
    c->evPool.push_back(e);
    c->evKind.push_back(-1);
  }
  c->evKind[c->evUsed] = kind;
  cudaEventRecord(c->evPool[c->evUsed], c->stream);
  c->evUsed += 1;
}

void phase_marks_collect(vd_ctx* c) {
  for (int k = 0; k + 1 < c->evUsed; ++k) {
    if (c->evKind[k] < 0) continue;
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, c->evPool[k], c->evPool[k + 1]) == cudaSuccess) c->phaseMs[c->evKind[k]] += ms;
    else cudaGetLastError();
  }
  c->evUsed = 0;
}

vd_status cuda_check(vd_ctx* c, cudaError_t e, const char* what) {
  if (e == cudaSuccess) return VD_OK;
  if (c) c->lastError = std::string(what) + ": " + cudaGetErrorString(e);
  return e == cudaErrorMemoryAllocation ? VD_E_NOMEM : VD_E_CUDA;
}

// Device memory comes from the stream-ordered allocator (cudaMallocAsync) with the default pool told to keep what is
// freed: creating and destroying contexts in a loop (bench.py's end-to-end leg, a Lloyd driver that rebuilds its
// context) then costs no cudaMalloc / cudaFree of multi-GB pools after the first round.  vd_set_allocator overrides it.
static void keep_freed_memory_in_pool() {
  static bool done[64] = {};
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64 || done[dev]) return;
  cudaMemPool_t pool;
  if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
    unsigned long long keep = ~0ull;
    cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
  }
  cudaGetLastError();
  done[dev] = true;
}

void release(vd_ctx* c, DevBuf& b) {
  if (!b.p) return;
  if (b.hooked && c->freeFn) c->freeFn(b.p, c->allocUser);
  else if (cudaFreeAsync(b.p, c->stream) != cudaSuccess) { cudaGetLastError(); cudaFree(b.p); }
  b.p = nullptr;
  b.cap = 0;
  b.hooked = false;
}

vd_status ensure(vd_ctx* c, DevBuf& b, size_t bytes) {
  if (bytes < 256) bytes = 256;
  if (b.cap >= bytes) return VD_OK;
  // a buffer that grows again gets a quarter of slack: the assemble stage sizes its buffers from pool cursors that differ
  // by a few entries from run to run, and re-allocating a gigabyte for them costs hundreds of milliseconds
  if (b.p) bytes += bytes / 4;
  else if (bytes > ((size_t)1 << 20)) bytes += bytes / 8;   // (large buffers: also the first time)
  // pending kernels may still use the old block
  if (b.p) sync_stream(c, "buffer grows");
  release(c, b);
  void* p = nullptr;
  if (c->allocFn) {
    p = c->allocFn(bytes, c->allocUser, (void*)c->stream);
    if (!p) { c->lastError = "allocator hook returned NULL"; return VD_E_NOMEM; }
    b.hooked = true;
  } else {
    cudaError_t e = cudaMallocAsync(&p, bytes, c->stream);
    if (e != cudaSuccess) { cudaGetLastError(); e = cudaMalloc(&p, bytes); }
    if (e != cudaSuccess) { cudaGetLastError(); c->lastError = "device memory allocation failed"; return VD_E_NOMEM; }
  }
  b.p = p;
  b.cap = bytes;
  return VD_OK;
}

// [n][dim] (host or device) -> device [n][3], z = 0 for dim 2; flags non-finite values
__global__ void __launch_bounds__(kBlock) k_pad3(const double* __restrict__ in, int64_t n, int dim, double* __restrict__ out, unsigned int* err) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    bool bad = false;
    for (int a = 0; a < 3; ++a) {
      const double v = a < dim ? in[i * dim + a] : 0.0;
      if (!(v == v) || fabs(v) > 1e150) bad = true;
      out[i * 3 + a] = v;
    }
    if (bad) atomicOr(err, ERR_INPUT);
  }
}

static vd_status upload_points(vd_ctx* c, const double* src, int64_t n, int dim, DevBuf& dst, const char* what) {
  vd_status s;
  DevBuf tmp;
  if ((s = ensure(c, dst, sizeof(double) * 3 * n))) return s;
  if ((s = ensure(c, tmp, sizeof(double) * dim * n))) return s;
  if ((s = ensure(c, c->control, sizeof(Control)))) { release(c, tmp); return s; }
  cudaError_t e = cudaMemcpyAsync(tmp.p, src, sizeof(double) * dim * n, cudaMemcpyDefault, c->stream);
  if (e != cudaSuccess) { release(c, tmp); return cuda_check(c, e, what); }
  cudaMemsetAsync(c->control.p, 0, sizeof(Control), c->stream);
  int blocks = (int)((n + kBlock - 1) / kBlock);
  if (blocks > sm_count() * 16) blocks = sm_count() * 16;
  VD_LAUNCH(k_pad3, blocks, kBlock, 0, c->stream)(tmp.as<double>(), n, dim, dst.as<double>(), &c->control.as<Control>()->err);
  Control h;
  e = cudaMemcpyAsync(&h, c->control.p, sizeof(Control), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  release(c, tmp);
  if (e != cudaSuccess) return cuda_check(c, e, what);
  if (h.err & ERR_INPUT) { c->lastError = std::string(what) + ": non-finite coordinate"; return VD_E_INPUT; }
  return VD_OK;
}

// Lloyd step ("we compute centroids of Voronoi cells as the new sites"): empty cells keep their site
__global__ void __launch_bounds__(kBlock) k_move_sites(const double* __restrict__ measure, const double* __restrict__ centroid,
                                                        int64_t n, int dim, double* __restrict__ sites3) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    if (measure[i] > 0.0)
      for (int a = 0; a < dim; ++a) sites3[i * 3 + a] = centroid[i * dim + a];
  }
}

// Lloyd iterations, whole-cell kinds (vd_options.reuse_nbrs): the neighbours of cell i in this iteration are the
// first clips of its cell in the next one -- sites move little between iterations, so nearly all of them bound the new cell
// too, and any B_ij is a valid clip of Omega_i anyway (Eq. 1; reading U19).  Up to K of them per site, nearest first (the
// clips of near sites shrink the polytope fastest), -1 padded; replaces the nearest-site lookup of k_near.
__global__ void __launch_bounds__(kBlock) k_near_from_nbrs(const int64_t* __restrict__ nbrOff, const int* __restrict__ nbr,
                                                            const double* __restrict__ sites3, int64_t n, int K, int* __restrict__ list) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const double x = sites3[i * 3 + 0], y = sites3[i * 3 + 1], z = sites3[i * 3 + 2];
    int ids[32];
    double ds[32];
    int cnt = 0;
    for (int64_t k = nbrOff[i]; k < nbrOff[i + 1]; ++k) {
      const int j = nbr[k];
      const double dx = sites3[(int64_t)j * 3 + 0] - x, dy = sites3[(int64_t)j * 3 + 1] - y, dz = sites3[(int64_t)j * 3 + 2] - z;
      const double d2 = dx * dx + dy * dy + dz * dz;
      int t = cnt < K ? cnt++ : K;          // insertion into the K nearest so far
      if (t == K) { if (!(d2 < ds[K - 1])) continue; t = K - 1; }
      while (t > 0 && ds[t - 1] > d2) { ds[t] = ds[t - 1]; ids[t] = ids[t - 1]; --t; }
      ds[t] = d2; ids[t] = j;
    }
    for (int t = 0; t < K; ++t) list[i * K + t] = t < cnt ? ids[t] : -1;
  }
}

__global__ void __launch_bounds__(kBlock) k_unpad3(const double* __restrict__ in3, int64_t n, int dim, double* __restrict__ out) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
    for (int a = 0; a < dim; ++a) out[i * dim + a] = in3[i * 3 + a];
}

// Power diagrams by lifting (section VII-C): p_i = (v_i, sqrt(eta - w_i)), eta >= max w.  Partial maxima
// of the weights, then the lift itself.  dim 2: the lifted coordinate becomes z of the 3-wide site record; dim 3: the
// fourth coordinate only ever enters a squared distance from the domain (height 0), as h_i^2 = eta - w_i: that additive
// term is what is stored (siteW).
__global__ void __launch_bounds__(kBlock) k_weight_max(const double* __restrict__ w, int64_t n, double* __restrict__ part, unsigned int* err) {
  double mx = -1e300;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const double v = w[i];
    if (!(v == v) || fabs(v) > 1e150) atomicOr(err, ERR_WEIGHT);
    mx = fmax(mx, v);
  }
  for (int off = kLanes / 2; off > 0; off >>= 1) mx = fmax(mx, __shfl_xor_sync(kFull, mx, off));
  __shared__ double sm[kWarpsPerBlock];
  if (lane_id() == 0) sm[threadIdx.x / kLanes] = mx;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int k = 1; k < (int)blockDim.x / kLanes; ++k) mx = fmax(mx, sm[k]);
    part[blockIdx.x] = mx;
  }
}

__global__ void __launch_bounds__(kBlock) k_lift(const double* __restrict__ w, int64_t n, int dim, const double* __restrict__ part, int nparts,
                                                  double eta, double* __restrict__ sites3, double* __restrict__ siteW, unsigned int* err) {
  double wmax = -1e300;
  for (int k = 0; k < nparts; ++k) wmax = fmax(wmax, part[k]);
  if (!(eta == eta)) eta = wmax;                    // NaN: the smallest admissible eta
  if (eta < wmax) { if (blockIdx.x == 0 && threadIdx.x == 0) atomicOr(err, ERR_WEIGHT); return; }
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const double h2 = eta - w[i];
    if (dim == 2) sites3[i * 3 + 2] = sqrt(h2);
    else siteW[i] = h2;
  }
}

// Sharded runs: the additive per-cell quantities (measure, measure x centroid), and the way back (vd.h)
__global__ void __launch_bounds__(kBlock) k_partial_moments(const double* __restrict__ measure, const double* __restrict__ centroid, int64_t n,
                                                             int dim, double* __restrict__ out) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const double ms = measure[i];
    out[i * (dim + 1)] = ms;
    for (int a = 0; a < dim; ++a) out[i * (dim + 1) + 1 + a] = ms * centroid[i * dim + a];
  }
}

__global__ void __launch_bounds__(kBlock) k_finish_centroids(const double* __restrict__ sums, const double* __restrict__ sites3, int64_t n, int dim,
                                                              double* __restrict__ measure, double* __restrict__ centroid) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const double ms = sums[i * (dim + 1)];
    measure[i] = ms;
    for (int a = 0; a < dim; ++a) centroid[i * dim + a] = ms > 0.0 ? sums[i * (dim + 1) + 1 + a] / ms : sites3[i * 3 + a];
  }
}

static void set_default_options(vd_options& o) {
  memset(&o, 0, sizeof(o));
  o.grid_density = 2.0;
  o.real_edges = 1;
  o.persistent = 1;
}

static int64_t next_pow2(int64_t v) {
  int64_t p = 1;
  while (p < v) p <<= 1;
  return p;
}

static vd_status alloc_pools(vd_ctx* c) {
  vd_status s;
  c->hashCap = next_pow2(2 * c->pairCap);
  c->ovfCap = c->pairCap;
  if ((s = ensure(c, c->pairs, sizeof(Pair) * c->pairCap))) return s;
  if ((s = ensure(c, c->pieces, sizeof(Piece) * c->pairCap))) return s;
  if ((s = ensure(c, c->visited, sizeof(unsigned long long) * c->hashCap))) return s;
  if ((s = ensure(c, c->ovf, sizeof(int) * c->ovfCap))) return s;
  if ((s = ensure(c, c->poolXYZ, sizeof(double) * 3 * c->vertCap))) return s;
  if ((s = ensure(c, c->poolFlags, sizeof(int) * c->nfl * c->vertCap))) return s;
  if ((s = ensure(c, c->poolNbr, sizeof(int) * c->nbrCap))) return s;
  if ((s = ensure(c, c->sitePieces, sizeof(int) * c->n))) return s;
  if ((s = ensure(c, c->siteNbrRaw, sizeof(int) * c->n))) return s;
  return VD_OK;
}

}  // namespace vd

using namespace vd;

extern "C" {

const char* vd_version(void) { return "vd-b200 0.1 (sm_100a, fp64)"; }

const char* vd_last_error(const vd_ctx* ctx) { return ctx ? ctx->lastError.c_str() : "null context"; }

vd_status vd_create(const double* sites, int64_t n, int dim, vd_ctx** out) {
  if (!sites || !out || n < 1) return VD_E_ARG;
  if (dim != 2 && dim != 3) return VD_E_DIM;
  if (n > 0x7fffffff) return VD_E_ARG;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return VD_E_CUDA; }
  keep_freed_memory_in_pool();
  vd_ctx* c = new (std::nothrow) vd_ctx();
  if (!c) return VD_E_NOMEM;
  c->n = n;
  c->dim = dim;
  set_default_options(c->opt);
  for (int k = 0; k < 6; ++k) cudaEventCreate(&c->ev[k]);
  if (cudaMallocHost(&c->pinned, 1024) != cudaSuccess) { cudaGetLastError(); c->pinned = nullptr; }
  const vd_status s = upload_points(c, sites, n, dim, c->sites, "vd_create");
  if (s != VD_OK) { vd_destroy(c); return s; }
  *out = c;
  return VD_OK;
}

vd_status vd_create_weighted(const double* sites, const double* weights, int64_t n, int dim, double eta, vd_ctx** out) {
  if (!weights || !out) return VD_E_ARG;
  vd_ctx* c = nullptr;
  vd_status s = vd_create(sites, n, dim, &c);
  if (s != VD_OK) return s;
  c->weighted = true;
  DevBuf w, part;
  const int blocks = (int)((n + kBlock - 1) / kBlock) < 256 ? (int)((n + kBlock - 1) / kBlock) : 256;
  if ((s = ensure(c, w, sizeof(double) * n)) || (s = ensure(c, part, sizeof(double) * 256)) ||
      (dim == 3 && (s = ensure(c, c->siteW, sizeof(double) * n)))) { vd_destroy(c); return s; }
  cudaError_t e = cudaMemcpyAsync(w.p, weights, sizeof(double) * n, cudaMemcpyDefault, c->stream);
  cudaMemsetAsync(c->control.p, 0, sizeof(Control), c->stream);
  unsigned int* err = &c->control.as<Control>()->err;
  VD_LAUNCH(k_weight_max, blocks, kBlock, 0, c->stream)(w.as<double>(), n, part.as<double>(), err);
  VD_LAUNCH(k_lift, blocks, kBlock, 0, c->stream)(w.as<double>(), n, dim, part.as<double>(), blocks, eta, c->sites.as<double>(),
                                                  c->siteW.as<double>(), err);
  Control h;
  if (e == cudaSuccess) e = cudaMemcpyAsync(&h, c->control.p, sizeof(Control), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  release(c, w);
  release(c, part);
  if (e != cudaSuccess) { vd_destroy(c); return VD_E_CUDA; }
  if (h.err & ERR_WEIGHT) { vd_destroy(c); return VD_E_INPUT; }
  *out = c;
  return VD_OK;
}

vd_status vd_partial_moments(vd_ctx* c, double* out_sums) {
  if (!c || !out_sums) return VD_E_ARG;
  if (!c->haveResult) { c->lastError = "vd_partial_moments before a successful vd_compute"; return VD_E_STATE; }
  int blocks = (int)((c->n + kBlock - 1) / kBlock);
  if (blocks > sm_count() * 16) blocks = sm_count() * 16;
  VD_LAUNCH(k_partial_moments, blocks, kBlock, 0, c->stream)(c->oMeasure.as<double>(), c->oCentroid.as<double>(), c->n, c->dim, out_sums);
  return cuda_check(c, cudaGetLastError(), "vd_partial_moments");
}

vd_status vd_finish_centroids(vd_ctx* c, const double* sums) {
  if (!c || !sums) return VD_E_ARG;
  if (!c->haveResult) { c->lastError = "vd_finish_centroids before a successful vd_compute"; return VD_E_STATE; }
  int blocks = (int)((c->n + kBlock - 1) / kBlock);
  if (blocks > sm_count() * 16) blocks = sm_count() * 16;
  VD_LAUNCH(k_finish_centroids, blocks, kBlock, 0, c->stream)(sums, c->sites.as<double>(), c->n, c->dim, c->oMeasure.as<double>(),
                                                              c->oCentroid.as<double>());
  return cuda_check(c, cudaGetLastError(), "vd_finish_centroids");
}

vd_status vd_update_sites(vd_ctx* c, const double* sites) {
  if (!c || !sites) return VD_E_ARG;
  if (c->weighted) { c->lastError = "vd_update_sites: a weighted context keeps its lifted sites (create a new one)"; return VD_E_STATE; }
  c->indexValid = false;
  c->heavyKnown = -1;
  c->haveResult = false;
  return upload_points(c, sites, c->n, c->dim, c->sites, "vd_update_sites");
}

vd_status vd_set_domain(vd_ctx* c, const double* verts, int64_t nv, const int32_t* simplices, int64_t m, vd_domain_kind kind) {
  const bool box = kind == VD_BOX_2D || kind == VD_BOX_3D;
  if (!c || !verts || (!simplices && !box) || nv < 1 || m < 1) return VD_E_ARG;
  if (kind < VD_TRI_2D || kind > VD_BOX_3D) return VD_E_ARG;
  if ((kind == VD_TRI_2D || kind == VD_BOX_2D) != (c->dim == 2)) return VD_E_DIM;
  if (c->weighted && (kind == VD_BOX_2D || kind == VD_TRI_SURFACE)) {
    c->lastError = "vd_set_domain: weighted sites take VD_TRI_2D (dim 2) or VD_TET_3D / VD_BOX_3D (dim 3)";
    return VD_E_DIM;
  }
  // weighted 2D sites were lifted to R^3 (vd_create_weighted): the triangles, at height 0, are a surface in R^3
  if (c->weighted && kind == VD_TRI_2D) kind = VD_TRI_SURFACE;
  if (m > 0x3fffffff || nv > 0x7fffffff) return VD_E_ARG;
  if (box && (nv != 2 || m != 1)) return VD_E_ARG;
  c->haveDomain = false;
  c->haveResult = false;
  dissolve_release(c);
  c->kind = (int)kind;
  const bool solid = kind == VD_TET_3D || kind == VD_BOX_3D;
  c->nc = kind == VD_BOX_3D ? 8 : ((kind == VD_TET_3D || kind == VD_BOX_2D) ? 4 : 3);
  c->nfl = solid ? 3 : 2;
  c->m = m;
  vd_status s;
  if (box) {
    // simple domain (section V-B): expand (lo, hi) into the 4 / 8 corners; they are the "mesh vertices" whose
    // nearest sites seed the pair list and classify the corners; corner c = bits (x, y, z)
    double lh[6] = {0, 0, 0, 0, 0, 0};
    cudaError_t e = cudaMemcpyAsync(lh, verts, sizeof(double) * 2 * c->dim, cudaMemcpyDefault, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_check(c, e, "vd_set_domain");
    const int dim = c->dim, ncorner = c->nc;
    double cv[8 * 3];
    int32_t ids[8], adj[8];
    for (int k = 0; k < ncorner; ++k) {
      for (int a = 0; a < dim; ++a) {
        const double lo = lh[a], hi = lh[dim + a];
        if (!(hi > lo)) { c->lastError = "vd_set_domain: empty box"; return VD_E_INPUT; }
        cv[k * dim + a] = ((k >> a) & 1) ? hi : lo;
      }
      ids[k] = k;
      adj[k] = (int32_t)m;
    }
    c->nv = ncorner;
    if ((s = upload_points(c, cv, ncorner, dim, c->verts, "vd_set_domain"))) return s;
    if ((s = ensure(c, c->simp, sizeof(int) * ncorner))) return s;
    if ((s = ensure(c, c->adj, sizeof(int) * ncorner))) return s;
    e = cudaMemcpyAsync(c->simp.p, ids, sizeof(int) * ncorner, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->adj.p, adj, sizeof(int) * ncorner, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_check(c, e, "vd_set_domain");
    c->haveDomain = true;
    return VD_OK;
  }
  c->nv = nv;
  s = upload_points(c, verts, nv, c->dim, c->verts, "vd_set_domain");
  if (s != VD_OK) return s;
  if ((s = ensure(c, c->simp, sizeof(int) * m * c->nc))) return s;
  cudaError_t e = cudaMemcpyAsync(c->simp.p, simplices, sizeof(int) * m * c->nc, cudaMemcpyDefault, c->stream);
  if (e != cudaSuccess) return cuda_check(c, e, "vd_set_domain");
  if ((s = stage_domain(c))) return s;
  c->haveDomain = true;
  return VD_OK;
}

vd_status vd_compute(vd_ctx* c, vd_cells* out) {
  if (!c || !out) return VD_E_ARG;
  if (!c->haveDomain) { c->lastError = "vd_compute before vd_set_domain"; return VD_E_STATE; }
  c->haveResult = false;
  if (c->opt.dissolve > 0) {
    // Alg. 5's site division: convex tet meshes only
    if (c->kind != VD_TET_3D || c->weighted || c->opt.simplex_end > 0) {
      c->lastError = "vd_compute: vd_options.dissolve takes VD_TET_3D, unweighted sites, the whole mesh";
      return VD_E_ARG;
    }
    if (!c->dissolveReady) {
      const vd_status sd = stage_dissolve_prepare(c);
      if (sd != VD_OK) return sd;
    }
  }
  if (c->pairCap == 0) {
    // pairs = pieces: a simplex meets ~2-20 cells in the paper-like workloads; corners ~11 per 3D piece.
    // Underestimates are repaired by doubling and rerunning (counters.reruns)
    const int64_t est = 16 * c->m + 2 * c->n;
    c->pairCap = c->opt.pair_capacity > 0 ? c->opt.pair_capacity : (est + 6 * c->n + (1 << 16));
    c->vertCap = c->opt.vert_capacity > 0 ? c->opt.vert_capacity : (14 * est + (1 << 16));
    c->nbrCap = 8 * est + (1 << 16);
    if (c->kind == VD_BOX_2D || c->kind == VD_BOX_3D) {
      // whole cells: one pair per site; a Poisson-Voronoi cell has 6 corners / edges in 2D, ~27.1 corners and
      // ~15.5 faces in 3D on average
      const bool solid = c->kind == VD_BOX_3D;
      c->pairCap = c->opt.pair_capacity > 0 ? c->opt.pair_capacity : (2 * c->n + (1 << 16));
      c->vertCap = c->opt.vert_capacity > 0 ? c->opt.vert_capacity : ((solid ? 32 : 8) * c->n + (1 << 16));
      c->nbrCap = (solid ? 20 : 8) * c->n + (1 << 16);
    }
  }
  memset(&c->counters, 0, sizeof(c->counters));
  c->syncs = 0;
  const unsigned long long launches0 = g_launches;
  cudaStream_t st = c->stream;
  vd_status s;
  for (int attempt = 0;; ++attempt) {
    for (double& v : c->phaseMs) v = 0.0;
    if ((s = alloc_pools(c))) return s;
    if ((s = ensure(c, c->control, sizeof(Control)))) return s;
    cudaMemsetAsync(c->control.p, 0, sizeof(Control), st);
    // NVTX ranges per stage: host-side brackets of where each stage is enqueued / waited for
    struct Range { explicit Range(const char* name) { nvtxRangePushA(name); } ~Range() { nvtxRangePop(); } };
    cudaEventRecord(c->ev[0], st);
    { Range r("vd S1 site index"); if ((s = stage_index(c))) return s; }
    cudaEventRecord(c->ev[1], st);
    // the full kernels only where a feature they alone carry is in use (header of vd_clip.cu)
    const bool ext = (c->weighted && c->dim == 3) || c->opt.step_out > 0 || c->opt.count_alg > 0 || c->opt.fp32_filter > 0;
    { Range r("vd S3 seeds"); if ((s = ext ? full::stage_seed(c) : lean::stage_seed(c))) return s; }
    cudaEventRecord(c->ev[2], st);
    { Range r("vd S4+S5 clip and propagate"); if ((s = ext ? full::stage_clip(c) : lean::stage_clip(c))) return s; }
    cudaEventRecord(c->ev[3], st);
    const unsigned err = c->hostControl.err;
    if (err & (ERR_PAIR_CAP | ERR_VERT_CAP | ERR_NBR_CAP)) {
      if (attempt >= 6) { c->lastError = "vd_compute: pools still too small after 6 regrowths"; return VD_E_CAPACITY; }
      if (err & ERR_PAIR_CAP) c->pairCap *= 2;
      if (err & ERR_VERT_CAP) c->vertCap *= 2;
      if (err & ERR_NBR_CAP) c->nbrCap *= 2;
      c->counters.reruns += 1;
      continue;
    }
    if (err & ERR_DUPLICATE) { c->lastError = "vd_compute: two sites have the same coordinates"; return VD_E_INPUT; }
    if (err & ERR_INPUT) { c->lastError = "vd_compute: non-finite site coordinate"; return VD_E_INPUT; }
    if (err & ERR_PIECE_CAP) { c->lastError = "vd_compute: a piece outgrew the large-capacity path"; return VD_E_CAPACITY; }
    if (err & (ERR_NOCONVERGE | ERR_TOPOLOGY)) {
      c->lastError = (err & ERR_NOCONVERGE) ? "vd_compute: bisector search hit its iteration cap (degenerate input?)"
                                            : "vd_compute: clip produced a non-simple rim (degenerate input?)";
      return VD_E_NOCONVERGE;
    }
    break;
  }
  nvtxRangePushA("vd S6 assemble");
  s = stage_assemble(c);
  nvtxRangePop();
  if (s) return s;
  cudaEventRecord(c->ev[4], st);
  Control h;
  cudaError_t e = cudaMemcpyAsync(&h, c->control.p, sizeof(Control), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = sync_stream(c, "totals");
  if (e != cudaSuccess) return cuda_check(c, e, "vd_compute");
  c->hostControl = h;
  float ms = 0;
  for (int k = 0; k < 4; ++k) { cudaEventElapsedTime(&ms, c->ev[k], c->ev[k + 1]); c->stageMs[k] = ms; }
  cudaEventElapsedTime(&ms, c->ev[0], c->ev[4]);
  c->stageMs[4] = ms;
  const int64_t reruns = c->counters.reruns, waves = c->counters.waves;
  auto fill = [](vd_counters& o, const Counters& k) {
    o.pairs = (int64_t)k.pairs; o.pieces = (int64_t)k.pieces; o.queries = (int64_t)k.queries; o.dist_evals = (int64_t)k.dist_evals;
    o.row_evals = (int64_t)k.rows; o.search_iters = (int64_t)k.search_iters; o.clips = (int64_t)k.clips;
    o.search_evals = (int64_t)k.search_evals; o.pre_clips = (int64_t)k.pre_clips; o.clip_corners = (int64_t)k.clip_corners;
    o.new_corners = (int64_t)k.new_corners; o.fan_simplices = (int64_t)k.fan_simplices; o.alg_evals = (int64_t)k.alg_evals;
    o.step_probes = (int64_t)k.step_probes; o.f32_survivors = (int64_t)k.f32_survivors;
  };
  fill(c->counters, counters_total(h));
  for (int k = 0; k < kCntKinds; ++k) { memset(&c->phaseCounters[k], 0, sizeof(vd_counters)); fill(c->phaseCounters[k], h.cnt[k]); }
  c->counters.syncs = c->syncs;
  c->counters.overflow_pairs = (int64_t)h.ovfTail;
  c->counters.reruns = reruns; c->counters.waves = waves;
  c->counters.launches = (int64_t)(g_launches - launches0);
  vd_cells& r = c->cells;
  r.n = c->n; r.dim = c->dim; r.nfl = c->nfl;
  r.n_nonempty = (int64_t)h.nNonEmpty; r.n_pieces = (int64_t)h.nPieces; r.n_verts = (int64_t)h.nVerts; r.n_nbrs = (int64_t)h.nNbrs;
  r.measure = c->oMeasure.as<double>(); r.centroid = c->oCentroid.as<double>();
  r.nbr_off = c->oNbrOff.as<int64_t>(); r.nbr = c->oNbr.as<int32_t>();
  r.piece_off = c->oPieceOff.as<int64_t>(); r.piece_simplex = c->oPieceSimplex.as<int32_t>();
  r.piece_measure = c->oPieceMeasure.as<double>();
  r.vert_off = c->oVertOff.as<int64_t>(); r.vert_xyz = c->oVertXYZ.as<double>(); r.vert_flags = c->oVertFlags.as<int32_t>();
  *out = r;
  c->haveResult = true;
  return VD_OK;
}

vd_status vd_lloyd(vd_ctx* c, int iterations, vd_cells* out, double* sites_out) {
  if (!c || !out || iterations < 0) return VD_E_ARG;
  vd_status s;
  int blocks = (int)((c->n + kBlock - 1) / kBlock);
  if (blocks > sm_count() * 16) blocks = sm_count() * 16;
  for (int it = 0; it < iterations; ++it) {
    if ((s = vd_compute(c, out))) return s;
    if (c->opt.reuse_nbrs >= 0 && c->kind == VD_BOX_3D && !c->weighted && c->nearList.p) {
      const int K = c->nearK;   // the width the clip kernels read the list with
      if (K > 0) {
        VD_LAUNCH(k_near_from_nbrs, blocks, kBlock, 0, c->stream)(c->oNbrOff.as<int64_t>(), c->oNbr.as<int>(), c->sites.as<double>(), c->n, K,
                                                                  c->nearList.as<int>());
        c->nearReady = true;
      }
    }
    VD_LAUNCH(k_move_sites, blocks, kBlock, 0, c->stream)(c->oMeasure.as<double>(), c->oCentroid.as<double>(), c->n, c->dim,
                                                         c->sites.as<double>());
    c->indexValid = false;
  c->heavyKnown = -1;
  }
  if ((s = vd_compute(c, out))) return s;
  if (sites_out) {
    DevBuf tmp;
    if ((s = ensure(c, tmp, sizeof(double) * c->n * c->dim))) return s;
    VD_LAUNCH(k_unpad3, blocks, kBlock, 0, c->stream)(c->sites.as<double>(), c->n, c->dim, tmp.as<double>());
    cudaError_t e = cudaMemcpyAsync(sites_out, tmp.p, sizeof(double) * c->n * c->dim, cudaMemcpyDefault, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    release(c, tmp);
    if (e != cudaSuccess) return cuda_check(c, e, "vd_lloyd");
  }
  return cuda_check(c, cudaGetLastError(), "vd_lloyd");
}

void vd_destroy(vd_ctx* c) {
  if (!c) return;
  dissolve_release(c);
  cudaStreamSynchronize(c->stream);
  DevBuf* all[] = {&c->sites, &c->verts, &c->simp, &c->adj, &c->grid, &c->bbox, &c->cellOf, &c->cellStart, &c->cellFill,
                   &c->scanTmp, &c->sorted32, &c->sortKeys, &c->sortVals, &c->sortHist, &c->delta, &c->siteW, &c->sortedW, &c->bTris, &c->bTet, &c->bPlanes, &c->boxVerts, &c->boxVnn, &c->heavyFlag, &c->heavyPrefix, &c->subNeed, &c->subOffRaw, &c->subOff, &c->subCount, &c->subStart,
                   &c->sorted2, &c->vnn, &c->nearList, &c->nearAuto, &c->phaseCells, &c->phaseLists, &c->control, &c->pairs, &c->pieces, &c->visited, &c->ovf, &c->poolXYZ, &c->poolFlags,
                   &c->poolNbr, &c->siteList, &c->seedPts, &c->seedNN, &c->sitePieces, &c->siteNbrRaw, &c->siteFill, &c->order, &c->nbrRawOff, &c->nbrRaw, &c->nbrCnt,
                   &c->vcount, &c->oMeasure, &c->oCentroid, &c->oNbrOff, &c->oNbr, &c->oPieceOff, &c->oPieceSimplex,
                   &c->oPieceMeasure, &c->oVertOff, &c->oVertXYZ, &c->oVertFlags};
  for (DevBuf* b : all) release(c, *b);
  for (int k = 0; k < 6; ++k)
    if (c->ev[k]) cudaEventDestroy(c->ev[k]);
  for (cudaEvent_t e : c->evPool) cudaEventDestroy(e);
  if (c->pinned) cudaFreeHost(c->pinned);
  delete c;
}

vd_status vd_set_stream(vd_ctx* c, void* stream) {
  if (!c) return VD_E_ARG;
  cudaStreamSynchronize(c->stream);
  c->stream = (cudaStream_t)stream;
  return VD_OK;
}

vd_status vd_set_allocator(vd_ctx* c, void* (*alloc)(size_t, void*, void*), void (*rel)(void*, void*), void* user) {
  if (!c || ((alloc == nullptr) != (rel == nullptr))) return VD_E_ARG;
  if (c->pairs.p || c->sorted2.p) { c->lastError = "vd_set_allocator must be called before the first vd_compute"; return VD_E_STATE; }
  c->allocFn = alloc; c->freeFn = rel; c->allocUser = user;
  return VD_OK;
}

vd_status vd_set_options(vd_ctx* c, const vd_options* o) {
  if (!c || !o) return VD_E_ARG;
  vd_options d;
  set_default_options(d);
  c->opt = *o;
  c->heavyKnown = -1;
  if (!(c->opt.grid_density > 0)) c->opt.grid_density = d.grid_density;
  if (c->opt.real_edges < 0) c->opt.real_edges = d.real_edges;
  if (c->opt.persistent < 0) c->opt.persistent = d.persistent;
  if (c->opt.simplex_begin < 0 || c->opt.simplex_end < 0 || (c->opt.simplex_end > 0 && c->opt.simplex_begin > c->opt.simplex_end)) {
    c->opt.simplex_begin = c->opt.simplex_end = 0;
    c->lastError = "vd_set_options: bad simplex range";
    return VD_E_ARG;
  }
  return VD_OK;
}

vd_status vd_get_counters(const vd_ctx* c, vd_counters* out) {
  if (!c || !out) return VD_E_ARG;
  *out = c->counters;
  return VD_OK;
}

vd_status vd_get_phase_counters(const vd_ctx* c, int which, vd_counters* out) {
  if (!c || !out || which < 0 || which >= kCntKinds) return VD_E_ARG;
  *out = c->phaseCounters[which];
  return VD_OK;
}

vd_status vd_get_phase_ms(const vd_ctx* c, double out_ms[5]) {
  if (!c || !out_ms) return VD_E_ARG;
  for (int k = 0; k < 5; ++k) out_ms[k] = c->phaseMs[k];
  return VD_OK;
}

vd_status vd_get_stage_ms(const vd_ctx* c, double out_ms[5]) {
  if (!c || !out_ms) return VD_E_ARG;
  for (int k = 0; k < 5; ++k) out_ms[k] = c->stageMs[k];
  return VD_OK;
}

#define VD_COPY(dst, src, bytes)                                                                          \
  if ((dst) && (bytes) > 0) {                                                                             \
    const cudaError_t e_ = cudaMemcpyAsync((dst), (src), (bytes), cudaMemcpyDefault, c->stream);          \
    if (e_ != cudaSuccess) return cuda_check(c, e_, "vd_cells_to_host");                                  \
  }

vd_status vd_cells_to_host(vd_ctx* c, double* measure, double* centroid, int64_t* nbr_off, int32_t* nbr, int64_t* piece_off,
                           int32_t* piece_simplex, double* piece_measure, int64_t* vert_off, double* vert_xyz, int32_t* vert_flags) {
  if (!c) return VD_E_ARG;
  if (!c->haveResult) { c->lastError = "vd_cells_to_host before a successful vd_compute"; return VD_E_STATE; }
  const vd_cells& r = c->cells;
  VD_COPY(measure, r.measure, sizeof(double) * r.n);
  VD_COPY(centroid, r.centroid, sizeof(double) * r.n * r.dim);
  VD_COPY(nbr_off, r.nbr_off, sizeof(int64_t) * (r.n + 1));
  VD_COPY(nbr, r.nbr, sizeof(int32_t) * r.n_nbrs);
  VD_COPY(piece_off, r.piece_off, sizeof(int64_t) * (r.n + 1));
  VD_COPY(piece_simplex, r.piece_simplex, sizeof(int32_t) * r.n_pieces);
  VD_COPY(piece_measure, r.piece_measure, sizeof(double) * r.n_pieces);
  VD_COPY(vert_off, r.vert_off, sizeof(int64_t) * (r.n_pieces + 1));
  VD_COPY(vert_xyz, r.vert_xyz, sizeof(double) * r.n_verts * r.dim);
  VD_COPY(vert_flags, r.vert_flags, sizeof(int32_t) * r.n_verts * r.nfl);
  return cuda_check(c, cudaStreamSynchronize(c->stream), "vd_cells_to_host");
}

vd_status vd_nearest(vd_ctx* c, const double* queries, int64_t nq, int32_t* out_index) {
  if (!c || !queries || !out_index || nq < 1) return VD_E_ARG;
  vd_status s;
  if (!c->indexValid) {
    if ((s = ensure(c, c->control, sizeof(Control)))) return s;
    cudaMemsetAsync(c->control.p, 0, sizeof(Control), c->stream);
    if ((s = stage_index(c))) return s;
  }
  DevBuf q3, res;
  if ((s = upload_points(c, queries, nq, c->dim, q3, "vd_nearest"))) return s;
  if ((s = ensure(c, res, sizeof(int) * nq))) { release(c, q3); return s; }
  s = stage_nearest_points(c, q3.as<double>(), nq, res.as<int>());
  cudaError_t e = cudaMemcpyAsync(out_index, res.p, sizeof(int) * nq, cudaMemcpyDefault, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  release(c, q3);
  release(c, res);
  if (s != VD_OK) return s;
  return cuda_check(c, e, "vd_nearest");
}

vd_status vd_get_adjacency(vd_ctx* c, int32_t* out) {
  if (!c || !out) return VD_E_ARG;
  if (!c->haveDomain) return VD_E_STATE;
  cudaError_t e = cudaMemcpyAsync(out, c->adj.p, sizeof(int) * c->m * c->nc, cudaMemcpyDefault, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  return cuda_check(c, e, "vd_get_adjacency");
}

}  // extern "C"
