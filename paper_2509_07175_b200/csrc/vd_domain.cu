// vd_domain.cu -- S0 (inside vd_set_domain): validate the simplices and derive the adjacency that
// initialises the edge/face flags of every T_a (Fig. 2a).  Two simplices are adjacent across a
// face iff they share its d vertices: faces are matched through a hash table of face owners.
#include "vd_internal.h"

namespace vd {

__device__ __forceinline__ void face_key(const int* __restrict__ simp, int nc, int owner, int key[3]) {
  const int a = owner / nc, k = owner % nc;
  int t = 0;
  key[2] = -1;
  for (int c = 0; c < nc; ++c)
    if (c != k) key[t++] = simp[(int64_t)a * nc + c];
  // ascending
  if (nc == 4) {
    int u;
    if (key[0] > key[1]) { u = key[0]; key[0] = key[1]; key[1] = u; }
    if (key[1] > key[2]) { u = key[1]; key[1] = key[2]; key[2] = u; }
    if (key[0] > key[1]) { u = key[0]; key[0] = key[1]; key[1] = u; }
  } else if (key[0] > key[1]) {
    const int u = key[0]; key[0] = key[1]; key[1] = u;
  }
}

__global__ void __launch_bounds__(kBlock) k_validate(const double* __restrict__ verts, int64_t nv, const int* __restrict__ simp, int64_t m,
                                                      int nc, int kind, unsigned int* err) {
  for (int64_t a = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; a < m; a += (int64_t)gridDim.x * blockDim.x) {
    double p[4][3];
    bool bad = false;
    for (int k = 0; k < nc; ++k) {
      const int v = simp[a * nc + k];
      if (v < 0 || v >= nv) { bad = true; break; }
      for (int t = 0; t < 3; ++t) p[k][t] = verts[(int64_t)v * 3 + t];
    }
    if (!bad) {
      const double ax = p[1][0] - p[0][0], ay = p[1][1] - p[0][1], az = p[1][2] - p[0][2];
      const double bx = p[2][0] - p[0][0], by = p[2][1] - p[0][1], bz = p[2][2] - p[0][2];
      const double cx = ay * bz - az * by, cy = az * bx - ax * bz, cz = ax * by - ay * bx;
      double meas;
      if (kind == KIND_TET_3D) {
        meas = cx * (p[3][0] - p[0][0]) + cy * (p[3][1] - p[0][1]) + cz * (p[3][2] - p[0][2]);
      } else {
        meas = sqrt(cx * cx + cy * cy + cz * cz);
      }
      if (!(meas != 0.0) || !(meas == meas) || fabs(meas) > 1e300) bad = true;   // zero measure or non-finite
    }
    if (bad) atomicOr(err, ERR_INPUT);
  }
}

__global__ void __launch_bounds__(kBlock) k_adjacency(const int* __restrict__ simp, int64_t m, int nc, int* __restrict__ table,
                                                       uint64_t mask, int* __restrict__ adj, unsigned int* err) {
  const int64_t total = m * nc;
  for (int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; f < total; f += (int64_t)gridDim.x * blockDim.x) {
    int key[3];
    face_key(simp, nc, (int)f, key);
    uint64_t h = hash64(((uint64_t)(uint32_t)key[0] * 0x9e3779b97f4a7c15ull) ^ ((uint64_t)(uint32_t)key[1] << 21) ^
                        ((uint64_t)(uint32_t)key[2] << 42)) & mask;
    for (uint64_t probe = 0; probe <= mask; ++probe) {
      const int cur = atomicCAS(&table[h], -1, (int)f);
      if (cur == -1) break;   // first owner of this face
      int other[3];
      face_key(simp, nc, cur, other);
      if (other[0] == key[0] && other[1] == key[1] && other[2] == key[2]) {
        // partner found: link both ways; a third simplex on the same face is non-manifold
        const int old = atomicExch(&adj[cur], (int)(f / nc));
        if (old != (int)m) atomicOr(err, ERR_INPUT);
        adj[f] = cur / nc;
        break;
      }
      h = (h + 1) & mask;
    }
  }
}

__global__ void __launch_bounds__(kBlock) k_fill_int(int* p, int64_t n, int v) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) p[i] = v;
}

vd_status stage_domain(vd_ctx* c) {
  const int64_t m = c->m;
  const int nc = c->nc;
  cudaStream_t st = c->stream;
  vd_status s;
  if ((s = ensure(c, c->adj, sizeof(int) * m * nc))) return s;
  if ((s = ensure(c, c->control, sizeof(Control)))) return s;
  uint64_t cap = 64;
  while (cap < (uint64_t)(2 * m * nc)) cap <<= 1;
  DevBuf table;
  if ((s = ensure(c, table, sizeof(int) * cap))) return s;
  cudaMemsetAsync(c->control.p, 0, sizeof(Control), st);
  int blocks = (int)((m * nc + kBlock - 1) / kBlock);
  if (blocks > sm_count() * 16) blocks = sm_count() * 16;
  VD_LAUNCH(k_validate, blocks, kBlock, 0, st)(c->verts.as<double>(), c->nv, c->simp.as<int>(), m, nc, c->kind,
                                                &c->control.as<Control>()->err);
  VD_LAUNCH(k_fill_int, blocks, kBlock, 0, st)(table.as<int>(), (int64_t)cap, -1);
  VD_LAUNCH(k_fill_int, blocks, kBlock, 0, st)(c->adj.as<int>(), m * nc, (int)m);
  Control h;
  cudaError_t e = cudaMemcpyAsync(&h, c->control.p, sizeof(Control), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) { release(c, table); return cuda_check(c, e, "set_domain"); }
  if (h.err & ERR_INPUT) {
    release(c, table);
    c->lastError = "vd_set_domain: vertex index out of range, non-finite coordinate or zero-measure simplex";
    return VD_E_INPUT;
  }
  VD_LAUNCH(k_adjacency, blocks, kBlock, 0, st)(c->simp.as<int>(), m, nc, table.as<int>(), cap - 1, c->adj.as<int>(),
                                                 &c->control.as<Control>()->err);
  e = cudaMemcpyAsync(&h, c->control.p, sizeof(Control), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  release(c, table);
  if (e != cudaSuccess) return cuda_check(c, e, "set_domain");
  if (h.err & ERR_INPUT) {
    c->lastError = "vd_set_domain: an edge/face is shared by more than two simplices";
    return VD_E_INPUT;
  }
  return VD_OK;
}

// ---- dissolve mode (Alg. 5 lines 2-6; vd_options.dissolve): what depends on the domain only ------------------

__global__ void __launch_bounds__(kBlock) k_boundary_count(const int* __restrict__ adj, int64_t m, unsigned long long* __restrict__ count) {
  unsigned mine = 0;
  for (int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; f < 4 * m; f += (int64_t)gridDim.x * blockDim.x)
    mine += adj[f] == (int)m ? 1u : 0u;
  mine = (unsigned)warp_sum((int)mine);
  if (lane_id() == 0 && mine) atomicAdd(count, (unsigned long long)mine);
}

// "extract the boundary triangles of M" (Alg. 5 line 2): the faces no other tet owns, with the tet behind each and its
// supporting plane (unit normal pointing out of the tet, offset)
__global__ void __launch_bounds__(kBlock) k_boundary_fill(const int* __restrict__ simp, const int* __restrict__ adj, const double* __restrict__ verts,
                                                           int64_t m, unsigned long long* __restrict__ cursor, int* __restrict__ tris,
                                                           int* __restrict__ tet, double4* __restrict__ planes) {
  for (int64_t f = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; f < 4 * m; f += (int64_t)gridDim.x * blockDim.x) {
    if (adj[f] != (int)m) continue;
    const int64_t a = f / 4;
    const int k = (int)(f % 4);
    int v[3], t = 0;
    for (int c = 0; c < 4; ++c)
      if (c != k) v[t++] = simp[a * 4 + c];
    const int vk = simp[a * 4 + k];
    const double* p0 = verts + (int64_t)v[0] * 3;
    const double* p1 = verts + (int64_t)v[1] * 3;
    const double* p2 = verts + (int64_t)v[2] * 3;
    const double* pk = verts + (int64_t)vk * 3;
    const double ax = p1[0] - p0[0], ay = p1[1] - p0[1], az = p1[2] - p0[2];
    const double bx = p2[0] - p0[0], by = p2[1] - p0[1], bz = p2[2] - p0[2];
    double nx = ay * bz - az * by, ny = az * bx - ax * bz, nz = ax * by - ay * bx;
    const double inv = 1.0 / sqrt(nx * nx + ny * ny + nz * nz);
    nx *= inv; ny *= inv; nz *= inv;
    if (nx * (pk[0] - p0[0]) + ny * (pk[1] - p0[1]) + nz * (pk[2] - p0[2]) > 0) { nx = -nx; ny = -ny; nz = -nz; }
    const unsigned long long slot = atomicAdd(cursor, 1ull);
    tris[slot * 3 + 0] = v[0]; tris[slot * 3 + 1] = v[1]; tris[slot * 3 + 2] = v[2];
    tet[slot] = (int)a;
    planes[slot] = make_double4(nx, ny, nz, nx * p0[0] + ny * p0[1] + nz * p0[2]);
  }
}

// the distinct supporting planes: triangle t keeps its plane unless an earlier triangle lies in the same one
__global__ void __launch_bounds__(kBlock) k_plane_unique(const double4* __restrict__ raw, int64_t nb, double tol, unsigned long long* __restrict__ cursor,
                                                          double4* __restrict__ out) {
  for (int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; t < nb; t += (int64_t)gridDim.x * blockDim.x) {
    const double4 p = raw[t];
    bool uniq = true;
    for (int64_t o = 0; o < t && uniq; ++o) {
      const double4 q = raw[o];
      if (p.x * q.x + p.y * q.y + p.z * q.z > 1.0 - 1e-12 && fabs(p.w - q.w) <= tol * fmax(1.0, fabs(p.w))) uniq = false;   // (relative to the offset's size)
    }
    if (uniq) out[atomicAdd(cursor, 1ull)] = p;
  }
}

// A domain is convex iff it lies on the inner side of every supporting plane of its boundary: every mesh vertex against every
// distinct plane.  Also the bounding box of the mesh (block 0), as the 8 corners the whole-cell kernels start from.
__global__ void __launch_bounds__(kBlock) k_convex_check(const double* __restrict__ verts, int64_t nv, const double4* __restrict__ planes, int np,
                                                          double tol, unsigned int* err, double* __restrict__ box) {
  for (int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; v < nv; v += (int64_t)gridDim.x * blockDim.x) {
    const double x = verts[v * 3 + 0], y = verts[v * 3 + 1], z = verts[v * 3 + 2];
    bool out = false;
    for (int k = 0; k < np; ++k) {
      const double4 p = planes[k];
      out |= p.x * x + p.y * y + p.z * z - p.w > tol * fmax(1.0, fmax(fabs(p.w), fabs(x) + fabs(y) + fabs(z)));   // (relative to the coordinates' size)
    }
    if (out) atomicOr(err, ERR_TOPOLOGY);
  }
  if (blockIdx.x == 0) {
    __shared__ double sm[kWarpsPerBlock][6];
    double lo[3] = {1e300, 1e300, 1e300}, hi[3] = {-1e300, -1e300, -1e300};
    for (int64_t v = threadIdx.x; v < nv; v += blockDim.x)
      for (int a = 0; a < 3; ++a) { lo[a] = fmin(lo[a], verts[v * 3 + a]); hi[a] = fmax(hi[a], verts[v * 3 + a]); }
    for (int a = 0; a < 3; ++a)
      for (int off = kLanes / 2; off > 0; off >>= 1) {
        lo[a] = fmin(lo[a], __shfl_xor_sync(kFull, lo[a], off));
        hi[a] = fmax(hi[a], __shfl_xor_sync(kFull, hi[a], off));
      }
    if (lane_id() == 0)
      for (int a = 0; a < 3; ++a) { sm[threadIdx.x / kLanes][a] = lo[a]; sm[threadIdx.x / kLanes][3 + a] = hi[a]; }
    __syncthreads();
    if (threadIdx.x == 0) {
      for (int w = 1; w < (int)blockDim.x / kLanes; ++w)
        for (int a = 0; a < 3; ++a) { sm[0][a] = fmin(sm[0][a], sm[w][a]); sm[0][3 + a] = fmax(sm[0][3 + a], sm[w][3 + a]); }
      for (int c = 0; c < 8; ++c)
        for (int a = 0; a < 3; ++a) box[c * 3 + a] = ((c >> a) & 1) ? sm[0][3 + a] : sm[0][a];
    }
  }
}

void dissolve_release(vd_ctx* c) {
  if (c->boundary) { vd_destroy(c->boundary); c->boundary = nullptr; }
  c->dissolveReady = false;
  c->nBoundary = 0;
  c->nBPlanes = 0;
}

vd_status stage_dissolve_prepare(vd_ctx* c) {
  dissolve_release(c);
  const int64_t m = c->m;
  cudaStream_t st = c->stream;
  vd_status s;
  if ((s = ensure(c, c->control, sizeof(Control)))) return s;
  Control* ctl = c->control.as<Control>();
  cudaMemsetAsync(ctl, 0, sizeof(Control), st);
  int blocks = (int)((4 * m + kBlock - 1) / kBlock);
  if (blocks > sm_count() * 16) blocks = sm_count() * 16;
  VD_LAUNCH(k_boundary_count, blocks, kBlock, 0, st)(c->adj.as<int>(), m, &ctl->pairTail);
  Control h;
  cudaError_t e = cudaMemcpyAsync(&h, ctl, sizeof(Control), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return cuda_check(c, e, "dissolve: boundary");
  const int64_t nb = (int64_t)h.pairTail;
  if (nb < 4) { c->lastError = "vd_compute (dissolve): the mesh has no closed boundary"; return VD_E_ARG; }
  DevBuf raw;
  if ((s = ensure(c, c->bTris, sizeof(int) * 3 * nb)) || (s = ensure(c, c->bTet, sizeof(int) * nb)) ||
      (s = ensure(c, raw, sizeof(double4) * nb)) || (s = ensure(c, c->bPlanes, sizeof(double4) * nb)) ||
      (s = ensure(c, c->boxVerts, sizeof(double) * 24)) || (s = ensure(c, c->boxVnn, sizeof(int) * 8))) { release(c, raw); return s; }
  VD_LAUNCH(k_boundary_fill, blocks, kBlock, 0, st)(c->simp.as<int>(), c->adj.as<int>(), c->verts.as<double>(), m, &ctl->vertTail,
                                                     c->bTris.as<int>(), c->bTet.as<int>(), raw.as<double4>());
  // scale of the domain for the tolerances: the bounding box comes with the convexity check, so a first rough scale from it later;
  // plane offsets of one supporting plane agree to rounding
  int pb = (int)((nb + kBlock - 1) / kBlock);
  if (pb > sm_count() * 16) pb = sm_count() * 16;
  VD_LAUNCH(k_plane_unique, pb, kBlock, 0, st)(raw.as<double4>(), nb, 1e-11, &ctl->nbrTail, c->bPlanes.as<double4>());
  e = cudaMemcpyAsync(&h, ctl, sizeof(Control), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  release(c, raw);
  if (e != cudaSuccess) return cuda_check(c, e, "dissolve: planes");
  const int np = (int)h.nbrTail;
  if (np > 8192) { c->lastError = "vd_compute (dissolve): more than 8192 distinct boundary planes (the inside test visits every one per site)"; return VD_E_ARG; }
  int vb = (int)((c->nv + kBlock - 1) / kBlock);
  if (vb > sm_count() * 16) vb = sm_count() * 16;
  VD_LAUNCH(k_convex_check, vb, kBlock, 0, st)(c->verts.as<double>(), c->nv, c->bPlanes.as<double4>(), np, 1e-10, &ctl->err, c->boxVerts.as<double>());
  e = cudaMemcpyAsync(&h, ctl, sizeof(Control), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return cuda_check(c, e, "dissolve: convexity");
  if (h.err & ERR_TOPOLOGY) { c->lastError = "vd_compute (dissolve): the tet mesh is not convex (Alg. 5's site division needs a convex domain, P:L351-355)"; return VD_E_ARG; }
  // the child context: restricted Voronoi diagram of the same sites on the boundary triangles (Alg. 5 line 3)
  vd_ctx* child = nullptr;
  if ((s = vd_create(c->sites.as<double>(), c->n, 3, &child))) { c->lastError = "vd_compute (dissolve): boundary context"; return s; }
  child->stream = st;
  child->allocFn = c->allocFn; child->freeFn = c->freeFn; child->allocUser = c->allocUser;
  if ((s = vd_set_domain(child, c->verts.as<double>(), c->nv, c->bTris.as<int>(), nb, VD_TRI_SURFACE))) {
    c->lastError = std::string("vd_compute (dissolve): boundary surface: ") + child->lastError;
    vd_destroy(child);
    return s;
  }
  c->boundary = child;
  c->nBoundary = nb;
  c->nBPlanes = np;
  c->dissolveReady = true;
  return VD_OK;
}

// Alg. 5 line 3: "compute the restricted Voronoi diagram on the boundary triangles" -- the surface path of this library, on the
// current sites.  A site with a non-empty restricted cell is a boundary site (line 4), the others are interior (line 5) or,
// when they lie outside M, own nothing (reading U13).
vd_status stage_dissolve_classify(vd_ctx* c) {
  vd_ctx* b = c->boundary;
  cudaError_t e = cudaMemcpyAsync(b->sites.p, c->sites.p, sizeof(double) * 3 * c->n, cudaMemcpyDeviceToDevice, c->stream);
  if (e != cudaSuccess) return cuda_check(c, e, "dissolve: sites");
  b->stream = c->stream;
  b->indexValid = false;
  b->heavyKnown = -1;
  b->opt.grid_density = c->opt.grid_density;
  b->opt.persistent = 3;   // the boundary surface is small: one queue launch drains it, one look at the device
  vd_cells cells;
  const vd_status s = vd_compute(b, &cells);
  c->syncs += b->syncs;
  if (s != VD_OK) c->lastError = std::string("vd_compute (dissolve): restricted diagram on the boundary: ") + b->lastError;
  return s;
}

}  // namespace vd
