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

}  // namespace vd
