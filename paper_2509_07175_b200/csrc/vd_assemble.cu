// vd_assemble.cu -- S6: assemble the domain-cell intersections Omega_i ∩ M = union of P_{a,i}
// ("Omega_i|M <- Omega_i|M ∪ P in atomic", Alg. 4 line 10; centroids P:L443).  Instead of
// floating-point atomics the pieces are grouped by site (counting sort), ordered by simplex id inside
// each site (warp bitonic sort) and reduced in that fixed order, so results are bitwise reproducible.
// Then compacted CSR output (include/vd.h).  All streaming, HBM-bound.
#include "vd_internal.h"
#include "vd_scan.cuh"

namespace vd {

// In-place ascending sort of keys[0..k) (and vals alongside) by one warp: normalized bitonic network,
// every compare-exchange ascending, so a length that is not a power of two needs no padding.
__device__ __forceinline__ void warp_sort(int* keys, int* vals, int k) {
  if (k < 2) return;
  const int lane = lane_id();
  for (int size = 2; (size >> 1) < k; size <<= 1) {
    for (int i = lane; i < k; i += kLanes) {   // flip
      const int off = i & (size - 1);
      if (off < (size >> 1)) {
        const int j = i - off + size - 1 - off;
        if (j < k && keys[i] > keys[j]) {
          const int t = keys[i]; keys[i] = keys[j]; keys[j] = t;
          if (vals) { const int u = vals[i]; vals[i] = vals[j]; vals[j] = u; }
        }
      }
    }
    __syncwarp();
    for (int s = size >> 2; s > 0; s >>= 1) {  // disperse
      for (int i = lane; i < k; i += kLanes) {
        if ((i & (2 * s - 1)) < s) {
          const int j = i + s;
          if (j < k && keys[i] > keys[j]) {
            const int t = keys[i]; keys[i] = keys[j]; keys[j] = t;
            if (vals) { const int u = vals[i]; vals[i] = vals[j]; vals[j] = u; }
          }
        }
      }
      __syncwarp();
    }
  }
}

__global__ void __launch_bounds__(kBlock) k_group_pieces(const Piece* __restrict__ pieces, int64_t total, const int64_t* __restrict__ pieceOff,
                                                          int* __restrict__ siteFill, int* __restrict__ order) {
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += (int64_t)gridDim.x * blockDim.x) {
    const Piece& p = pieces[k];
    if (p.nverts <= 0) continue;
    const int64_t pos = pieceOff[p.site] + atomicAdd(&siteFill[p.site], 1);
    order[pos] = (int)k;
  }
}

struct AsmArgs {
  const Piece* pieces;
  const double* sites;
  const int* poolNbr;
  const int64_t* pieceOff;
  const int64_t* nbrRawOff;
  int* order;
  int* vcount;      // scratch keys, then corners per piece (in final piece order)
  int* nbrRaw;
  int* nbrCnt;
  double* oMeasure;
  double* oCentroid;
  int* oPieceSimplex;
  double* oPieceMeasure;
  Control* ctl;
  int64_t n;
  int dim;
};

// one THREAD per site: an empty cell gets measure 0, centroid = the site (include/vd.h); the others are listed for the
// warp-per-site kernels (when nearly every cell is empty -- far sites, BASELINE config 5: 0.07 % own a part of the
// domain -- a warp per site would spend the stage on two million empty visits)
__global__ void __launch_bounds__(kBlock) k_site_empty(AsmArgs A, int* __restrict__ list) {
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < A.n; i += (int64_t)gridDim.x * blockDim.x) {
    if (A.pieceOff[i + 1] == A.pieceOff[i]) {
      A.oMeasure[i] = 0.0;
      for (int a = 0; a < A.dim; ++a) A.oCentroid[i * A.dim + a] = A.sites[i * 3 + a];
      A.nbrCnt[i] = 0;
    } else {
      list[atomicAdd(&A.ctl->nListed, 1u)] = (int)i;
    }
  }
}

// one warp per listed (non-empty) site
__global__ void __launch_bounds__(kBlock) k_site_assemble(AsmArgs A, const int* __restrict__ list) {
  const int lane = lane_id();
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / kLanes;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) / kLanes;
  int nonEmpty = 0;
  const int64_t listed = A.ctl->nListed;
  for (int64_t li = warp; li < listed; li += nwarps) {
    const int64_t i = list[li];
    const int64_t b = A.pieceOff[i], e = A.pieceOff[i + 1];
    const int k = (int)(e - b);
    ++nonEmpty;
    for (int t = lane; t < k; t += kLanes) A.vcount[b + t] = A.pieces[A.order[b + t]].simplex;
    __syncwarp();
    warp_sort(A.vcount + b, A.order + b, k);
    double ms = 0, mx = 0, my = 0, mz = 0;
    int64_t ro = A.nbrRawOff[i];
    for (int t0 = 0; t0 < k; t0 += kLanes) {
      const int t = t0 + lane;
      int nn = 0;
      int64_t nb = 0;
      if (t < k) {
        const Piece& p = A.pieces[A.order[b + t]];
        ms += p.measure; mx += p.mx; my += p.my; mz += p.mz;
        A.oPieceSimplex[b + t] = p.simplex;
        A.oPieceMeasure[b + t] = p.measure;
        A.vcount[b + t] = p.nverts;
        nn = p.nnbr; nb = p.nbase;
      }
      // face flags of the site's pieces, concatenated
      int incl = nn;
      for (int off = 1; off < kLanes; off <<= 1) {
        const int o = __shfl_up_sync(kFull, incl, off);
        if (lane >= off) incl += o;
      }
      for (int q = 0; q < nn; ++q) A.nbrRaw[ro + incl - nn + q] = A.poolNbr[nb + q];
      ro += shfl(incl, kLanes - 1);
    }
    ms = warp_sum(ms); mx = warp_sum(mx); my = warp_sum(my); mz = warp_sum(mz);
    __syncwarp();
    // neighbours: ascending, each once
    const int64_t r0 = A.nbrRawOff[i];
    const int rk = (int)(ro - r0);
    warp_sort(A.nbrRaw + r0, nullptr, rk);
    int uniq = 0;
    for (int t = lane; t < rk; t += kLanes) uniq += (t == 0 || A.nbrRaw[r0 + t] != A.nbrRaw[r0 + t - 1]) ? 1 : 0;
    uniq = warp_sum(uniq);
    if (lane == 0) {
      A.oMeasure[i] = ms;
      const double inv = 1.0 / ms;
      A.oCentroid[i * A.dim + 0] = mx * inv;
      A.oCentroid[i * A.dim + 1] = my * inv;
      if (A.dim == 3) A.oCentroid[i * A.dim + 2] = mz * inv;
      A.nbrCnt[i] = uniq;
    }
  }
  nonEmpty = shfl(nonEmpty, 0);
  if (lane == 0 && nonEmpty) atomicAdd(&A.ctl->nNonEmpty, (unsigned long long)nonEmpty);
}

__global__ void __launch_bounds__(kBlock) k_compact_nbr(const int* __restrict__ nbrRaw, const int64_t* __restrict__ nbrRawOff,
                                                         const int64_t* __restrict__ nbrOff, const Control* __restrict__ ctl,
                                                         const int* __restrict__ list, int* __restrict__ oNbr) {
  const int lane = lane_id();
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / kLanes;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) / kLanes;
  const int64_t listed = ctl->nListed;
  for (int64_t li = warp; li < listed; li += nwarps) {
    const int64_t i = list[li];
    const int64_t r0 = nbrRawOff[i];
    const int rk = (int)(nbrRawOff[i + 1] - r0);
    int64_t out = nbrOff[i];
    for (int t0 = 0; t0 < rk; t0 += kLanes) {
      const int t = t0 + lane;
      const bool first = t < rk && (t == 0 || nbrRaw[r0 + t] != nbrRaw[r0 + t - 1]);
      const unsigned m = __ballot_sync(kFull, first);
      if (first) oNbr[out + __popc(m & ((1u << lane) - 1u))] = nbrRaw[r0 + t];
      out += __popc(m);
    }
  }
}

// one warp per piece (final order): copy its corners from the pool into the compact arrays
__global__ void __launch_bounds__(kBlock) k_gather_verts(const Piece* __restrict__ pieces, const int* __restrict__ order,
                                                          const int64_t* __restrict__ vertOff, int64_t nPieces,
                                                          const double* __restrict__ poolXYZ, const int* __restrict__ poolFlags, int dim,
                                                          int nfl, double* __restrict__ oXYZ, int* __restrict__ oFlags) {
  const int lane = lane_id();
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / kLanes;
  const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) / kLanes;
  for (int64_t p = warp; p < nPieces; p += nwarps) {
    const Piece& pc = pieces[order[p]];
    const int64_t dst = vertOff[p];
    const int nv = pc.nverts;
    for (int t = lane; t < nv * dim; t += kLanes) {
      const int v = t / dim, a = t % dim;
      oXYZ[dst * dim + t] = poolXYZ[(pc.vbase + v) * 3 + a];
    }
    for (int t = lane; t < nv * nfl; t += kLanes) oFlags[dst * nfl + t] = poolFlags[pc.vbase * nfl + t];
  }
}

__global__ void k_totals(Control* ctl, const int64_t* pieceOff, const int64_t* vertOff, const int64_t* nbrOff, int64_t n, int64_t nPieces) {
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    ctl->nPieces = (unsigned long long)pieceOff[n];
    ctl->nVerts = (unsigned long long)vertOff[nPieces];
    ctl->nNbrs = (unsigned long long)nbrOff[n];
  }
}

static int blocks_for(int64_t items, int perBlock) {
  int64_t b = (items + perBlock - 1) / perBlock;
  if (b > sm_count() * 16) b = sm_count() * 16;
  if (b < 1) b = 1;
  return (int)b;
}

vd_status stage_assemble(vd_ctx* c) {
  const int64_t n = c->n;
  const int64_t total = (int64_t)c->hostControl.pairTail;
  const int64_t nPieces = (int64_t)counters_total(c->hostControl).pieces;
  const int64_t nVerts = (int64_t)c->hostControl.vertTail;
  const int64_t nRaw = (int64_t)c->hostControl.nbrTail;
  const int dim = c->dim, nfl = c->nfl;
  cudaStream_t st = c->stream;
  vd_status s;
  if ((s = ensure(c, c->siteFill, sizeof(int) * n))) return s;
  if ((s = ensure(c, c->order, sizeof(int) * (nPieces + 1)))) return s;
  if ((s = ensure(c, c->vcount, sizeof(int) * (nPieces + 1)))) return s;
  if ((s = ensure(c, c->nbrRawOff, sizeof(int64_t) * (n + 1)))) return s;
  if ((s = ensure(c, c->nbrRaw, sizeof(int) * (nRaw + 1)))) return s;
  if ((s = ensure(c, c->nbrCnt, sizeof(int) * n))) return s;
  if ((s = ensure(c, c->oMeasure, sizeof(double) * n))) return s;
  if ((s = ensure(c, c->oCentroid, sizeof(double) * n * dim))) return s;
  if ((s = ensure(c, c->oNbrOff, sizeof(int64_t) * (n + 1)))) return s;
  if ((s = ensure(c, c->oNbr, sizeof(int) * (nRaw + 1)))) return s;
  if ((s = ensure(c, c->oPieceOff, sizeof(int64_t) * (n + 1)))) return s;
  if ((s = ensure(c, c->oPieceSimplex, sizeof(int) * (nPieces + 1)))) return s;
  if ((s = ensure(c, c->oPieceMeasure, sizeof(double) * (nPieces + 1)))) return s;
  if ((s = ensure(c, c->oVertOff, sizeof(int64_t) * (nPieces + 1)))) return s;
  if ((s = ensure(c, c->oVertXYZ, sizeof(double) * (nVerts * dim + 1)))) return s;
  if ((s = ensure(c, c->oVertFlags, sizeof(int) * (nVerts * nfl + 1)))) return s;
  const int64_t scanN = n > nPieces ? n : nPieces;
  if ((s = ensure(c, c->scanTmp, sizeof(int64_t) * scan_scratch_elems(scanN) * 2))) return s;
  int64_t* tmp = c->scanTmp.as<int64_t>();

  exclusive_scan<int, int64_t>(c->sitePieces.as<int>(), n, c->oPieceOff.as<int64_t>(), tmp, st);
  exclusive_scan<int, int64_t>(c->siteNbrRaw.as<int>(), n, c->nbrRawOff.as<int64_t>(), tmp, st);
  cudaMemsetAsync(c->siteFill.p, 0, sizeof(int) * n, st);
  VD_LAUNCH(k_group_pieces, blocks_for(total, kBlock), kBlock, 0, st)(c->pieces.as<Piece>(), total, c->oPieceOff.as<int64_t>(),
                                                                      c->siteFill.as<int>(), c->order.as<int>());
  AsmArgs A;
  A.pieces = c->pieces.as<Piece>(); A.sites = c->sites.as<double>(); A.poolNbr = c->poolNbr.as<int>();
  A.pieceOff = c->oPieceOff.as<int64_t>(); A.nbrRawOff = c->nbrRawOff.as<int64_t>();
  A.order = c->order.as<int>(); A.vcount = c->vcount.as<int>(); A.nbrRaw = c->nbrRaw.as<int>(); A.nbrCnt = c->nbrCnt.as<int>();
  A.oMeasure = c->oMeasure.as<double>(); A.oCentroid = c->oCentroid.as<double>();
  A.oPieceSimplex = c->oPieceSimplex.as<int>(); A.oPieceMeasure = c->oPieceMeasure.as<double>();
  A.ctl = c->control.as<Control>(); A.n = n; A.dim = dim;
  if ((s = ensure(c, c->siteList, sizeof(int) * n))) return s;
  VD_LAUNCH(k_site_empty, blocks_for(n, kBlock), kBlock, 0, st)(A, c->siteList.as<int>());
  VD_LAUNCH(k_site_assemble, blocks_for(n, kWarpsPerBlock), kBlock, 0, st)(A, c->siteList.as<int>());
  exclusive_scan<int, int64_t>(c->vcount.as<int>(), nPieces, c->oVertOff.as<int64_t>(), tmp, st);
  exclusive_scan<int, int64_t>(c->nbrCnt.as<int>(), n, c->oNbrOff.as<int64_t>(), tmp, st);
  VD_LAUNCH(k_gather_verts, blocks_for(nPieces, kWarpsPerBlock), kBlock, 0, st)(
      c->pieces.as<Piece>(), c->order.as<int>(), c->oVertOff.as<int64_t>(), nPieces, c->poolXYZ.as<double>(), c->poolFlags.as<int>(),
      dim, nfl, c->oVertXYZ.as<double>(), c->oVertFlags.as<int>());
  VD_LAUNCH(k_compact_nbr, blocks_for(n, kWarpsPerBlock), kBlock, 0, st)(c->nbrRaw.as<int>(), c->nbrRawOff.as<int64_t>(),
                                                                          c->oNbrOff.as<int64_t>(), c->control.as<Control>(), c->siteList.as<int>(), c->oNbr.as<int>());
  VD_LAUNCH(k_totals, 1, 1, 0, st)(c->control.as<Control>(), c->oPieceOff.as<int64_t>(), c->oVertOff.as<int64_t>(),
                                   c->oNbrOff.as<int64_t>(), n, nPieces);
  return cuda_check(c, cudaGetLastError(), "assemble");
}

}  // namespace vd
