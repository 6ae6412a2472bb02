// vd_internal.h -- the context behind the C ABI (include/vd.h) and the stage entry points.
#pragma once
#include <string>
#include <vector>

#include "../../include/vd.h"
#ifndef VD_VARIANT
#define VD_VARIANT full
#endif
#include "vd_common.cuh"

namespace vd {

// Device-side control block: queue tails, pool cursors, sticky error word, work counters.
struct Control {
  unsigned long long pairTail;   // pairs pushed so far
  unsigned long long ovfTail;    // pairs deferred to the large-capacity path
  unsigned long long vertTail;   // corners allocated in the pool
  unsigned long long nbrTail;    // face flags allocated in the pool
  unsigned long long fetch[2];   // work cursors: fast tier, large tier
  unsigned long long finished;   // pairs the fast tier has completed (persistent mode: termination)
  unsigned int err;              // ERR_* bits
  unsigned int nHeavy;           // refined cells of the site index (second level)
  Counters cnt[kCntKinds];       // per kernel kind (CNT_*): k_ph_init, verify, fix, finish, tail, everything else
  unsigned long long nPieces, nNonEmpty, nVerts, nNbrs;   // totals written by S6
  // wave programs (vd_clip.cu): the wavefronts of Alg. 4 / 5 advance on the device
  unsigned long long waveEnd;    // pairs [0, waveEnd) of the list have been dispatched to a wave
  unsigned long long ovfDone;    // deferred pairs [0, ovfDone) have been dispatched to the large tier
  unsigned long long ovfBegin, ovfEnd;   // the large tier's range in the current program
  unsigned long long nWaves;     // non-empty wavefronts so far
  unsigned int nListed, padListed;                        // S6: non-empty sites listed for the warp-per-site kernels
};

inline Counters counters_total(const Control& h) {
  Counters t = {};
  const int nf = (int)(sizeof(Counters) / sizeof(unsigned long long));
  for (int k = 0; k < kCntKinds; ++k)
    for (int f = 0; f < nf; ++f)
      reinterpret_cast<unsigned long long*>(&t)[f] += reinterpret_cast<const unsigned long long*>(&h.cnt[k])[f];
  return t;
}

struct DevBuf {
  void* p = nullptr;
  size_t cap = 0;
  bool hooked = false;   // came from the caller's allocator hook (vd_set_allocator): goes back through its release hook
  template <typename T> T* as() const { return reinterpret_cast<T*>(p); }
};

}  // namespace vd

struct vd_ctx {
  int64_t n = 0, nv = 0, m = 0;
  int dim = 0, kind = -1, nc = 0, nfl = 0;   // dim = the caller's dimension (inputs and outputs); kind = the kind the kernels run
  bool weighted = false;   // vd_create_weighted: dim 2 -> sites lifted to R^3, VD_TRI_2D runs as a flat surface;
                           //                     dim 3 -> siteW holds the additive term eta - w_i of every site
  int64_t syncs = 0;       // host waits on the stream inside the current vd_compute
  bool nearReady = false;  // nearList already holds the first clips of the next compute (vd_lloyd: the previous neighbours)
  int nearK = 0;           // entries per site of nearList in the last compute (0: no list)
  int heavyKnown = -1;     // refined cells of the site index as last built, while sites and grid options are unchanged; else -1
  bool haveDomain = false, haveResult = false, indexValid = false;
  cudaStream_t stream = nullptr;
  void* (*allocFn)(size_t, void*, void*) = nullptr;
  void (*freeFn)(void*, void*) = nullptr;
  void* allocUser = nullptr;
  vd_options opt{};
  vd_counters counters{};
  vd_counters phaseCounters[6] = {};   // per kernel kind (vd_get_phase_counters)
  double stageMs[5] = {0, 0, 0, 0, 0};
  double phaseMs[5] = {0, 0, 0, 0, 0};
  // device times of the step kernels: an event before every launch of a wave program, read after the batch's one
  // synchronisation (the interval that starts at event k belongs to step kernel evKind[k]; -1: not a step kernel)
  std::vector<cudaEvent_t> evPool;
  std::vector<int> evKind;
  int evUsed = 0;
  std::string lastError;
  cudaEvent_t ev[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};

  int64_t pairCap = 0, vertCap = 0, nbrCap = 0, hashCap = 0, ovfCap = 0, gridCap = 0;

  // inputs
  vd::DevBuf sites;       // double [n][3] (z = 0 for dim 2; z = sqrt(eta - w_i) for weighted 2D sites)
  vd::DevBuf siteW;       // double [n]  eta - w_i (weighted 3D sites), else empty
  vd::DevBuf verts;       // double [nv][3]
  vd::DevBuf simp;        // int [m][nc]
  vd::DevBuf adj;         // int [m][nc]
  // S1
  vd::DevBuf grid;        // GridIndex (device copy)
  vd::DevBuf bbox;        // double partial min/max
  vd::DevBuf cellOf;      // int [n]
  vd::DevBuf cellStart;   // int [gridCap+1]
  vd::DevBuf cellFill;    // int [gridCap+1]
  vd::DevBuf sorted32;    // float4 [n]  the sorted sites in fp32 (vd_options.fp32_filter)
  vd::DevBuf sortKeys, sortVals, sortHist;   // S1 radix sort: keys / site ids (two halves each), per-(digit, segment) counts
  vd::DevBuf sortedW;     // double [n]  additive terms of weighted 3-D sites in index order
  vd::DevBuf delta;       // double [n]  S1b: half the distance to the nearest other site (vd_options.step_out)
  vd::DevBuf scanTmp;     // scan scratch
  vd::DevBuf heavyFlag, heavyPrefix, subNeed, subOffRaw, subOff, subCount, subStart;   // second level
  vd::DevBuf sorted2;     // double4 [n]  the sites in index order (x, y, z, id bits)
  int64_t subCap = 0;
  // dissolve mode (Alg. 5 lines 2-6, vd_options.dissolve): prepared once per domain (vd_domain.cu)
  bool dissolveReady = false;
  vd_ctx* boundary = nullptr;   // child context: the restricted Voronoi diagram on the boundary triangles of M (Alg. 5 line 3)
  int64_t nBoundary = 0;        // boundary triangles
  int nBPlanes = 0;             // distinct supporting planes of the (convex) domain
  vd::DevBuf bTris;             // int [nBoundary][3]
  vd::DevBuf bTet;              // int [nBoundary]  the tet behind every boundary triangle
  vd::DevBuf bPlanes;           // double4 [nBPlanes]  outward unit normal, offset: inside iff n.x <= d
  vd::DevBuf boxVerts;          // double [8][3]  corners of the mesh's bounding box (corner c = bits x, y, z)
  vd::DevBuf boxVnn;            // int [8]  their nearest sites
  // S3-S5
  vd::DevBuf vnn;         // int [nv]   nearest site of every mesh vertex
  vd::DevBuf seedPts, seedNN;   // extra seed points inside the simplices and their nearest sites (few simplices, many sites)
  vd::DevBuf nearList;    // int [n][nearClips]  sites nearest to every site, nearest first, -1 padded (reading U19)
  vd::DevBuf nearAuto;    // 7 x uint64: the domain's box (sortable keys of lo / hi) and the number of sites inside it (tet meshes: whether U19 pays)
  vd::DevBuf control;     // Control
  vd::DevBuf phaseCells;  // phased mode: polytopes of one wave parked between the step kernels (vd_phase.cu)
  vd::DevBuf phaseLists;  // phased mode: work lists + counters
  vd::DevBuf pairs;       // Pair [pairCap]
  vd::DevBuf pieces;      // Piece [pairCap]
  vd::DevBuf visited;     // u64 [hashCap]
  vd::DevBuf ovf;         // int [ovfCap]
  vd::DevBuf poolXYZ;     // double [vertCap][3]
  vd::DevBuf poolFlags;   // int [vertCap][nfl]
  vd::DevBuf poolNbr;     // int [nbrCap]
  // S6
  vd::DevBuf sitePieces;  // int [n]  pieces per site
  vd::DevBuf siteNbrRaw;  // int [n]  face flags per site (with repeats)
  vd::DevBuf siteFill;    // int [n]
  vd::DevBuf order;       // int [pieces]  piece list grouped by site, sorted by simplex
  vd::DevBuf nbrRawOff;   // int64 [n+1]
  vd::DevBuf nbrRaw;      // int [sum raw]
  vd::DevBuf nbrCnt;      // int [n]
  vd::DevBuf siteList;    // int [n]  the non-empty sites
  vd::DevBuf vcount;      // int [pieces]
  // outputs (vd_cells)
  vd::DevBuf oMeasure, oCentroid, oNbrOff, oNbr, oPieceOff, oPieceSimplex, oPieceMeasure, oVertOff, oVertXYZ, oVertFlags;
  vd_cells cells{};
  vd::Control hostControl{};
  void* pinned = nullptr;   // page-locked staging for the small device -> host reads of a compute (round / wave counters)
};

namespace vd {

int sm_count();   // multiprocessors of the current device (cudaDevAttrMultiProcessorCount, cached): launch grids are multiples of it
cudaError_t sync_stream(vd_ctx* c, const char* why = nullptr);   // cudaStreamSynchronize on the context's stream, counted (vd_counters.syncs)

// memory
vd_status ensure(vd_ctx* c, DevBuf& b, size_t bytes);
void release(vd_ctx* c, DevBuf& b);
vd_status cuda_check(vd_ctx* c, cudaError_t e, const char* what);

void phase_mark(vd_ctx* c, int kind);      // record the next event of the pool; the launches up to the next mark are `kind`
void phase_marks_collect(vd_ctx* c);       // after a synchronisation: add the intervals to c->phaseMs, reset the pool

// stages (each enqueues kernels on c->stream)
vd_status stage_domain(vd_ctx* c);                 // S0  vd_domain.cu
vd_status stage_dissolve_prepare(vd_ctx* c);       // S0, dissolve mode: boundary triangles, convexity, planes, bounding box, child context
vd_status stage_dissolve_classify(vd_ctx* c);      // Alg. 5 lines 3-5: restricted VD on the boundary (child context) -> V_B / V_I
void dissolve_release(vd_ctx* c);
vd_status stage_index(vd_ctx* c);                  // S1  vd_index.cu
vd_status stage_nearest_points(vd_ctx* c, const double* q3, int64_t nq, int* out);  // S2 as a kernel (vd_nearest, vnn)
// S3 and S4+S5 (vd_clip.cu, vd_phase.cu) exist twice: lean (no optional query features compiled in) and full
namespace lean { vd_status stage_seed(vd_ctx* c); vd_status stage_clip(vd_ctx* c); }
namespace full { vd_status stage_seed(vd_ctx* c); vd_status stage_clip(vd_ctx* c); }
vd_status stage_assemble(vd_ctx* c);               // S6  vd_assemble.cu

}  // namespace vd
