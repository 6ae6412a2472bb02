/* vd.h -- C ABI of libvd.so: clipped / restricted Voronoi cells by point-in-cell clipping on one B200.
 *
 * The calls follow the problem statement of "Efficient Computation of Voronoi Diagrams Using
 * Point-in-Cell Tests" (Xiao, Cao, Chen; /root/reference/PAPER.md, cited below as P:Lnnn):
 * input sites V = {v_i} in R^d and a domain M = {T_a} of simplices, output the domain-cell
 * intersections {Omega_i ∩ M}, i = 1..n  (Eq. 1 at P:L77), each the union of
 * simplex-cell pieces P_{a,i} = T_a ∩ Omega_i whose edges / faces carry flags.
 *
 * Everything behind these calls runs in hand-written CUDA kernels for sm_100a, in fp64.  There is
 * no CPU fallback: every entry point that needs the device returns VD_E_CUDA when it is missing.
 *
 * Pointers: every INPUT pointer may be a host pointer or a device pointer (resolved with
 * cudaPointerGetAttributes); inputs are copied, the caller keeps ownership and may free them as
 * soon as the call returns.  Every OUTPUT pointer inside vd_cells is a DEVICE pointer owned by the
 * context, valid until the next vd_compute on that context or vd_destroy.  One context must be
 * used by one host thread at a time.  Errors are return codes only; a failed call leaves the
 * context usable; vd_last_error() gives a one-line description.
 */
#ifndef VD_H_
#define VD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct vd_ctx vd_ctx; /* opaque; owns all device state */

typedef enum {
  VD_OK = 0,
  VD_E_ARG = 1,        /* null pointer, n < 1, m < 1, bad kind                                   */
  VD_E_DIM = 2,        /* dim not in {2,3} or kind / dim mismatch                                */
  VD_E_STATE = 3,      /* vd_compute before vd_set_domain, vd_cells_to_host before vd_compute    */
  VD_E_INPUT = 4,      /* NaN/Inf, duplicate sites, index out of range, zero-measure simplex,
                          non-manifold face, eta below the largest weight                        */
  VD_E_CUDA = 5,       /* no device, or a CUDA runtime error                                     */
  VD_E_NOMEM = 6,
  VD_E_CAPACITY = 7,   /* a piece outgrew every capacity tier (see vd_options)                   */
  VD_E_NOCONVERGE = 8  /* an iteration cap was hit (degenerate input)                            */
} vd_status;

/* Domain kinds.  dim == 2 <=> VD_TRI_2D, VD_BOX_2D;  dim == 3 <=> VD_TRI_SURFACE, VD_TET_3D, VD_BOX_3D. */
typedef enum {
  VD_TRI_2D = 0, VD_TRI_SURFACE = 1, VD_TET_3D = 2,
  /* "simple domains" of section V-B ("e.g. a cube"): an axis-aligned rectangle (dim 2) or box
   * (dim 3) given by its two opposite corners, verts = [lo, hi], nv = 2, simplices ignored (may be NULL), m = 1.
   * The whole domain is ONE piece per cell (piece_simplex = 0): the dissolved clipped cell, every domain face
   * flagged ~m = ~1. */
  VD_BOX_2D = 3, VD_BOX_3D = 4
} vd_domain_kind;

/* Result of vd_compute: CSR arrays, 0-based, DEVICE pointers.
 *
 * Flags (P:L85, 0-based restatement): flag >= 0 is a site id j (the edge/face lies on the bisector
 * B_ij); flag < 0 means ~flag is the id of the simplex adjacent across that edge/face of T_a, with
 * ~flag == m marking a face on the domain boundary.
 *
 * cell i:   measure[i] = sum_a |P_{a,i}|,  centroid[i*dim..] = sum_a |P|.c(P) / measure[i];
 *           an empty cell has measure 0, centroid = the site itself, no pieces, no neighbours.
 *           nbr[nbr_off[i] .. nbr_off[i+1])   : ascending site ids j, each once, such that some piece
 *                                               of cell i has an edge/face on B_ij (restricted neighbours).
 *           pieces piece_off[i] .. piece_off[i+1], ascending simplex id piece_simplex[p].
 * piece p:  corners vert_off[p] .. vert_off[p+1]: vert_xyz[v*dim..], and vert_flags[v*nfl..] = the
 *           flags of the nfl edges/faces meeting at the corner, ascending (nfl = 2 for triangle
 *           kinds, 3 for tets); corners are sorted lexicographically by that flag tuple.
 */
typedef struct vd_cells {
  int64_t n;           /* number of sites = number of cells                                      */
  int32_t dim, nfl;
  int64_t n_nonempty, n_pieces, n_verts, n_nbrs;
  const double* measure;        /* [n]            */
  const double* centroid;       /* [n*dim]        */
  const int64_t* nbr_off;       /* [n+1]          */
  const int32_t* nbr;           /* [n_nbrs]       */
  const int64_t* piece_off;     /* [n+1]          */
  const int32_t* piece_simplex; /* [n_pieces]     */
  const double* piece_measure;  /* [n_pieces]     */
  const int64_t* vert_off;      /* [n_pieces+1]   */
  const double* vert_xyz;       /* [n_verts*dim]  */
  const int32_t* vert_flags;    /* [n_verts*nfl]  */
} vd_cells;

/* Tunables (P:L383 grid density; P:L369 step-out).  Zero / negative fields mean "default". */
typedef struct vd_options {
  double grid_density;    /* average sites per grid cell of the site index (default 2.0, measured; paper 2~4) */
  int32_t ball_cells;     /* one-shot bisector search (reading U18): most grid cells its ball
                             scan may cover; 0 = default (64); < 0: only the stepwise search of P:L137.
                             (The step-out of section VI-A, is not needed: U7.)            */
  int32_t real_edges;     /* 1 (default): search on a real edge p_s p_t when the outside corner has
                             a known-inside neighbour (Alg. 1); 0: always the virtual
                             edge from the pair's witness point (Alg. 3)               */
  int32_t persistent;     /* how S4 is scheduled (P:L257's wavefronts).  In every mode the wavefront loop runs on the
                             device ("wave programs": a fixed sequence of launches per wavefront, each kernel reading
                             from device memory whether it has work; the host looks once per batch of programs):
                             1 (default): 3D kinds "phased" -- every step of Alg. 3 is its own small kernel
                                over a whole wave, polytopes parked in HBM between steps (the one-kernel form is
                                bound by instruction fetch); 2D / surface kinds: one launch per wavefront;
                             2: phased (3D kinds), device-side queue (2D / surface kinds);
                             3: device-side work queue: one launch of the one-kernel form drains everything;
                             0: one launch of the one-kernel form per wavefront                          */
  int64_t pair_capacity;  /* initial capacity of the (simplex, site) pair list; grows on demand     */
  int64_t vert_capacity;  /* initial capacity of the corner pool; grows on demand                   */
  int32_t near_clips;     /* every piece of cell i is first clipped by the bisectors of this many of the
                             sites nearest to v_i (reading U19), so that the point-in-cell loop
                             starts from a small polytope; 0 = default: 24 for VD_BOX_3D; 16 for VD_TET_3D when at
                             least half of the sites lie inside the domain's bounding box and m <= 4 x that count
                             (decided on the device in every compute: cells about as large as the simplices or
                             smaller -- else the lists stay empty); > 0: that many, always; < 0: none; at most 32.
                             3D kinds only.                                                              */
  int32_t simplex_begin;  /* multi-GPU sharding: only simplices a in [simplex_begin, simplex_end) are   */
  int32_t simplex_end;    /* processed -- every piece P_{a,i} of such a simplex, and no other (pairs never leave their
                             simplex: propagation is by positive flags).  measure / centroid / neighbours /
                             pieces of a cell are then its PARTIAL sums over that block of M; ranks combine measure and
                             measure x centroid by one sum.  0, 0 (default) = all of M.  Meshed kinds only.            */
  int32_t tail_pairs;     /* phased schedule: a round that leaves at most this many pairs with a corner outside hands
                             them to one kernel that tests and clips them to completion (no further rounds for the
                             wave); 0 = default (65536); < 0: only what the program's rounds (`rounds`) leave             */
  int32_t first_clip;     /* 0 / 1 (default): a pair (T_a, v_i) discovered through the face of P_{a,u} on B_ui is first
                             clipped by that bisector, without a search -- the first clip of G_{a,j};
                             < 0: every clip is found by a search (Alg. 3 as printed).  3D kinds.                   */
  int32_t seed_corners;   /* corners of every simplex whose nearest site seeds a pair (Alg. 2 line 4): 0 = default
                             (1: the first corner, as in Alg. 2); >= 3 / 4: all of them.  The result does not depend
                             on it; discovered pairs are cheaper than seeds (first_clip).  Meshed kinds.             */
  int32_t small_wave;     /* phased schedule: a wavefront of fewer pairs than this is drained -- with every pair it sets
                             off -- by ONE launch of the one-kernel form as a device-side queue (the last wavefronts of a
                             step hold a few hundred pairs); 0 = default (8192); < 0: never (every wavefront phased)  */
  int32_t step_out;       /* improved bisector search of section VI-A: before the search on a segment p_s p_t
                             longer than 2 delta_i (delta_i = half the distance from v_i to its nearest other site, computed
                             for every site by S1b), step out from p_s: g = p_s + lambda delta_i dir, while N_g = v_i, then
                             search on p_s g.  0 (default): off (witness points keep segments short, U7);
                             1: lambda = 2, 3, 4, ... as printed;  2: lambda doubles.  Same result either way.     */
  int32_t dissolve;       /* Alg. 5 lines 2-6, VD_TET_3D on a CONVEX mesh only: sites whose cell does
                             not reach the domain boundary (empty restricted cell on the boundary triangles, site inside M)
                             get their WHOLE cell as one piece (piece_simplex = m, no simplex flags) from the whole-cell
                             kernel against the bounding box; the other (boundary) cells are clipped tet by tet as usual.
                             0 (default): every cell as per-simplex pieces.  VD_E_ARG when the mesh is not convex.        */
  int32_t fp32_filter;    /* 1: mixed precision -- every candidate site of a nearest-site query is first tested in fp32
                             (16-byte float records, a rigorous error bound on the squared distance from the coordinates'
                             magnitude); only the survivors are loaded and evaluated in fp64.  The paper's GPU runs are
                             fp32 throughout; here decisions and results stay fp64-exact (same cells, bit for bit in
                             structure).  0 (default): fp64 throughout.  Not combined with weighted 3-D sites.              */
  int32_t count_alg;      /* measurement runs.  0 (default): the clip kernels keep no per-query statistics (vd_counters.queries
                             and dist_evals count only the seeds' queries of the mesh vertices; row_evals and search_evals
                             stay 0: the bookkeeping alone is 3-4 % of a step) and no work counters of the clip path (clips,
                             pre_clips, search_iters, clip_corners, new_corners, fan_simplices stay 0: another 2-4 %);
                             1: statistics and work counters are collected (the "full" kernels run);  2: and D_alg as well
                             (vd_counters.alg_evals): after every nearest-site query the sites of the grid cells that meet
                             the ball (q, |q - N_q|) -- the least an exact grid search must examine; slower.    */
  int32_t reuse_nbrs;     /* vd_lloyd, whole-cell kinds: 0 / 1 (default): iteration k+1 clips every cell first by the bisectors
                             of its neighbours of iteration k instead of looking up the nearest sites again;
                             < 0: off                                                                                      */
  int32_t rounds;         /* phased schedule: rounds of {point-in-cell tests of all open corners, one search + clip per pair
                             with a corner outside} a wave program holds before its finishing kernel (which alternates tests
                             and clips per pair, Alg. 3's loop as printed, without parking the polytope in between).
                             0 = default, measured per kind: no rounds on tet meshes with the plain site index
                             (initialise, finishing kernel, emit), 3 in whole-cell mode, 5 on the refined (clustered) index;
                             1 ... 6: that many; < 0: none                                                                  */
  int32_t reserved[2];
} vd_options;

/* Work counters of the last vd_compute (a few atomics per warp and kernel).  Per-query statistics (queries, dist_evals, row_evals,
 * search_evals) and the clip path's work counters (search_iters, clips, pre_clips, clip_corners, new_corners, fan_simplices,
 * step_probes, f32_survivors) are collected only with vd_options.count_alg >= 1 (or another option that selects the full kernels:
 * step_out, fp32_filter, weighted 3-D sites) -- the default kernels carry no bookkeeping in their inner loops (it was 3-4 % + 2-4 %
 * of a step) and leave them 0.  pairs, pieces, waves, overflow_pairs, reruns, launches and syncs are counted always. */
typedef struct vd_counters {
  int64_t pairs;          /* (simplex, site) pairs processed = Alg. 3 runs          */
  int64_t pieces;         /* non-empty pieces                                                      */
  int64_t queries;        /* nearest-site queries = point-in-cell tests + seeds     */
  int64_t dist_evals;     /* site distance evaluations inside those queries                        */
  int64_t search_iters;   /* iterations of the edge-based bisector search                 */
  int64_t clips;          /* clippings performed                                    */
  int64_t waves;          /* wavefronts; 1 in persistent mode                       */
  int64_t overflow_pairs; /* pairs that needed the large-capacity path                             */
  int64_t reruns;         /* times the whole compute was repeated after growing a pool            */
  int64_t launches;       /* kernels this library launched inside the last vd_compute               */
  int64_t row_evals;      /* grid rows examined by those queries (index efficiency)                    */
  int64_t search_evals;   /* the part of dist_evals spent inside bisector searches                     */
  int64_t pre_clips;      /* the part of clips done without a search (discovery tuple, nearest sites)  */
  int64_t clip_corners;   /* corners side-tested by those clips (2d flop each)              */
  int64_t new_corners;    /* corners created by those clips (one 3 x 3 solve each in 3D)               */
  int64_t fan_simplices;  /* fan tetrahedra / triangles summed for measures and moments (S6 input)     */
  int64_t alg_evals;      /* D_alg (vd_options.count_alg), else 0                                      */
  int64_t syncs;          /* host waits on the stream inside the last vd_compute                       */
  int64_t step_probes;    /* step-out probes of section VI-A (vd_options.step_out)                     */
  int64_t f32_survivors;  /* vd_options.fp32_filter: candidates that passed the fp32 filter and were
                             evaluated in fp64 (the others of dist_evals cost 16 bytes and fp32 only)  */
  int64_t reserved[1];
} vd_counters;

/* vd_create: copy n sites of dimension dim (row-major [n][dim], fp64).  Builds nothing heavy: the
 * site index (line 1 of Alg. 2/4/5) is built inside vd_compute.
 * Errors: VD_E_ARG, VD_E_DIM, VD_E_INPUT (non-finite coordinate), VD_E_CUDA, VD_E_NOMEM. */
vd_status vd_create(const double* sites, int64_t n, int dim, vd_ctx** out);

/* vd_create_weighted: sites with weights w_i -- the POWER diagram (section VII-C): cell i =
 * { x : |x - v_i|^2 - w_i <= |x - v_j|^2 - w_j for all j }.  The paper lifts every site to p_i = (v_i, sqrt(eta - w_i))
 * in R^(d+1), eta >= max w, and restricts the Voronoi diagram of the lifted sites to the domain at height 0
 * (P:L465-471); the library does exactly that on the device: dim 2 -> lifted 3-D sites, the 2D triangle domain
 * becomes a flat surface (results stay 2-D: centroids and corners [..][2]); dim 3 -> lifted 4-D sites, whose fourth
 * coordinate enters every squared distance as the additive term eta - w_i (tets and boxes).
 * weights [n] fp64, host or device.  eta: NaN = the smallest admissible value max_i w_i (advised).
 * Errors: as vd_create; VD_E_INPUT when eta < max w or a weight is not finite.  Box kind in 2D: VD_E_DIM. */
vd_status vd_create_weighted(const double* sites, const double* weights, int64_t n, int dim, double eta, vd_ctx** out);

/* vd_update_sites: replace the coordinates of the n sites (same n, dim) -- for Lloyd iterations
 * (P:L483-492).  Same errors as vd_create. */
vd_status vd_update_sites(vd_ctx* ctx, const double* sites);

/* vd_lloyd: `iterations` steps of Lloyd's method with density 1 (section VII-D, Eq. 3): compute
 * the clipped / restricted cells, move every site with a non-empty cell to its cell's centroid, repeat; then
 * one more vd_compute so that *out_cells describes the final sites.  Everything stays on the device.
 * sites_out (host or device, [n][dim], may be NULL) receives the final sites.  Errors as vd_compute. */
vd_status vd_lloyd(vd_ctx* ctx, int iterations, vd_cells* out_cells, double* sites_out);

/* vd_set_domain: copy the domain M = {T_a}: verts [nv][dim] fp64, simplices [m][3]
 * (both triangle kinds) or [m][4] (tets), int32, 0-based, any orientation.  Derives the simplex
 * adjacency that initialises the edge/face flags (Fig. 2a).  May be called again.
 * Errors: VD_E_ARG, VD_E_DIM, VD_E_INPUT (index out of range, zero-measure simplex, an edge/face
 * shared by more than two simplices), VD_E_CUDA, VD_E_NOMEM. */
vd_status vd_set_domain(vd_ctx* ctx, const double* verts, int64_t nv, const int32_t* simplices, int64_t m,
                        vd_domain_kind kind);

/* vd_compute: the whole hot path -- site index, seeds, (simplex, site) clipping by point-in-cell
 * tests (Alg. 3/4/5), propagation over flags, assembly.  Asynchronous on the context's
 * stream except for one small read-back of counts at the end.  Fills *out_cells.
 * Errors: VD_E_ARG, VD_E_STATE, VD_E_CUDA, VD_E_NOMEM, VD_E_CAPACITY, VD_E_NOCONVERGE. */
vd_status vd_compute(vd_ctx* ctx, vd_cells* out_cells);

void vd_destroy(vd_ctx* ctx);

/* ---- support calls ---- */

/* Stream all later work of this context is issued on (e.g. torch.cuda.current_stream().cuda_stream). */
vd_status vd_set_stream(vd_ctx* ctx, void* cuda_stream);

/* Device allocator hooks (e.g. the torch caching allocator).  NULL restores cudaMalloc / cudaFree. */
vd_status vd_set_allocator(vd_ctx* ctx, void* (*alloc)(size_t bytes, void* user, void* stream),
                           void (*release)(void* ptr, void* user), void* user);

vd_status vd_set_options(vd_ctx* ctx, const vd_options* opt);
vd_status vd_get_counters(const vd_ctx* ctx, vd_counters* out);

/* Per-stage device times (ms, CUDA events) of the last vd_compute:
 * [0] site index (S1)  [1] seeds (S3)  [2] clip + propagate (S4+S5)  [3] assemble (S6)  [4] total. */
vd_status vd_get_stage_ms(const vd_ctx* ctx, double out_ms[5]);

/* Phased schedule (vd_options.persistent): device time (ms, CUDA events, summed over all launches) of the step
 * kernels of S4 in the last vd_compute: [0] k_ph_init  [1] k_ph_verify  [2] k_ph_fix  [3] k_ph_finish
 * [4] k_ph_tail (the last few pairs of a wave: tests and clips to completion in one launch); all 0 when another
 * schedule ran. */
vd_status vd_get_phase_ms(const vd_ctx* ctx, double out_ms[5]);

/* The work counters of the last vd_compute split by the kernel that did the work: which = 0 k_ph_init, 1 k_ph_verify,
 * 2 k_ph_fix, 3 k_ph_finish, 4 k_ph_tail, 5 every other kernel (one-kernel schedule, seeds).  Only the fields counted
 * inside kernels are filled (pairs .. step_probes); they add up to vd_get_counters.  bench.py derives each step kernel's
 * algorithmic flop from them. */
vd_status vd_get_phase_counters(const vd_ctx* ctx, int which, vd_counters* out);

/* Copy the last result into caller HOST buffers (any may be NULL to skip).  Sizes are those of
 * vd_cells.  Synchronises the context's stream. */
vd_status vd_cells_to_host(vd_ctx* ctx, double* measure, double* centroid, int64_t* nbr_off, int32_t* nbr,
                           int64_t* piece_off, int32_t* piece_simplex, double* piece_measure,
                           int64_t* vert_off, double* vert_xyz, int32_t* vert_flags);

/* Nearest site N_q of nq query points [nq][dim] through the site index (built on demand):
 * out_index[q] = argmin_j |q - v_j|, ties to the lowest id.  queries / out_index: host or device. */
vd_status vd_nearest(vd_ctx* ctx, const double* queries, int64_t nq, int32_t* out_index);

/* vd_nearest_static: vd_nearest for callers that must not allocate device memory (code next to a CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc).  Same result as vd_nearest; the call makes NO cudaMalloc / cudaFree or
 * other allocating call: queries and results are staged in one fixed device array inside the library (about 1.8 MB, held by
 * every GPU that loads libvd.so until the process exits).  Limits: nq <= 65536 per call (more: VD_E_ARG, with a message --
 * split the batch); the site index must already exist (VD_E_STATE otherwise: building it allocates -- run vd_compute or
 * vd_nearest once); every call of every context shares the array, which keeps the previous call's contents (the call clears
 * what must start at zero), so calls that overlap on the GPU race: one at a time.  queries / out_index: host or device.
 * Synchronises the context's stream.  Errors: VD_E_ARG, VD_E_STATE, VD_E_INPUT (non-finite query), VD_E_CUDA. */
vd_status vd_nearest_static(vd_ctx* ctx, const double* queries, int64_t nq, int32_t* out_index);

/* Sharded runs (vd_options.simplex_begin / simplex_end): vd_partial_moments writes, for every cell of
 * the last vd_compute, (measure, measure x centroid) = 1 + dim doubles per site into out [n][1 + dim] (DEVICE pointer,
 * caller-owned) -- the additive quantities the ranks sum with one all-reduce; vd_finish_centroids takes the summed
 * array back and rewrites the context's measure / centroid arrays from it (centroid = moment / measure; the site
 * itself for an empty cell).  Both run as kernels on the context's stream and do not synchronise. */
vd_status vd_partial_moments(vd_ctx* ctx, double* out_sums);
vd_status vd_finish_centroids(vd_ctx* ctx, const double* sums);

/* Simplex adjacency derived by vd_set_domain, [m][3 or 4] int32: adj[a][k] = simplex across the
 * edge/face opposite local corner k, or m on the domain boundary.  out: host or device. */
vd_status vd_get_adjacency(vd_ctx* ctx, int32_t* out);

/* Measurement support, not part of the path: the plain FP64 FMA rate of the current device (TFLOP/s, best of three
 * launches of a dependent-FMA-chain kernel on `cuda_stream`, 2 flop per FMA) -- the denominator of the "alu" roofline
 * that bench.py reports (the path's inner work is fp64 subtract / multiply-add / compare).
 * ms_out (may be NULL): duration of that launch.  Errors: VD_E_ARG, VD_E_CUDA, VD_E_NOMEM. */
vd_status vd_dfma_peak(void* cuda_stream, double* tflops_out, double* ms_out);

const char* vd_last_error(const vd_ctx* ctx);
const char* vd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* VD_H_ */
