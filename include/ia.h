/* ia.h - C ABI of libia_b200: the interval-arithmetic helix vote of arxiv 2401.04576 on one B200.
 *
 * Citations "L<n>" are line numbers of the paper text; "S<n>"/"G<n>" are the step and
 * reading numbers of DESIGN.md.
 *
 * The method (section 3.1): the 5-D helix parameter space (xc, yc, R, z0, lambda)
 * is tiled into interval boxes; a drift-distance hit votes for a box iff 0 lies in the interval
 * extension of the stereo-generalised Apollonius residual, eq. (2)/(A.5a) with d_Ax of (A.5b) and
 * Phi from the series (A.8a-d), for either drift sign (condition (4), L74-78).  The boxes with the
 * most votes are kept (L94) and, per BASELINE, subdivided into 2^5 children and voted again.
 *
 * Conventions
 *   - extern "C"; no exception crosses the boundary; every call returns IA_OK (0) or a negative
 *     IA_ERR_* code; ia_strerror() names it, ia_last_cuda_error() gives the CUDA error behind
 *     IA_ERR_CUDA.
 *   - Pointers named *_dev are DEVICE pointers owned by the caller (e.g. torch tensors'
 *     data_ptr()); pointers named *_host, the 5-element box/grid arrays, ia_wire[] and ia_params
 *     are HOST memory.  Nothing is retained after the call returns except what the context copies.
 *   - Calls enqueue work on the context's CUDA stream and do NOT synchronise; results are valid
 *     after the caller synchronises that stream.  The *_host entry points copy in and out with
 *     cudaMemcpyAsync on the same stream and DO synchronise before returning.
 *   - Errors that only the device can see (a hit naming an unknown wire) do not fail the call:
 *     the hit is dropped (it never votes) and a sticky flag is raised that ia_device_status()
 *     reads (it synchronises).  The *_host entry points validate hits on the host instead.
 *   - The library allocates device memory only inside the context (geometry, staged hits, child
 *     boxes, partial top-K lists, vote scratch) and frees it in ia_destroy().  No global state - with one
 *     exception, the fixed device array of ia_topk_static, the entry point for callers that must not allocate -
 *     and no CPU fallback: every step below runs in CUDA kernels compiled for sm_100a.
 *   - Units: cm and rad.  Order of the five axes everywhere: xc, yc, R, z0, lambda.
 */
#ifndef IA_B200_H
#define IA_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  IA_OK = 0,
  IA_ERR_ARG = -1,      /* null pointer, non-positive size, hi <= lo, k > number of cells ...       */
  IA_ERR_GEOMETRY = -2, /* no geometry loaded, or (host entry points) a hit names an unknown wire  */
  IA_ERR_DOMAIN = -3,   /* R.lo <= 0, or max|lambda| * max|tan tau| >= 0.5: u_d^2 > 0 and R+delta>0 */
                        /* of (A.3a)/(A.5b) cannot be guaranteed (G9)                               */
  IA_ERR_CAPACITY = -4, /* n_hits per event > IA_MAX_HITS, k > IA_MAX_K, too many cells             */
  IA_ERR_CUDA = -5      /* a CUDA runtime call failed; see ia_last_cuda_error()                     */
};

/* Hits per event.  SURVEY 8(b) proposed 65,535 (the range of the uint16 accumulator); the bound built is 1,024:
 * every vote kernel stages one event's hits in the shared memory of a CTA and reads them by broadcast
 * (120 B per hit in the explicit-box kernels, 184 B in the general dense kernel: 1,024 hits = 188 KB of the
 * 227 KB a CTA can have), and the paper's events hold 25-62 hits (L88).  More hits return IA_ERR_CAPACITY. */
#define IA_MAX_HITS 1024
#define IA_MAX_K 32      /* top-K list = one key per lane of a warp                                */
#define IA_N_PARAMS 20   /* doubles per event in params_out: centre[5], half-width[5], hull lo[5], hull hi[5]       */

typedef struct ia_ctx ia_ctx; /* opaque: device geometry, parameters, stream, scratch */

/* One sense wire, eq. (A.1a,b) L147-152: point (x0,y0) of the wire in the plane z=0, projection
 * angle phi_s (given as sin/cos, computed by the caller in double), signed tan of the stereo
 * angle tau.  half_len and layer are carried for the caller's benefit; the vote does not use
 * them.  40 bytes + 16. */
typedef struct {
  double x0, y0;
  double sin_phi_s, cos_phi_s;
  double tan_tau;
  double half_len;
  int32_t layer;
  int32_t _pad;
} ia_wire;

/* One hit, L88: "a hit is defined by this drift distance and the ... wire".  drift = |d_St| >= 0. */
typedef struct {
  int32_t wire; /* index into the loaded geometry */
  int32_t _pad;
  double drift; /* cm */
} ia_hit;

/* Bits of ia_params.flags.  Every bit but IA_FLAG_FULL_TURN, IA_FLAG_RIGOROUS_PHI leaves the results unchanged. */
enum {
  /* dense vote: the general, sign-agnostic kernel (interval DAG S4-S8 as written, (A.5b) L183 / (A.8a-c) L211-216)
   * instead of the sign-specialised one; same results, kept for cross-checks */
  IA_FLAG_GENERAL = 1u << 0,
  /* sign-specialised dense kernel: force the one-body variant (sign classes decided at run time; default for coarse
   * xy cells) ... */
  IA_FLAG_ONE_BODY = 1u << 1,
  /* ... or the three-body variant (one body per sign class of the hit; default for fine xy cells).  Same results:
   * the default is picked from the xy cell width for speed only */
  IA_FLAG_THREE_BODY = 1u << 2,
  /* paper-mode calls only: tracks of up to one turn emitted near the z axis (reading M6) - the
   * turning angle phi_Ax - phi0 of (A.8d) L218 is theta(wire point) - theta(reference point), theta in
   * [-0.3, 2 pi - 0.3) counted from the point of the base circle closest to the axis, instead of the principal value
   * in (-pi, pi] */
  IA_FLAG_FULL_TURN = 1u << 3,
  /* 5-D interval calls: Phi - Phi_Ax is not the series (A.8a-c) L211-216 but a verified enclosure of the fixed point of
   * the angular equation (A.6) L187 ("solved numerically", L220), obtained by inflation from the series enclosure
   * (reading f3): restores the guarantee of L80 at tol -> 0.  ia_vote runs it in the sign-specialised dense and
   * children kernels (several times the cost of the series mode), the explicit-box kernel in the general form */
  IA_FLAG_RIGOROUS_PHI = 1u << 4,
  /* ia_refine / ia_refine_batch always enqueue their launches one by one (default: a call repeated with identical
   * arguments and buffers is replayed as a CUDA graph from its third occurrence on) */
  IA_FLAG_NO_GRAPH = 1u << 5,
  /* sign-specialised dense kernel: before the fine evaluation of a hit a warp asks a crude enclosure of the same
   * residual (magnitude bounds of every step of S4-S8, both drift signs, all the z0 cells of its tile at once) whether
   * 0 can be excluded for all its cells, and skips the hit if so.  The votes are identical (a wider enclosure that
   * excludes 0 implies the finer one does, L80), but the kernel no longer evaluates every (cell, hit) in full -
   * default off: north_star's metric is the brute-force evaluation of condition (4) L74-78 */
  IA_FLAG_PREFILTER = 1u << 6,
  /* the kernels of the vote / top-K / refinement chain are launched without the programmatic-dependent-launch
   * attribute (default: with it - each of them starts by waiting for the kernels in front, so that its launch overlaps
   * their execution) */
  IA_FLAG_NO_PDL = 1u << 7,
  IA_FLAG_ALL = (1u << 8) - 1 /* other bits must be 0 (IA_ERR_ARG) */
};

/* tol: vote tolerance on the drift distance, D = [max(d-tol,0), d+tol] (S1, G6).
 * (x_ref, y_ref): reference point of eq. (1d); z_ref: reference plane of (A.4c-e) L172-176.
 * precision: 64 or 32 = type of the interval endpoints (G22).  flags: an OR of IA_FLAG_* bits. */
typedef struct {
  double tol;
  double x_ref, y_ref, z_ref;
  int32_t precision;
  uint32_t flags;
} ia_params;

/* A box with its vote count: 88 bytes. */
typedef struct {
  double lo[5], hi[5];
  uint16_t votes;
  uint16_t _pad[3];
} ia_box;

/* Create a context on CUDA device `device` that enqueues on `cuda_stream` (a cudaStream_t cast
 * to void*; NULL = the legacy default stream).  Parameters default to tol=0.045, ref=(0,0,0),
 * precision=64. */
int ia_create(ia_ctx** ctx_out, int device, void* cuda_stream);
void ia_destroy(ia_ctx* ctx);

/* a1 - copy the wires (HOST array, n_wires > 0) to a device SoA x0,y0,sin,cos,tan.  Replaces any
 * geometry loaded before.  Synchronises the stream. */
int ia_load_geometry(ia_ctx* ctx, const ia_wire* wires_host, int n_wires);
int ia_set_params(ia_ctx* ctx, const ia_params* params_host);

/* a2-a6 - dense single-level vote, condition (4) L74-78.  The box [box_lo, box_hi] is cut into
 * grid_dims[0..4] cells per axis, edges e_k = lo + k*((hi-lo)/n), e_n = hi (S9, G14);
 * votes_out_dev[((((ix*ny+iy)*nR+iR)*nz+iz)*nl+il)] = number of hits whose enclosure contains 0
 * for either drift sign (uint16, lambda fastest; prod(grid_dims) entries, at most 2^40). */
int ia_vote(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const double box_lo[5], const double box_hi[5],
            const int32_t grid_dims[5], uint16_t* votes_out_dev);

/* (e) SURVEY.md 8(e), "Dense vote: split the slowest axis (ix) across GPUs" - the same vote for the xc cells
 * [ix_begin, ix_end) of the grid only.  Cell edges are those of the FULL grid (e_k = lo + k*w with w = (hi-lo)/n over
 * all grid_dims[0] cells, G14), so the slabs of several calls - or of several GPUs - tile ia_vote's accumulator
 * exactly, count for count.  votes_out_dev holds (ix_end - ix_begin)*ny*nR*nz*nl counts: the slab, in the layout of
 * the full accumulator (a cell's index in it = its full-grid index - ix_begin*ny*nR*nz*nl).  An empty range is a no-op.
 * Errors as ia_vote; IA_ERR_ARG for a range outside [0, grid_dims[0]]. */
int ia_vote_slab(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const double box_lo[5], const double box_hi[5],
                 const int32_t grid_dims[5], int ix_begin, int ix_end, uint16_t* votes_out_dev);

/* Same vote on an explicit list of boxes: lo_dev/hi_dev are [n_boxes][5] doubles. */
int ia_vote_boxes(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const double* lo_dev, const double* hi_dev,
                  int64_t n_boxes, uint16_t* votes_out_dev);

/* f1 - the paper's own configuration of the vote (readings M1-M5 of DESIGN.md):
 * 4-D voxels xc x yc x R x z0 (L64), the momentum fixed to its true value - given as the length
 * momentum_radius = R sqrt(1 + lambda^2) (cm), so that |lambda| = sqrt((P/R_m)^2 - 1) at a voxel's mid
 * radius - and one accumulator per sign of lambda (L78).  d_Ax of (A.5b) is a NUMBER evaluated at the
 * voxel's mid-point in round-to-nearest double arithmetic (L82); only condition (4), L74-76,
 * 0 in (x_Ax - xc)^2 + (y_Ax - yc)^2 - (R + d_Ax)^2, is evaluated in intervals, for both drift signs,
 * one count per hit.  With tol > 0, d_Ax is the hull of its values at d - tol and d + tol; tol = 0 is
 * the paper's literal form.  Voxels whose mid radius exceeds momentum_radius have no lambda and get 0.
 * The guarantee "no vote => no solution in the voxel" does not hold in this mode (L80-82).
 * votes_out_dev[s*N + (((ix*ny+iy)*nR+iR)*nz+iz)], N = prod(grid_dims), s = 0: lambda >= 0, 1: lambda < 0
 * (2*N uint16, z0 fastest).  Always double precision (params.precision is not consulted).
 * Errors: IA_ERR_ARG (null, sizes, momentum_radius <= 0), IA_ERR_DOMAIN (box_lo[2] <= 0).
 * hit_mask_dev (may be NULL): uint8 per hit, 0 = the hit is not used (L96: "Only the selected hits are used
 * for the next iteration").  r_disk >= 0: disk pre-filter, conditions (3a),(3b) L66-70 - a voxel is
 * considered only if 0 in xc^2 + yc^2 - (R + [-r_disk, r_disk])^2 (interval arithmetic), the others get
 * 0 in both accumulators; r_disk < 0: no filter. */
int ia_vote_paper(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const uint8_t* hit_mask_dev, double momentum_radius,
                  double r_disk, const double box_lo[4], const double box_hi[4], const int32_t grid_dims[4],
                  uint16_t* votes_out_dev);

/* f2 (pieces of the paper's iteration scheme; readings F2b, F2c of DESIGN.md).
 * Result of the selection: 112 bytes. */
typedef struct {
  double value[4], error[4]; /* xc, yc, R, z0: centre of the mean cell index / half-extent of the selected voxels */
  double lambda;             /* signed, sqrt((P/value[2])^2 - 1); 0 if value[2] > P */
  int32_t lambda_sign;       /* +1: accumulator 0 holds the maximum (ties included), -1: accumulator 1 */
  int32_t vmax;              /* the maximum count */
  int64_t n_sel;             /* number of selected voxels */
  double x_ref, y_ref;       /* the reference point the pass was voted with: z0 = z where the helix is closest to it */
  double z0_centre;          /* ia_track_paper: the previous pass's z0 re-expressed for this pass's reference point */
} ia_paper_fit;

/* L94: "the values and the errors of the parameters are computed using voxels corresponding to selected
 * cells where the maximum of votes in the accumulator are found.  The central values and the size of the
 * selected voxels are used": vmax = the largest count of votes_dev[2][N] (as written by ia_vote_paper on
 * the same grid); the sign of lambda = the accumulator that holds it (L121); with k_d the cell indices of
 * the voxels of that accumulator whose count equals vmax,
 *   value_d = lo_d + ((2 sum k_d + n)/(2 n)) * w_d,   error_d = 0.5 * ((max k_d - min k_d + 1) * w_d),
 * w_d = (hi_d - lo_d)/n_d - integer sums, round-to-nearest unfused arithmetic, independent of any order.
 * fit_out_dev: DEVICE pointer.
 * which: 0 = the accumulator holding the larger maximum (ties: lambda >= 0), +1 / -1 = that accumulator. */
int ia_select_max_paper(ia_ctx* ctx, const uint16_t* votes_dev, double momentum_radius, const double box_lo[4],
                        const double box_hi[4], const int32_t grid_dims[4], int which, ia_paper_fit* fit_out_dev);

/* L96: "An multidimensional interval is constructed.  Its central value is given by the parameter values ...
 * and its radius is given by their errors multiplied by a factor of 5 ... One hit is selected when the
 * condition (4) is true for this multidimensional interval": flags_out_dev[h] = 1 iff the paper-mode
 * condition (4) holds for hit h on [value - factor*error, value + factor*error] (d_Ax at its mid-point,
 * lambda of the fit's sign, either drift sign).  fit_dev: DEVICE pointer (as written by
 * ia_select_max_paper), so that no host round trip separates the two calls. */
int ia_find_hits_paper(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, double momentum_radius, const ia_paper_fit* fit_dev,
                       double factor, uint8_t* flags_out_dev);

/* f2 - the paper's iteration scheme as one call, nothing returning to the host in between.
 * A pass is a fixed grid [lo, hi] x dims (Table 1, iterations 1-2) or, windowed != 0, a window of half-widths
 * lo[0..3] around the value found by the previous pass (iteration 3; hi is ignored).  Pass i votes its grid
 * (ia_vote_paper, disk pre-filter r_disk) with the hits found by pass i-1 - all hits for the first pass -,
 * selects the maximum-vote voxels (ia_select_max_paper) and finds the hits for the next pass on
 * value -/+ factor*error (ia_find_hits_paper; "all hits are always considered for the hit finding", L96).
 * "This procedure is applied for each sign of the lambda value" (L78): one chain per sign (reading F2e) -
 * fits_out_dev[pass][s], s = 0: lambda >= 0, 1: lambda < 0 - and sign_out_dev = +1 / -1 = the sign whose last
 * pass has the larger maximum (L121; ties: +1).
 * Reference point (L98, reading F2d' of DESIGN.md): the first pass is voted with the one of ia_set_params ("The
 * reference point is set to (0,0)"); a later pass with move_ref != 0 is voted with "the position of measurement point
 * closest to the recovered circle": of the hits the previous pass of its chain found, the one whose wire point in the
 * plane z = z_ref, (x_Ax, y_Ax) of (A.4d,e), minimises | |(x_Ax, y_Ax) - (xc, yc)| - R | for that pass's values
 * (round-to-nearest; ties: lowest hit index; no hit found: the point stays); move_ref == 0 keeps the previous pass's
 * point.  Every fit records the point of its pass, and its z0 is relative to it; a windowed pass is centred on the
 * previous pass's value with z0 re-expressed for the new point, z0 + lambda R (theta(new) - theta(old)).  With ia_params.flags bit 3 the turning angles are unwrapped independently of
 * the reference point (reading M6), which is what lets it move along a track of up to one turn.
 * passes_host: HOST; fits_out_dev (2*n_passes), sign_out_dev: DEVICE.  Windows are expected to stay inside R > 0.
 * The first pass must be a fixed grid with move_ref == 0. */
typedef struct {
  double lo[4], hi[4];
  int32_t dims[4];
  int32_t windowed;
  int32_t move_ref;
} ia_paper_pass;
int ia_track_paper(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, double momentum_radius, double r_disk, double factor,
                   const ia_paper_pass* passes_host, int n_passes, ia_paper_fit* fits_out_dev, int32_t* sign_out_dev);

/* a7 - the k largest entries by key (votes descending, index ascending) (L94, G16):
 * idx_out_dev[k] (int64 linear indices), votes_out_dev[k].  1 <= k <= min(n_cells, IA_MAX_K). */
int ia_topk(ia_ctx* ctx, const uint16_t* votes_dev, int64_t n_cells, int k, int64_t* idx_out_dev,
            uint16_t* votes_out_dev);

/* (e) SURVEY.md 8(e), the one exchange of the split dense vote ("all-gather of K (index, votes) pairs and a K-way
 * merge").  ia_topk_keys: the k best cells of one slab as keys_out_dev[IA_KEY_LIST] (uint64, sorted descending;
 * entries from k on are 0): key = votes << 48 | (2^48 - 1 - (index_base + index)) - larger key = more votes, then lower
 * index, the selection order of ia_topk (L94, G16) - with index_base the slab's first cell in the full accumulator
 * (ix_begin*ny*nR*nz*nl).  ia_merge_keys: n_lists such lists, rank after rank (what an all-gather of the lists
 * delivers), merged into the k best cells of the whole accumulator, idx_out_dev[k] / votes_out_dev[k] as ia_topk
 * writes them; entries of empty keys (fewer than k cells in all lists) come back as index 2^48 - 1, votes 0. */
#define IA_KEY_LIST 32
int ia_topk_keys(ia_ctx* ctx, const uint16_t* votes_dev, int64_t n_cells, int k, int64_t index_base, uint64_t* keys_out_dev);
int ia_merge_keys(ia_ctx* ctx, const uint64_t* keys_dev, int n_lists, int k, int64_t* idx_out_dev, uint16_t* votes_out_dev);

/* a7 again, for callers that must not allocate device memory.  ia_topk keeps the per-block candidate lists of its first
 * pass in a buffer of the context that it cudaMalloc's the first time it is needed and grows when a larger launch comes
 * along; ia_create allocates too.  That is a problem for three kinds of caller this library expects: an online event
 * filter that has handed the whole device to its framework's memory pool (a raw cudaMalloc behind the pool's back can fail
 * although memory is "free", and the pool's owner usually forbids it); a latency-bound loop (one event every few hundred
 * microseconds) in which cudaMalloc's implicit device-wide synchronisation stalls every other stream; and code that runs
 * while a stream is being captured, where cudaMalloc is not allowed at all.  ia_topk_static is the same selection (same
 * two kernels, same keys, same order: votes descending, index ascending, L94 / G16) with those lists in a fixed array
 * that is part of the library's device image: IA_TOPK_STATIC_BYTES = 256 KB per GPU, resident on every GPU that loads
 * the library's device code, from that moment until the process exits.  It takes no context: the device and the stream
 * are arguments, inputs and outputs stay the caller's (DEVICE pointers), and it calls no cudaMalloc, no cudaFree and no
 * library routine that allocates.
 *   - Limits: 1 <= k <= min(n_cells, IA_MAX_K); n_cells <= IA_TOPK_STATIC_MAX_CELLS (2^40, the accumulator bound of
 *     ia_vote); the first pass never uses more than IA_TOPK_STATIC_LISTS lists (it takes two blocks per SM, fewer on a
 *     small accumulator, and is cut to the array's capacity on a device that would want more).  Anything beyond these
 *     returns IA_ERR_CAPACITY (IA_ERR_ARG for null pointers, n_cells <= 0, k <= 0, k > n_cells, a device that does
 *     not exist) before anything is launched, and ia_topk_static_error() says which limit and by how much.
 *   - First call per device: the entry point asks the runtime where the array lives on that device (with the device
 *     current, return code checked) and remembers the answer; this is also what makes the driver load the library's
 *     device code there if nothing has yet.  Make that first call during set-up, before any stream capture begins.
 *   - The array is shared by every call on a device and keeps whatever the last call left in it.  Nothing in it has to
 *     start at zero: the merge pass reads exactly the lists the first pass of the same call has just written.  But two
 *     calls whose kernels can overlap on one GPU - different streams without an event between them, or two host threads -
 *     write the same lists and race; order them (one stream, or an event dependency).
 *   - Like the other calls it only enqueues: results are valid once the caller has synchronised cuda_stream
 *     (a cudaStream_t cast to void*; NULL = the legacy default stream). */
#define IA_TOPK_STATIC_LISTS 1024
#define IA_TOPK_STATIC_BYTES (IA_TOPK_STATIC_LISTS * 32 * 8)
#define IA_TOPK_STATIC_MAX_CELLS (((int64_t)1) << 40)
int ia_topk_static(int device, void* cuda_stream, const uint16_t* votes_dev, int64_t n_cells, int k, int64_t* idx_out_dev,
                   uint16_t* votes_out_dev);
/* Text describing why the calling thread's most recent ia_topk_static call failed ("" after a success).  The pointer
 * stays valid until that thread calls ia_topk_static again. */
const char* ia_topk_static_error(void);

/* a8-a9 - adaptive refinement of one event, entirely on the device: vote the dense grid0, keep the
 * top k, then (levels-1) times: cut every kept box at its per-axis midpoints into 2^5 children
 * (child c of rank r at list index r*32+c, bit (4-dim) of c set = upper half), vote the 32k
 * children, keep the top k.  boxes_out_dev[level][rank] (levels*k ia_box); params_out_dev[IA_N_PARAMS] =
 * centre (5) and half-width (5) of the rank-0 box of the last pass (L94, G19), then lower (5) and upper (5)
 * corner of the hull of the last pass's kept boxes whose votes equal rank 0's ("the cells where the maximum of
 * votes ... are found", L94). */
int ia_refine(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const double box_lo[5], const double box_hi[5],
              const int32_t grid0[5], int levels, int k, ia_box* boxes_out_dev, double* params_out_dev);

/* a10 - the same for n_events independent events in one launch sequence.  Hits in CSR form:
 * event e owns hits_dev[hit_offsets_dev[e] .. hit_offsets_dev[e+1]); max_hits_per_event bounds
 * every event's count (<= IA_MAX_HITS).  boxes_out_dev[n_events][levels][k], params_out_dev
 * [n_events][IA_N_PARAMS]. */
int ia_refine_batch(ia_ctx* ctx, const ia_hit* hits_dev, const int32_t* hit_offsets_dev, int n_events,
                    int max_hits_per_event, const double box_lo[5], const double box_hi[5], const int32_t grid0[5],
                    int levels, int k, ia_box* boxes_out_dev, double* params_out_dev);

/* End-to-end variants: every pointer is HOST memory (pinned for full copy speed).  They validate
 * the hits, copy them to the device, run the call above and copy the result back, then
 * synchronise the stream.  ia_vote_host sends a large accumulator in slabs of xc cells (the launches of
 * ia_vote_slab), slab i copied on a second stream while slab i+1 is voted: same counts.  The number of slabs is
 * min(8, grid_dims[0], cells / min_cells) with min_cells = 16 Mi cells (32 MB of counts) by default, and the split is
 * taken from 2 slabs on - that is, for accumulators of 64 MB and more.  On any error both streams are synchronised
 * before the call returns: nothing writes to votes_out_host afterwards. */
int ia_vote_host(ia_ctx* ctx, const ia_hit* hits_host, int n_hits, const double box_lo[5], const double box_hi[5],
                 const int32_t grid_dims[5], uint16_t* votes_out_host);
int ia_refine_batch_host(ia_ctx* ctx, const ia_hit* hits_host, const int32_t* hit_offsets_host, int n_events,
                         const double box_lo[5], const double box_hi[5], const int32_t grid0[5], int levels, int k,
                         ia_box* boxes_out_host, double* params_out_host);
/* Smallest slab of ia_vote_host, in cells (>= 1; default 16 Mi).  A tuning knob - smaller slabs start the first copy
 * earlier but add partial waves of blocks to every launch - and the handle by which the tests drive the slab pipeline
 * on small, ragged grids.  The counts do not depend on it. */
int ia_set_host_slab_min(ia_ctx* ctx, int64_t min_cells);

/* Diagnostics for parity tracing (G25): the enclosure f = R_Ax^2 - (R + d_Ax)^2 of every
 * (box, hit, drift sign): out_dev[((b*n_hits + h)*2 + s)*4 + {0,1,2,3}] = f.lo, f.hi,
 * scale = max(Q.hi, |rad|), forced (1 if a domain rule forced the vote, G15); s = 0 for +d. */
int ia_residual(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const double* lo_dev, const double* hi_dev,
                int64_t n_boxes, double* out_dev);

/* The same record from the sign-specialised ("fast") form that the dense and children kernels run, for the cell
 * [lo, hi] taken as a one-cell grid: slot 3 = form (0: fast form, scale = R_Ax^2.hi; 1: forced vote; 2: this
 * (box, hit) takes the general form - guards of the fast form, lambda straddling 0 - whose enclosure is written;
 * 3: invalid hit).  The two forms enclose the same function f of eq. (2) with different roundings; the tests bound
 * their difference (the FP32 variant uses the fast form as a filter in front of the general one). */
int ia_residual_fast(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const double* lo_dev, const double* hi_dev,
                     int64_t n_boxes, double* out_dev);

/* Device interval primitives exposed for unit tests: n independent operations
 * out_dev[i] = op(a_dev[i], b_dev[i]) on intervals stored as (lo, hi) pairs of doubles; prec = 64 or 32.
 * op: 0 add 1 sub 2 mul 3 sqr(a) 4 div(a, b>0) 5 sqrt(a) 6 sin(a) 7 cos(a) 8 atan2(y=a, x=b)
 *     9 recip(a>0) 10 scale(b.lo, a)
 *     primitives of the dense fast path (enclosures at most a few ulps wider than the tightest):
 *     11 a*b with a >= 0 taken in midpoint-radius form  12 the same for a of any sign
 *     13 a / sqrt(b) for a >= 0 and b in [1/4, 4] (delta = d_St/u_d of S6, one fused enclosure)
 *     14 sqr(a) branch-free  15 sin(a), 16 cos(a) for a inside [-1/4, 1/4] (Taylor, padded)
 *     17 a intersected with [-1, 1]  18 sin(a), 19 cos(a) for a inside (-1, 1) (longer Taylor forms, padded) */
int ia_prim(ia_ctx* ctx, int op, int prec, const double* a_dev, const double* b_dev, int64_t n, double* out_dev);

/* Roofline probe: enqueue a kernel of `blocks` x 256 threads, each running 8 independent FP64
 * dependency chains for `iters` rounds (blocks*256*8*iters FP64 instructions in total).
 * mode 0: DFMA round-to-nearest; 1: DADD.RM / DMUL.RP alternating; 2: DFMA.RM / DFMA.RP alternating;
 * 3, 4, 5: DFMA.RM / DFMA.RP on only 1, 2, 4 independent chains per thread (same instruction count);
 * 6, 7: mode 2 with one independent integer (LOP3) resp. FP32 (FFMA) instruction after every DFMA - do
 * non-FP64 instructions issue in the shadow of the FP64 pipe?  (only the DFMAs are counted);
 * 8, 9: DFMA.RM/RP with three distinct register operands, DMUL.RM/DADD.RP with two (the modes above take
 * the multiplier and the addend from uniform registers) - is operand fetch a limit?
 * 10, 11: mode 8 with the multiplier register shared by 4 resp. 2 consecutive DFMAs (operand reuse cache).
 * The caller times it with events on the context's stream.  sink_dev: one double, never written. */
int ia_probe_fp64(ia_ctx* ctx, int mode, int iters, int blocks, double* sink_dev);

/* Synchronise the stream and return IA_OK, IA_ERR_GEOMETRY (a hit named an unknown wire since
 * the last call of this function) or IA_ERR_CUDA. */
int ia_device_status(ia_ctx* ctx);

/* Number of kernels this context has launched so far (for the bench's gpu_launches). */
int64_t ia_launch_count(const ia_ctx* ctx);

/* Number of ia_refine / ia_refine_batch calls of this context that were served by replaying the cached CUDA graph of
 * the call (third identical call on; needs a capturable stream, i.e. not the legacy default stream). */
int64_t ia_graph_replays(const ia_ctx* ctx);

const char* ia_strerror(int code);
const char* ia_last_cuda_error(const ia_ctx* ctx);
/* Outward padding of the sin/cos/atan2 enclosures, in ulps (lower bound of the relative pad). */
int ia_pad_ulps(void);

#ifdef __cplusplus
}
#endif
#endif /* IA_B200_H */
