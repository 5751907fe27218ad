// ia_internal.h - host-side context and the launcher interface between ia_api.cu and the kernel files.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ia.h"

namespace ia {

// dense grid descriptor (S9, G14): cell k of axis d is [edge(k), edge(k+1)], edge(k) = lo + k*w, edge(n) = hi
struct GridDesc {
  double lo[5], hi[5], w[5];
  int32_t n[5];
  int64_t cells;      // prod(n); for a slab (ia_vote_slab): the cells of the slab = the accumulator the vote writes
  int64_t col_cells;  // n[2]*n[3]*n[4]: cells of one (xc, yc) column
  int32_t ix0;        // dense vote: first xc cell voted and how many (the whole axis: 0, n[0]); edges are always those
  int32_t nx_run;     // of the full grid (n[0] cells on [lo[0], hi[0]])
};

// where the hits of event e live: staged[e*max_hits + i], i < count(e)
struct HitSpan {
  const ia_hit* hits;          // device
  const int32_t* offsets;      // device, n_events+1 entries, or nullptr: one event of n_hits_single hits
  int32_t n_hits_single;
  int32_t max_hits;            // slots per event in the staged array
  int32_t n_events;
};

struct Scratch {
  void* p = nullptr;
  size_t cap = 0;
};

}  // namespace ia

namespace ia {
// Cached CUDA graph of one refinement call (ia_refine / ia_refine_batch).  A refinement is a fixed sequence of
// small launches (C2: 38 of them for one event): the second call with the same arguments - same buffers, grid,
// parameters and scratch - is captured, later ones are one cudaGraphLaunch.  Any difference re-records.
struct RefineKey {
  HitSpan sp;
  double lo[5], hi[5];
  int32_t grid[5];
  int32_t levels, k;
  const void* boxes;
  const void* params_out;
  ia_params params;
  const void* wires;
  int64_t n_wires;
  const void* scratch[5];     // staged, votes, partial, keys, misc: the kernels of the graph point into them
};
struct RefineGraph {
  RefineKey key;
  int seen = 0;               // calls seen with this key (1: ran directly, 2+: graph)
  cudaGraphExec_t exec = nullptr;
  int64_t launches = 0;       // kernels inside the graph (for ia_launch_count)
};
}  // namespace ia

struct ia_ctx {
  int device = 0;
  cudaStream_t stream = nullptr;
  ia_params params{};
  // geometry SoA (a1)
  int n_wires = 0;
  double* wires = nullptr;   // 5 * n_wires doubles: x0 | y0 | sin | cos | tan
  double max_abs_tan = 0.0;
  double max_wire_r = 0.0;   // largest |(x0, y0)|: picks the dense kernel variant (performance only)
  // scratch, grown on demand, freed in ia_destroy
  ia::Scratch staged;        // HitC<T>[n_events * max_hits]
  ia::Scratch votes;         // uint16 dense votes of the refinement start grid
  ia::Scratch partial;       // uint16 partial child votes / uint64 partial top-K keys
  ia::Scratch keys;          // uint64 top-K keys
  ia::Scratch misc;          // idx / votes of internal top-K, host-variant device buffers
  ia::Scratch io_a, io_b, io_c, io_d;   // *_host entry points: device mirrors of host buffers
  int* status = nullptr;     // device: sticky error flag
  cudaStream_t copy_stream = nullptr;   // ia_vote_host: device->host copies of finished slabs, beside the vote
  cudaEvent_t slab_done = nullptr;
  int64_t host_slab_min = int64_t(16) << 20;   // ia_vote_host: smallest slab, in cells (ia_set_host_slab_min)
  int64_t launches = 0;
  int64_t graph_replays = 0;  // refinement calls served by cudaGraphLaunch
  cudaError_t last_err = cudaSuccess;
  ia::RefineGraph rgraph;
};

namespace ia {

// ---- programmatic dependent launch (sm_90+) --------------------------------------------------------
// A refinement is a chain of short dependent kernels (C2: 25 launches in 0.22 ms).  Launched with the
// programmatic-stream-serialization attribute, kernel N+1 does not wait for kernel N to be retired before it is launched:
// its blocks start as the last blocks of N leave and wait in griddepcontrol.wait - the first statement of every kernel
// of the chain, pdl_wait() - until the grids in front have completed and their writes are visible (it returns at once
// if there are none).  Nothing is read or written early, and completion stays transitive along the chain.  Only kernels
// that begin with pdl_wait() may be launched through launch_k.  IA_FLAG_NO_PDL switches the attribute off.
// Measured on C2: 0.2175 ms against 0.2249 replayed as a graph, 0.2187 against 0.2772 launched one by one.
#ifdef __CUDACC__
// (an early griddepcontrol.launch_dependents after the wait was tried: C2 0.222 ms against 0.2175 without it)
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <class... KArgs, class... Args>
cudaError_t launch_k(ia_ctx* ctx, void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = ctx->stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = (ctx->params.flags & IA_FLAG_NO_PDL) ? 0 : 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}
#endif

// All launchers enqueue on ctx->stream, bump ctx->launches and return the launch's cudaError_t.
// prec selects the endpoint type (64: double, 32: float).

cudaError_t launch_stage_hits(ia_ctx* ctx, const HitSpan& span);

cudaError_t launch_vote_dense(ia_ctx* ctx, const HitSpan& span, const GridDesc& g, uint16_t* votes_out);

// explicit boxes, one event: lo/hi [n_boxes][5]
cudaError_t launch_vote_boxes(ia_ctx* ctx, const HitSpan& span, const double* lo, const double* hi, int64_t n_boxes,
                              uint16_t* votes_out);

cudaError_t launch_residual(ia_ctx* ctx, const HitSpan& span, const double* lo, const double* hi, int64_t n_boxes,
                            double* out);

// the same record from the sign-specialised form of the dense kernel (ia_vote_dense.cu)
cudaError_t launch_residual_fast(ia_ctx* ctx, const HitSpan& span, const double* lo, const double* hi, int64_t n_boxes,
                                 double* out);

cudaError_t launch_prim(ia_ctx* ctx, int op, int prec, const double* a, const double* b, int64_t n, double* out);

// top-K of n_events independent arrays of n entries each (stride n): idx_out/votes_out [n_events][k]
// idx_base: added to every index (a slab of a larger accumulator); keys_out != nullptr: write the sorted 32-key list
// per event (first k entries, the rest 0) instead of idx_out/votes_out
cudaError_t launch_topk(ia_ctx* ctx, const uint16_t* votes, int64_t n, int n_events, int k, int64_t* idx_out,
                        uint16_t* votes_out, int64_t idx_base = 0, unsigned long long* keys_out = nullptr);
cudaError_t launch_merge_keys(ia_ctx* ctx, const unsigned long long* keys, int n_lists, int k, int64_t* idx_out,
                              uint16_t* votes_out);

// refinement steps (a8-a9)
cudaError_t launch_gather_dense(ia_ctx* ctx, const GridDesc& g, const int64_t* idx, const uint16_t* v, int n_events,
                                int k, int levels, ia_box* boxes_out);
// one level: children of boxes_out[e][lev-1][*] voted, top-k written to boxes_out[e][lev][*]
cudaError_t launch_refine_level(ia_ctx* ctx, const HitSpan& span, int lev, int levels, int k, ia_box* boxes_out);
// sign-specialised vote of the 32k children of every event (ia_vote_dense.cu); returns where the partial
// counts are and how many hit splits were used
cudaError_t launch_vote_children_fast(ia_ctx* ctx, const HitSpan& span, int lev, int levels, int k, int n_sm,
                                      ia_box* boxes, int* n_splits_out, uint16_t** partial_out);
cudaError_t launch_params(ia_ctx* ctx, int n_events, int levels, int k, const ia_box* boxes, double* params_out);

// paper mode (ia_vote_paper.cu).  PaperGrid: a fixed 4-D grid in g (axis 4 unused, n = 1), or - centre != nullptr -
// a window of half-widths `half` around a fit on the device (g then carries only the dims)
struct PaperGrid {
  GridDesc g;
  const ia_paper_fit* centre;   // previous pass: value[0..2] centre the window
  double half[4];
  const ia_paper_fit* self;     // this pass's slot: z0_centre (the previous z0 seen from this pass's reference point); may be nullptr
};
// ref (device, may be nullptr): the fit slot that holds the reference point of this pass; nullptr: ia_params'
cudaError_t launch_vote_paper(ia_ctx* ctx, const ia_hit* hits, int n_hits, const uint8_t* hit_mask, double P, double r_disk,
                              const PaperGrid& pg, int signs, const ia_paper_fit* ref, uint16_t* votes_out);   // votes_out [2][cells]; signs: bit 0 / 1
// keep_ref: fit_out already holds the reference point of its pass (ia_track_paper); else ia_params' is written
cudaError_t launch_select_max_paper(ia_ctx* ctx, const uint16_t* votes, const PaperGrid& pg, double P, int which,
                                    int keep_ref, ia_paper_fit* fit_out);
// F2d' (L98): next->x_ref, y_ref = the reference point of prev (move == 0; prev == nullptr: ia_params') or the wire point
// of the selected hit closest to prev's circle (move != 0)
cudaError_t launch_paper_ref(ia_ctx* ctx, const ia_hit* hits, int n_hits, const uint8_t* mask, const ia_paper_fit* prev, int move,
                             ia_paper_fit* next);
cudaError_t launch_find_hits_paper(ia_ctx* ctx, const ia_hit* hits, int n_hits, double P, const ia_paper_fit* fit, double factor,
                                   uint8_t* flags_out);
cudaError_t launch_paper_sign(ia_ctx* ctx, const ia_paper_fit* last, int32_t* sign_out);

// FP64 pipe probe (roofline denominator check): blocks x 256 threads x 8 chains x iters instructions
cudaError_t launch_fp64_probe(ia_ctx* ctx, int mode, int iters, int blocks, double* sink);

// scratch helper: grow-only device buffer
cudaError_t scratch_reserve(Scratch& s, size_t bytes);

}  // namespace ia
