// ia_api.cu - the C ABI of include/ia.h: argument checks, scratch management, launch sequences.
// Every computation is in the kernels; nothing here touches votes, boxes or hits on the host except
// the *_host entry points' copies and their hit validation.
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "ia_internal.h"

using namespace ia;

namespace {

struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(int dev) {
    cudaGetDevice(&prev);
    if (prev != dev) cudaSetDevice(dev);
  }
  ~DeviceGuard() {
    int cur = -1;
    cudaGetDevice(&cur);
    if (prev >= 0 && cur != prev) cudaSetDevice(prev);
  }
};

int fail_cuda(ia_ctx* ctx, cudaError_t err) {
  ctx->last_err = err;
  cudaGetLastError();  // clear the sticky flag of launch-configuration errors
  return IA_ERR_CUDA;
}

#define IA_CUDA(ctx, expr)                                 \
  do {                                                     \
    cudaError_t _e = (expr);                               \
    if (_e != cudaSuccess) return fail_cuda((ctx), _e);    \
  } while (0)

int make_grid(const double lo[5], const double hi[5], const int32_t n[5], GridDesc& g) {
  if (!lo || !hi || !n) return IA_ERR_ARG;
  g.cells = 1;
  for (int d = 0; d < 5; ++d) {
    if (n[d] <= 0 || !(hi[d] > lo[d]) || !std::isfinite(lo[d]) || !std::isfinite(hi[d])) return IA_ERR_ARG;
    g.lo[d] = lo[d];
    g.hi[d] = hi[d];
    g.n[d] = n[d];
    // (hi-lo)/n in round-to-nearest, unfused: two separate IEEE operations (S9, G14)
    volatile double span = hi[d] - lo[d];
    volatile double w = span / double(n[d]);
    g.w[d] = w;
    if (g.cells > (int64_t(1) << 40) / n[d]) return IA_ERR_CAPACITY;
    g.cells *= n[d];
  }
  g.col_cells = int64_t(n[2]) * n[3] * n[4];
  g.ix0 = 0;
  g.nx_run = n[0];
  if (int64_t(n[0]) * n[1] * ((g.col_cells + 1023) / 1024) > 0x7fffffffLL) return IA_ERR_CAPACITY;
  return IA_OK;
}

// R.lo > 0 (G9) and max|lambda| max|tan tau| < 0.5 so that u_d^2 of (A.3a) stays positive
int check_domain(const ia_ctx* ctx, const double lo[5], const double hi[5]) {
  if (!(lo[2] > 0.0)) return IA_ERR_DOMAIN;
  const double lmax = std::fmax(std::fabs(lo[4]), std::fabs(hi[4]));
  if (!(lmax * ctx->max_abs_tan < 0.5)) return IA_ERR_DOMAIN;
  return IA_OK;
}

int check_ready(const ia_ctx* ctx) {
  if (!ctx) return IA_ERR_ARG;
  if (ctx->n_wires <= 0 || !ctx->wires) return IA_ERR_GEOMETRY;
  return IA_OK;
}

HitSpan single_span(const ia_hit* hits, int n_hits) {
  HitSpan sp;
  sp.hits = hits;
  sp.offsets = nullptr;
  sp.n_hits_single = n_hits;
  sp.max_hits = n_hits;
  sp.n_events = 1;
  return sp;
}

int refine_impl(ia_ctx* ctx, const HitSpan& sp, const double lo[5], const double hi[5], const int32_t grid0[5],
                int levels, int k, ia_box* boxes_out, double* params_out) {
  GridDesc g;
  int rc = make_grid(lo, hi, grid0, g);
  if (rc) return rc;
  if (levels < 1 || k < 1 || !boxes_out || !params_out) return IA_ERR_ARG;
  if (k > g.cells) return IA_ERR_ARG;
  if (k > IA_MAX_K || sp.n_events > 65535) return IA_ERR_CAPACITY;
  rc = check_domain(ctx, lo, hi);
  if (rc) return rc;
  // the same call again (same buffers, grid, parameters, scratch): replay its CUDA graph
  RefineKey key;
  std::memset(&key, 0, sizeof(key));
  key.sp.hits = sp.hits; key.sp.offsets = sp.offsets; key.sp.n_hits_single = sp.n_hits_single;
  key.sp.max_hits = sp.max_hits; key.sp.n_events = sp.n_events;          // field by field: no padding bytes copied
  for (int d = 0; d < 5; ++d) { key.lo[d] = lo[d]; key.hi[d] = hi[d]; key.grid[d] = grid0[d]; }
  key.levels = levels; key.k = k; key.boxes = boxes_out; key.params_out = params_out;
  std::memcpy(&key.params, &ctx->params, sizeof(ia_params));
  key.wires = ctx->wires;
  key.n_wires = ctx->n_wires;
  auto fill_scratch = [&](RefineKey& kk) {
    kk.scratch[0] = ctx->staged.p; kk.scratch[1] = ctx->votes.p; kk.scratch[2] = ctx->partial.p;
    kk.scratch[3] = ctx->keys.p; kk.scratch[4] = ctx->misc.p;
  };
  fill_scratch(key);
  RefineGraph& rg = ctx->rgraph;
  const bool use_graphs = !(ctx->params.flags & IA_FLAG_NO_GRAPH);
  const bool same = rg.seen > 0 && std::memcmp(&rg.key, &key, sizeof(key)) == 0;
  if (use_graphs && same && rg.exec) {
    IA_CUDA(ctx, cudaGraphLaunch(rg.exec, ctx->stream));
    ctx->graph_replays++;
    ctx->launches += rg.launches;
    return IA_OK;
  }
  auto enqueue = [&]() -> cudaError_t {
    const int ne = sp.n_events;
    cudaError_t e = launch_stage_hits(ctx, sp);
    if (e != cudaSuccess) return e;
    // level 0: dense start grid -> top k -> boxes
    if ((e = scratch_reserve(ctx->votes, size_t(ne) * g.cells * sizeof(uint16_t))) != cudaSuccess) return e;
    uint16_t* votes = static_cast<uint16_t*>(ctx->votes.p);
    if ((e = launch_vote_dense(ctx, sp, g, votes)) != cudaSuccess) return e;
    if ((e = scratch_reserve(ctx->misc, size_t(ne) * k * (sizeof(int64_t) + sizeof(uint16_t)) + 64)) != cudaSuccess) return e;
    int64_t* idx = static_cast<int64_t*>(ctx->misc.p);
    uint16_t* kv = reinterpret_cast<uint16_t*>(idx + size_t(ne) * k);
    if ((e = launch_topk(ctx, votes, g.cells, ne, k, idx, kv)) != cudaSuccess) return e;
    if ((e = launch_gather_dense(ctx, g, idx, kv, ne, k, levels, boxes_out)) != cudaSuccess) return e;
    // levels 1..: subdivide, vote the children, keep the top k - all stream-ordered, no host round trip
    for (int lev = 1; lev < levels; ++lev)
      if ((e = launch_refine_level(ctx, sp, lev, levels, k, boxes_out)) != cudaSuccess) return e;
    return launch_params(ctx, ne, levels, k, boxes_out, params_out);
  };
  if (use_graphs && same && rg.seen == 1) {
    // second identical call: the scratch buffers have their final sizes (no allocation inside the capture)
    const int64_t l0 = ctx->launches;
    cudaGraph_t graph = nullptr;
    cudaError_t e = cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal);
    if (e == cudaSuccess) {
      const cudaError_t eq = enqueue();
      e = cudaStreamEndCapture(ctx->stream, &graph);
      if (eq != cudaSuccess) e = eq;
    }
    const int64_t n_launch = ctx->launches - l0;
    ctx->launches = l0;
    if (e == cudaSuccess && graph) e = cudaGraphInstantiate(&rg.exec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (e == cudaSuccess && rg.exec) {
      rg.launches = n_launch;
      rg.seen = 2;
      IA_CUDA(ctx, cudaGraphLaunch(rg.exec, ctx->stream));
      ctx->graph_replays++;
      ctx->launches += rg.launches;
      return IA_OK;
    }
    // capture not possible here (e.g. the caller's stream is already capturing): run directly from now on
    cudaGetLastError();
    rg.exec = nullptr;
    rg.seen = 3;
  }
  IA_CUDA(ctx, enqueue());
  if (!same) {
    if (rg.exec) cudaGraphExecDestroy(rg.exec);
    rg.exec = nullptr;
    rg.seen = 1;
    fill_scratch(key);           // the pointers after this call's reservations
    rg.key = key;
  }
  return IA_OK;
}

int validate_hits_host(const ia_ctx* ctx, const ia_hit* hits, int64_t n) {
  for (int64_t i = 0; i < n; ++i) {
    if (hits[i].wire < 0 || hits[i].wire >= ctx->n_wires) return IA_ERR_GEOMETRY;
    if (!(hits[i].drift >= 0.0)) return IA_ERR_ARG;
  }
  return IA_OK;
}

}  // namespace

extern "C" {

int ia_create(ia_ctx** ctx_out, int device, void* cuda_stream) {
  if (!ctx_out) return IA_ERR_ARG;
  *ctx_out = nullptr;
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || device < 0 || device >= n_dev) {
    cudaGetLastError();
    return IA_ERR_CUDA;
  }
  ia_ctx* ctx = new (std::nothrow) ia_ctx();
  if (!ctx) return IA_ERR_ARG;
  ctx->device = device;
  ctx->stream = static_cast<cudaStream_t>(cuda_stream);
  ctx->params.tol = 0.045;
  ctx->params.x_ref = ctx->params.y_ref = ctx->params.z_ref = 0.0;
  ctx->params.precision = 64;
  ctx->params.flags = 0;
  DeviceGuard guard(device);
  if (cudaMalloc(&ctx->status, sizeof(int)) != cudaSuccess || cudaMemset(ctx->status, 0, sizeof(int)) != cudaSuccess) {
    cudaGetLastError();
    delete ctx;
    return IA_ERR_CUDA;
  }
  *ctx_out = ctx;
  return IA_OK;
}

void ia_destroy(ia_ctx* ctx) {
  if (!ctx) return;
  DeviceGuard guard(ctx->device);
  cudaStreamSynchronize(ctx->stream);
  Scratch* all[] = {&ctx->staged, &ctx->votes, &ctx->partial, &ctx->keys, &ctx->misc,
                    &ctx->io_a,   &ctx->io_b,  &ctx->io_c,    &ctx->io_d};
  for (Scratch* s : all)
    if (s->p) cudaFree(s->p);
  if (ctx->rgraph.exec) cudaGraphExecDestroy(ctx->rgraph.exec);
  if (ctx->copy_stream) { cudaStreamSynchronize(ctx->copy_stream); cudaStreamDestroy(ctx->copy_stream); }
  if (ctx->slab_done) cudaEventDestroy(ctx->slab_done);
  if (ctx->wires) cudaFree(ctx->wires);
  if (ctx->status) cudaFree(ctx->status);
  delete ctx;
}

int ia_load_geometry(ia_ctx* ctx, const ia_wire* wires_host, int n_wires) {
  if (!ctx || !wires_host || n_wires <= 0) return IA_ERR_ARG;
  DeviceGuard guard(ctx->device);
  std::vector<double> soa(size_t(5) * n_wires);
  double tmax = 0.0, rmax = 0.0;
  for (int i = 0; i < n_wires; ++i) {
    const ia_wire& w = wires_host[i];
    if (!std::isfinite(w.x0) || !std::isfinite(w.y0) || !std::isfinite(w.sin_phi_s) || !std::isfinite(w.cos_phi_s) ||
        !std::isfinite(w.tan_tau))
      return IA_ERR_ARG;
    soa[i] = w.x0;
    soa[size_t(n_wires) + i] = w.y0;
    soa[size_t(2) * n_wires + i] = w.sin_phi_s;
    soa[size_t(3) * n_wires + i] = w.cos_phi_s;
    soa[size_t(4) * n_wires + i] = w.tan_tau;
    tmax = std::fmax(tmax, std::fabs(w.tan_tau));
    rmax = std::fmax(rmax, std::hypot(w.x0, w.y0));
  }
  IA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  if (ctx->wires) cudaFree(ctx->wires);
  ctx->wires = nullptr;
  ctx->n_wires = 0;
  IA_CUDA(ctx, cudaMalloc(&ctx->wires, soa.size() * sizeof(double)));
  IA_CUDA(ctx, cudaMemcpyAsync(ctx->wires, soa.data(), soa.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
  IA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  ctx->n_wires = n_wires;
  ctx->max_abs_tan = tmax;
  ctx->max_wire_r = rmax;
  return IA_OK;
}

int ia_set_params(ia_ctx* ctx, const ia_params* p) {
  if (!ctx || !p) return IA_ERR_ARG;
  if (!(p->tol >= 0.0) || !std::isfinite(p->tol) || !std::isfinite(p->x_ref) || !std::isfinite(p->y_ref) ||
      !std::isfinite(p->z_ref))
    return IA_ERR_ARG;
  if (p->precision != 64 && p->precision != 32) return IA_ERR_ARG;
  if (p->flags & ~unsigned(IA_FLAG_ALL)) return IA_ERR_ARG;
  ctx->params = *p;
  return IA_OK;
}

int ia_vote(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const double box_lo[5], const double box_hi[5],
            const int32_t grid_dims[5], uint16_t* votes_out_dev) {
  int rc = check_ready(ctx);
  if (rc) return rc;
  if (n_hits < 0 || (n_hits > 0 && !hits_dev) || !votes_out_dev) return IA_ERR_ARG;
  if (n_hits > IA_MAX_HITS) return IA_ERR_CAPACITY;
  GridDesc g;
  rc = make_grid(box_lo, box_hi, grid_dims, g);
  if (rc) return rc;
  rc = check_domain(ctx, box_lo, box_hi);
  if (rc) return rc;
  DeviceGuard guard(ctx->device);
  HitSpan sp = single_span(hits_dev, n_hits);
  IA_CUDA(ctx, launch_stage_hits(ctx, sp));
  IA_CUDA(ctx, launch_vote_dense(ctx, sp, g, votes_out_dev));
  return IA_OK;
}

int ia_vote_slab(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const double box_lo[5], const double box_hi[5],
                 const int32_t grid_dims[5], int ix_begin, int ix_end, uint16_t* votes_out_dev) {
  int rc = check_ready(ctx);
  if (rc) return rc;
  if (n_hits < 0 || (n_hits > 0 && !hits_dev) || !votes_out_dev) return IA_ERR_ARG;
  if (n_hits > IA_MAX_HITS) return IA_ERR_CAPACITY;
  GridDesc g;
  rc = make_grid(box_lo, box_hi, grid_dims, g);
  if (rc) return rc;
  if (ix_begin < 0 || ix_end > g.n[0] || ix_begin > ix_end) return IA_ERR_ARG;
  rc = check_domain(ctx, box_lo, box_hi);
  if (rc) return rc;
  if (ix_begin == ix_end) return IA_OK;                   // an empty slab (more ranks than xc cells)
  // the edges stay those of the full grid (cell_edge with n[0] cells on [lo[0], hi[0]], G14); only the range of xc
  // cells and the accumulator the blocks write - the slab - change
  g.ix0 = ix_begin;
  g.nx_run = ix_end - ix_begin;
  g.cells = int64_t(g.nx_run) * g.n[1] * g.col_cells;
  DeviceGuard guard(ctx->device);
  HitSpan sp = single_span(hits_dev, n_hits);
  IA_CUDA(ctx, launch_stage_hits(ctx, sp));
  IA_CUDA(ctx, launch_vote_dense(ctx, sp, g, votes_out_dev));
  return IA_OK;
}

static int make_grid4(const double box_lo[4], const double box_hi[4], const int32_t grid_dims[4], GridDesc& g) {
  if (!box_lo || !box_hi || !grid_dims) return IA_ERR_ARG;
  const double lo5[5] = {box_lo[0], box_lo[1], box_lo[2], box_lo[3], 0.0};
  const double hi5[5] = {box_hi[0], box_hi[1], box_hi[2], box_hi[3], 1.0};
  const int32_t n5[5] = {grid_dims[0], grid_dims[1], grid_dims[2], grid_dims[3], 1};
  int rc = make_grid(lo5, hi5, n5, g);
  if (rc) return rc;
  if (int64_t(grid_dims[0]) * grid_dims[1] > 0x7fffffffLL || int64_t(grid_dims[2]) * grid_dims[3] > 0x7fffffffLL)
    return IA_ERR_CAPACITY;
  return IA_OK;
}

int ia_vote_paper(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const uint8_t* hit_mask_dev, double momentum_radius,
                  double r_disk, const double box_lo[4], const double box_hi[4], const int32_t grid_dims[4],
                  uint16_t* votes_out_dev) {
  int rc = check_ready(ctx);
  if (rc) return rc;
  if (n_hits < 0 || (n_hits > 0 && !hits_dev) || !votes_out_dev) return IA_ERR_ARG;
  if (!(momentum_radius > 0.0) || !std::isfinite(momentum_radius) || std::isnan(r_disk)) return IA_ERR_ARG;
  if (n_hits > IA_MAX_HITS) return IA_ERR_CAPACITY;
  GridDesc g;
  rc = make_grid4(box_lo, box_hi, grid_dims, g);
  if (rc) return rc;
  if (!(box_lo[2] > 0.0)) return IA_ERR_DOMAIN;
  DeviceGuard guard(ctx->device);
  PaperGrid pg = {g, nullptr, {0, 0, 0, 0}, nullptr};
  IA_CUDA(ctx, launch_vote_paper(ctx, hits_dev, n_hits, hit_mask_dev, momentum_radius, r_disk, pg, 3, nullptr, votes_out_dev));
  return IA_OK;
}

int ia_select_max_paper(ia_ctx* ctx, const uint16_t* votes_dev, double momentum_radius, const double box_lo[4],
                        const double box_hi[4], const int32_t grid_dims[4], int which, ia_paper_fit* fit_out_dev) {
  if (!ctx || !votes_dev || !fit_out_dev || !(momentum_radius > 0.0) || which < -1 || which > 1) return IA_ERR_ARG;
  GridDesc g;
  int rc = make_grid4(box_lo, box_hi, grid_dims, g);
  if (rc) return rc;
  DeviceGuard guard(ctx->device);
  PaperGrid pg = {g, nullptr, {0, 0, 0, 0}, nullptr};
  IA_CUDA(ctx, launch_select_max_paper(ctx, votes_dev, pg, momentum_radius, which, 0, fit_out_dev));
  return IA_OK;
}

int ia_find_hits_paper(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, double momentum_radius, const ia_paper_fit* fit_dev,
                       double factor, uint8_t* flags_out_dev) {
  int rc = check_ready(ctx);
  if (rc) return rc;
  if (n_hits < 0 || (n_hits > 0 && (!hits_dev || !flags_out_dev)) || !fit_dev) return IA_ERR_ARG;
  if (!(momentum_radius > 0.0) || !(factor > 0.0) || !std::isfinite(factor)) return IA_ERR_ARG;
  DeviceGuard guard(ctx->device);
  IA_CUDA(ctx, launch_find_hits_paper(ctx, hits_dev, n_hits, momentum_radius, fit_dev, factor, flags_out_dev));
  return IA_OK;
}

int ia_track_paper(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, double momentum_radius, double r_disk, double factor,
                   const ia_paper_pass* passes_host, int n_passes, ia_paper_fit* fits_out_dev, int32_t* sign_out_dev) {
  int rc = check_ready(ctx);
  if (rc) return rc;
  if (n_hits <= 0 || !hits_dev || !passes_host || n_passes < 1 || !fits_out_dev || !sign_out_dev) return IA_ERR_ARG;
  if (!(momentum_radius > 0.0) || !(factor > 0.0) || std::isnan(r_disk) || passes_host[0].windowed || passes_host[0].move_ref)
    return IA_ERR_ARG;
  if (n_hits > IA_MAX_HITS) return IA_ERR_CAPACITY;
  std::vector<PaperGrid> grids(n_passes);
  int64_t max_cells = 0;
  for (int i = 0; i < n_passes; ++i) {
    const ia_paper_pass& ps = passes_host[i];
    if (ps.windowed) {
      // dims only; lo/hi are placeholders that make_grid4 accepts, the kernels rebuild them from the centre
      const double zero[4] = {0, 0, 0, 0}, one[4] = {1, 1, 1, 1};
      rc = make_grid4(zero, one, ps.dims, grids[i].g);
      for (int d = 0; d < 4; ++d) {
        if (!(ps.lo[d] > 0.0) || !std::isfinite(ps.lo[d])) return IA_ERR_ARG;
        grids[i].half[d] = ps.lo[d];
      }
    } else {
      rc = make_grid4(ps.lo, ps.hi, ps.dims, grids[i].g);
      if (!rc && !(ps.lo[2] > 0.0)) rc = IA_ERR_DOMAIN;
    }
    if (rc) return rc;
    grids[i].centre = nullptr;
    grids[i].self = nullptr;
    max_cells = std::max(max_cells, grids[i].g.cells);
  }
  DeviceGuard guard(ctx->device);
  IA_CUDA(ctx, scratch_reserve(ctx->votes, size_t(2) * max_cells * sizeof(uint16_t)));
  IA_CUDA(ctx, scratch_reserve(ctx->misc, size_t(2) * n_hits));
  uint16_t* votes = static_cast<uint16_t*>(ctx->votes.p);
  uint8_t* mask[2] = {static_cast<uint8_t*>(ctx->misc.p), static_cast<uint8_t*>(ctx->misc.p) + n_hits};
  for (int i = 0; i < n_passes; ++i) {
    for (int s = 0; s < 2; ++s) {
      PaperGrid pg = grids[i];
      ia_paper_fit* fit = fits_out_dev + i * 2 + s;
      if (passes_host[i].windowed) { pg.centre = fit - 2; pg.self = fit; }
      // the reference point of this pass goes into its fit slot first: ia_params' for the first pass, then the previous
      // pass's of the chain, moved along the track where the pass asks for it (F2d', L98)
      IA_CUDA(ctx, launch_paper_ref(ctx, hits_dev, n_hits, i == 0 ? nullptr : mask[s], i == 0 ? nullptr : fit - 2,
                                    i > 0 && passes_host[i].move_ref ? 1 : 0, fit));
      // the first pass is the same vote for both chains (all hits, fixed grid, same reference point): voted once
      if (i > 0 || s == 0)
        IA_CUDA(ctx, launch_vote_paper(ctx, hits_dev, n_hits, i == 0 ? nullptr : mask[s], momentum_radius, r_disk, pg,
                                       i == 0 ? 3 : (s == 0 ? 1 : 2), fit, votes));
      IA_CUDA(ctx, launch_select_max_paper(ctx, votes, pg, momentum_radius, s == 0 ? +1 : -1, 1, fit));
      IA_CUDA(ctx, launch_find_hits_paper(ctx, hits_dev, n_hits, momentum_radius, fit, factor, mask[s]));
    }
  }
  IA_CUDA(ctx, launch_paper_sign(ctx, fits_out_dev + (n_passes - 1) * 2, sign_out_dev));
  return IA_OK;
}

int ia_vote_boxes(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const double* lo_dev, const double* hi_dev,
                  int64_t n_boxes, uint16_t* votes_out_dev) {
  int rc = check_ready(ctx);
  if (rc) return rc;
  if (n_hits < 0 || (n_hits > 0 && !hits_dev) || n_boxes < 0 || (n_boxes > 0 && (!lo_dev || !hi_dev || !votes_out_dev)))
    return IA_ERR_ARG;
  if (n_hits > IA_MAX_HITS) return IA_ERR_CAPACITY;
  DeviceGuard guard(ctx->device);
  HitSpan sp = single_span(hits_dev, n_hits);
  IA_CUDA(ctx, launch_stage_hits(ctx, sp));
  IA_CUDA(ctx, launch_vote_boxes(ctx, sp, lo_dev, hi_dev, n_boxes, votes_out_dev));
  return IA_OK;
}

int ia_topk(ia_ctx* ctx, const uint16_t* votes_dev, int64_t n_cells, int k, int64_t* idx_out_dev,
            uint16_t* votes_out_dev) {
  if (!ctx || !votes_dev || !idx_out_dev || !votes_out_dev || n_cells <= 0 || k <= 0 || k > n_cells) return IA_ERR_ARG;
  if (k > IA_MAX_K || n_cells > (int64_t(1) << 40)) return IA_ERR_CAPACITY;
  DeviceGuard guard(ctx->device);
  IA_CUDA(ctx, launch_topk(ctx, votes_dev, n_cells, 1, k, idx_out_dev, votes_out_dev));
  return IA_OK;
}

int ia_topk_keys(ia_ctx* ctx, const uint16_t* votes_dev, int64_t n_cells, int k, int64_t index_base, uint64_t* keys_out_dev) {
  if (!ctx || !votes_dev || !keys_out_dev || n_cells <= 0 || k <= 0 || k > n_cells || index_base < 0) return IA_ERR_ARG;
  if (k > IA_MAX_K || n_cells > (int64_t(1) << 40) || index_base > (int64_t(1) << 40)) return IA_ERR_CAPACITY;
  DeviceGuard guard(ctx->device);
  IA_CUDA(ctx, launch_topk(ctx, votes_dev, n_cells, 1, k, nullptr, nullptr, index_base,
                           reinterpret_cast<unsigned long long*>(keys_out_dev)));
  return IA_OK;
}

int ia_merge_keys(ia_ctx* ctx, const uint64_t* keys_dev, int n_lists, int k, int64_t* idx_out_dev, uint16_t* votes_out_dev) {
  if (!ctx || !keys_dev || !idx_out_dev || !votes_out_dev || n_lists <= 0 || k <= 0) return IA_ERR_ARG;
  if (k > IA_MAX_K || n_lists > 65535) return IA_ERR_CAPACITY;
  DeviceGuard guard(ctx->device);
  IA_CUDA(ctx, launch_merge_keys(ctx, reinterpret_cast<const unsigned long long*>(keys_dev), n_lists, k, idx_out_dev,
                                 votes_out_dev));
  return IA_OK;
}

int ia_refine(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const double box_lo[5], const double box_hi[5],
              const int32_t grid0[5], int levels, int k, ia_box* boxes_out_dev, double* params_out_dev) {
  int rc = check_ready(ctx);
  if (rc) return rc;
  if (n_hits < 0 || (n_hits > 0 && !hits_dev)) return IA_ERR_ARG;
  if (n_hits > IA_MAX_HITS) return IA_ERR_CAPACITY;
  DeviceGuard guard(ctx->device);
  return refine_impl(ctx, single_span(hits_dev, n_hits), box_lo, box_hi, grid0, levels, k, boxes_out_dev, params_out_dev);
}

int ia_refine_batch(ia_ctx* ctx, const ia_hit* hits_dev, const int32_t* hit_offsets_dev, int n_events,
                    int max_hits_per_event, const double box_lo[5], const double box_hi[5], const int32_t grid0[5],
                    int levels, int k, ia_box* boxes_out_dev, double* params_out_dev) {
  int rc = check_ready(ctx);
  if (rc) return rc;
  if (n_events <= 0 || !hit_offsets_dev || max_hits_per_event < 0 || (max_hits_per_event > 0 && !hits_dev))
    return IA_ERR_ARG;
  if (max_hits_per_event > IA_MAX_HITS) return IA_ERR_CAPACITY;
  DeviceGuard guard(ctx->device);
  HitSpan sp;
  sp.hits = hits_dev;
  sp.offsets = hit_offsets_dev;
  sp.n_hits_single = 0;
  sp.max_hits = max_hits_per_event;
  sp.n_events = n_events;
  return refine_impl(ctx, sp, box_lo, box_hi, grid0, levels, k, boxes_out_dev, params_out_dev);
}

int ia_vote_host(ia_ctx* ctx, const ia_hit* hits_host, int n_hits, const double box_lo[5], const double box_hi[5],
                 const int32_t grid_dims[5], uint16_t* votes_out_host) {
  int rc = check_ready(ctx);
  if (rc) return rc;
  if (n_hits < 0 || (n_hits > 0 && !hits_host) || !votes_out_host) return IA_ERR_ARG;
  GridDesc g;
  rc = make_grid(box_lo, box_hi, grid_dims, g);
  if (rc) return rc;
  rc = validate_hits_host(ctx, hits_host, n_hits);
  if (rc) return rc;
  DeviceGuard guard(ctx->device);
  IA_CUDA(ctx, scratch_reserve(ctx->io_a, size_t(n_hits) * sizeof(ia_hit) + 16));
  IA_CUDA(ctx, scratch_reserve(ctx->io_b, size_t(g.cells) * sizeof(uint16_t)));
  if (n_hits > 0)
    IA_CUDA(ctx, cudaMemcpyAsync(ctx->io_a.p, hits_host, size_t(n_hits) * sizeof(ia_hit), cudaMemcpyHostToDevice, ctx->stream));
  uint16_t* acc = static_cast<uint16_t*>(ctx->io_b.p);
  const ia_hit* hits_dev = static_cast<const ia_hit*>(ctx->io_a.p);
  // A large accumulator (C4: 2.1 GB, 38 ms of PCIe after 1.2 s of vote) goes out in slabs of xc cells: slab i is copied
  // on a second stream while slab i+1 is voted (ia_vote_slab's launch: same edges, same counts), so only the last copy
  // is exposed.  At most 8 slabs of at least host_slab_min cells (16 M = 32 MB unless ia_set_host_slab_min changed it):
  // more would add partial waves of blocks to every launch.
  const int64_t slab_min = ctx->host_slab_min;
  int n_slabs = int(std::min<int64_t>(std::min<int64_t>(8, g.n[0]), g.cells / slab_min));
  if (n_slabs < 2) {
    rc = ia_vote(ctx, hits_dev, n_hits, box_lo, box_hi, grid_dims, acc);
    if (rc) return rc;
    IA_CUDA(ctx, cudaMemcpyAsync(votes_out_host, acc, size_t(g.cells) * sizeof(uint16_t), cudaMemcpyDeviceToHost, ctx->stream));
    IA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
    return IA_OK;
  }
  rc = check_domain(ctx, box_lo, box_hi);
  if (rc) return rc;
  if (n_hits > IA_MAX_HITS) return IA_ERR_CAPACITY;
  if (!ctx->copy_stream) IA_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
  if (!ctx->slab_done) IA_CUDA(ctx, cudaEventCreateWithFlags(&ctx->slab_done, cudaEventDisableTiming));
  HitSpan sp = single_span(hits_dev, n_hits);
  IA_CUDA(ctx, launch_stage_hits(ctx, sp));
  const int64_t per_ix = g.cells / g.n[0];
  auto pipeline = [&]() -> cudaError_t {
    cudaError_t e;
    for (int i = 0; i < n_slabs; ++i) {
      const int b0 = int(int64_t(g.n[0]) * i / n_slabs), e0 = int(int64_t(g.n[0]) * (i + 1) / n_slabs);
      GridDesc gs = g;
      gs.ix0 = b0;
      gs.nx_run = e0 - b0;
      gs.cells = per_ix * gs.nx_run;
      if ((e = launch_vote_dense(ctx, sp, gs, acc + per_ix * b0)) != cudaSuccess) return e;
      if ((e = cudaEventRecord(ctx->slab_done, ctx->stream)) != cudaSuccess) return e;
      if ((e = cudaStreamWaitEvent(ctx->copy_stream, ctx->slab_done, 0)) != cudaSuccess) return e;
      if ((e = cudaMemcpyAsync(votes_out_host + per_ix * b0, acc + per_ix * b0, size_t(gs.cells) * sizeof(uint16_t),
                               cudaMemcpyDeviceToHost, ctx->copy_stream)) != cudaSuccess)
        return e;
    }
    return cudaSuccess;
  };
  const cudaError_t pe = pipeline();
  // success or not, nothing may still be writing into the caller's buffer when this call returns
  const cudaError_t s1 = cudaStreamSynchronize(ctx->stream);
  const cudaError_t s2 = cudaStreamSynchronize(ctx->copy_stream);
  IA_CUDA(ctx, pe);
  IA_CUDA(ctx, s1);
  IA_CUDA(ctx, s2);
  return IA_OK;
}

int ia_set_host_slab_min(ia_ctx* ctx, int64_t min_cells) {
  if (!ctx || min_cells < 1) return IA_ERR_ARG;
  ctx->host_slab_min = min_cells;
  return IA_OK;
}

int ia_refine_batch_host(ia_ctx* ctx, const ia_hit* hits_host, const int32_t* hit_offsets_host, int n_events,
                         const double box_lo[5], const double box_hi[5], const int32_t grid0[5], int levels, int k,
                         ia_box* boxes_out_host, double* params_out_host) {
  int rc = check_ready(ctx);
  if (rc) return rc;
  if (n_events <= 0 || !hit_offsets_host || !boxes_out_host || !params_out_host || levels < 1 || k < 1) return IA_ERR_ARG;
  int max_hits = 0;
  if (hit_offsets_host[0] != 0) return IA_ERR_ARG;
  for (int e = 0; e < n_events; ++e) {
    const int c = hit_offsets_host[e + 1] - hit_offsets_host[e];
    if (c < 0) return IA_ERR_ARG;
    if (c > max_hits) max_hits = c;
  }
  const int64_t total = hit_offsets_host[n_events];
  if (total > 0 && !hits_host) return IA_ERR_ARG;
  if (max_hits > IA_MAX_HITS) return IA_ERR_CAPACITY;
  rc = validate_hits_host(ctx, hits_host, total);
  if (rc) return rc;
  DeviceGuard guard(ctx->device);
  const size_t nb = size_t(n_events) * levels * k;
  IA_CUDA(ctx, scratch_reserve(ctx->io_a, size_t(total) * sizeof(ia_hit) + 16));
  IA_CUDA(ctx, scratch_reserve(ctx->io_b, size_t(n_events + 1) * sizeof(int32_t)));
  IA_CUDA(ctx, scratch_reserve(ctx->io_c, nb * sizeof(ia_box)));
  IA_CUDA(ctx, scratch_reserve(ctx->io_d, size_t(n_events) * IA_N_PARAMS * sizeof(double)));
  if (total > 0)
    IA_CUDA(ctx, cudaMemcpyAsync(ctx->io_a.p, hits_host, size_t(total) * sizeof(ia_hit), cudaMemcpyHostToDevice, ctx->stream));
  IA_CUDA(ctx, cudaMemcpyAsync(ctx->io_b.p, hit_offsets_host, size_t(n_events + 1) * sizeof(int32_t), cudaMemcpyHostToDevice,
                               ctx->stream));
  rc = ia_refine_batch(ctx, static_cast<const ia_hit*>(ctx->io_a.p), static_cast<const int32_t*>(ctx->io_b.p), n_events,
                       max_hits, box_lo, box_hi, grid0, levels, k, static_cast<ia_box*>(ctx->io_c.p),
                       static_cast<double*>(ctx->io_d.p));
  if (rc) return rc;
  IA_CUDA(ctx, cudaMemcpyAsync(boxes_out_host, ctx->io_c.p, nb * sizeof(ia_box), cudaMemcpyDeviceToHost, ctx->stream));
  IA_CUDA(ctx, cudaMemcpyAsync(params_out_host, ctx->io_d.p, size_t(n_events) * IA_N_PARAMS * sizeof(double), cudaMemcpyDeviceToHost,
                               ctx->stream));
  IA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  return IA_OK;
}

int ia_residual(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const double* lo_dev, const double* hi_dev,
                int64_t n_boxes, double* out_dev) {
  int rc = check_ready(ctx);
  if (rc) return rc;
  if (n_hits <= 0 || !hits_dev || n_boxes <= 0 || !lo_dev || !hi_dev || !out_dev) return IA_ERR_ARG;
  if (n_hits > IA_MAX_HITS) return IA_ERR_CAPACITY;
  DeviceGuard guard(ctx->device);
  HitSpan sp = single_span(hits_dev, n_hits);
  IA_CUDA(ctx, launch_stage_hits(ctx, sp));
  IA_CUDA(ctx, launch_residual(ctx, sp, lo_dev, hi_dev, n_boxes, out_dev));
  return IA_OK;
}

int ia_residual_fast(ia_ctx* ctx, const ia_hit* hits_dev, int n_hits, const double* lo_dev, const double* hi_dev,
                     int64_t n_boxes, double* out_dev) {
  int rc = check_ready(ctx);
  if (rc) return rc;
  if (n_hits <= 0 || !hits_dev || n_boxes <= 0 || !lo_dev || !hi_dev || !out_dev) return IA_ERR_ARG;
  if (n_hits > IA_MAX_HITS) return IA_ERR_CAPACITY;
  DeviceGuard guard(ctx->device);
  HitSpan sp = single_span(hits_dev, n_hits);
  IA_CUDA(ctx, launch_stage_hits(ctx, sp));
  IA_CUDA(ctx, launch_residual_fast(ctx, sp, lo_dev, hi_dev, n_boxes, out_dev));
  return IA_OK;
}

int ia_prim(ia_ctx* ctx, int op, int prec, const double* a_dev, const double* b_dev, int64_t n, double* out_dev) {
  if (!ctx || !a_dev || !out_dev || n < 0 || op < 0 || op > 19 || (prec != 64 && prec != 32)) return IA_ERR_ARG;
  const bool binary = (op == 0 || op == 1 || op == 2 || op == 4 || op == 8 || op == 10 || op == 11 || op == 12 || op == 13);
  if (binary && !b_dev) return IA_ERR_ARG;
  DeviceGuard guard(ctx->device);
  IA_CUDA(ctx, launch_prim(ctx, op, prec, a_dev, b_dev, n, out_dev));
  return IA_OK;
}

int ia_probe_fp64(ia_ctx* ctx, int mode, int iters, int blocks, double* sink_dev) {
  if (!ctx || !sink_dev || mode < 0 || mode > 11 || iters <= 0 || blocks <= 0) return IA_ERR_ARG;
  DeviceGuard guard(ctx->device);
  IA_CUDA(ctx, launch_fp64_probe(ctx, mode, iters, blocks, sink_dev));
  return IA_OK;
}

int ia_device_status(ia_ctx* ctx) {
  if (!ctx) return IA_ERR_ARG;
  DeviceGuard guard(ctx->device);
  int flag = 0;
  IA_CUDA(ctx, cudaMemcpyAsync(&flag, ctx->status, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
  IA_CUDA(ctx, cudaMemsetAsync(ctx->status, 0, sizeof(int), ctx->stream));
  IA_CUDA(ctx, cudaStreamSynchronize(ctx->stream));
  return flag ? IA_ERR_GEOMETRY : IA_OK;
}

int64_t ia_launch_count(const ia_ctx* ctx) { return ctx ? ctx->launches : 0; }

int64_t ia_graph_replays(const ia_ctx* ctx) { return ctx ? ctx->graph_replays : 0; }

const char* ia_strerror(int code) {
  switch (code) {
    case IA_OK: return "ok";
    case IA_ERR_ARG: return "invalid argument";
    case IA_ERR_GEOMETRY: return "no geometry loaded, or a hit names an unknown wire";
    case IA_ERR_DOMAIN: return "parameter box outside the domain (R.lo <= 0 or max|lambda|*max|tan tau| >= 0.5)";
    case IA_ERR_CAPACITY: return "capacity exceeded (hits per event, k, or number of cells)";
    case IA_ERR_CUDA: return "CUDA error";
    default: return "unknown error code";
  }
}

const char* ia_last_cuda_error(const ia_ctx* ctx) { return cudaGetErrorString(ctx ? ctx->last_err : cudaSuccess); }

int ia_pad_ulps(void) { return 4; }

}  // extern "C"
