// ia_kernels.cu - hit staging (a2), explicit-box vote, refinement level (a8-a9), diagnostics.
#include "ia_internal.h"
#include "ia_residual.cuh"
#include "ia_fast.cuh"
#include "ia_topk.cuh"

namespace ia {

cudaError_t scratch_reserve(Scratch& s, size_t bytes) {
  if (bytes <= s.cap) return cudaSuccess;
  if (s.p) cudaFree(s.p);
  s.p = nullptr;
  s.cap = 0;
  size_t want = bytes + bytes / 4 + 256;
  cudaError_t err = cudaMalloc(&s.p, want);
  if (err == cudaSuccess) s.cap = want;
  return err;
}

namespace {

// ---- a2: staging ------------------------------------------------------------------------------
// per-hit scalars of S1-S3 in round-to-nearest, unfused (__dmul_rn/__dadd_rn are never contracted).
// FP32 mode converts every scalar input to float first and then computes in float.
template <class T>
__device__ HitC<T> make_hitc(const double* __restrict__ wires, int n_wires, ia_hit h, ia_params p, int* status) {
  using R = Rnd<T>;
  HitC<T> c;
  int w = h.wire;
  c.valid = (w >= 0 && w < n_wires && h.drift >= 0.0);
  if (!c.valid) {
    if (status) atomicOr(status, 1);
    w = 0;
    h.drift = 0.0;
  }
  const T x0 = R::from_rn(wires[w]), y0 = R::from_rn(wires[n_wires + w]);
  const T s = R::from_rn(wires[2 * n_wires + w]), co = R::from_rn(wires[3 * n_wires + w]);
  const T t = R::from_rn(wires[4 * n_wires + w]);
  const T xr = R::from_rn(p.x_ref), yr = R::from_rn(p.y_ref), zr = R::from_rn(p.z_ref);
  c.sphi = s; c.cphi = co; c.Tn = t;
  c.xA = R::add_rn(x0, R::mul_rn(R::mul_rn(zr, s), t));          // (A.4d) L174
  c.yA = R::add_rn(y0, -R::mul_rn(R::mul_rn(zr, co), t));        // (A.4e) L176
  c.k0 = R::add_rn(R::mul_rn(xr, c.yA), -R::mul_rn(yr, c.xA));
  c.ky = R::add_rn(yr, -c.yA);
  c.kx = R::add_rn(c.xA, -xr);
  c.mx = R::mul_rn(T(0.5), R::add_rn(xr, c.xA));
  c.my = R::mul_rn(T(0.5), R::add_rn(yr, c.yA));
  const T hx = R::mul_rn(T(0.5), R::add_rn(c.xA, -xr)), hy = R::mul_rn(T(0.5), R::add_rn(c.yA, -yr));
  c.h2 = R::add_rn(R::mul_rn(hx, hx), R::mul_rn(hy, hy));
  const T d = R::from_rn(h.drift), tol = R::from_rn(p.tol);
  c.Dlo = mx(R::add_dn(d, -tol), T(0));                          // S1 (G6)
  c.Dhi = R::add_up(d, tol);
  c.zref = zr;
  c._pad = (p.flags & IA_FLAG_RIGOROUS_PHI) ? 1 : 0;        // rigorous-Phi mode travels with the staged hit (HitS::rig)
  return c;
}

__device__ __forceinline__ void event_hits(const HitSpan& sp, int e, int& first, int& count) {
  if (sp.offsets) {
    first = sp.offsets[e];
    count = sp.offsets[e + 1] - first;
    if (count > sp.max_hits) count = sp.max_hits;
    if (count < 0) count = 0;
  } else {
    first = 0;
    count = sp.n_hits_single;
  }
}

template <class T>
__global__ void stage_hits_kernel(HitSpan sp, const double* __restrict__ wires, int n_wires, ia_params p,
                                  HitC<T>* __restrict__ staged, int* status) {
  pdl_wait();                 // programmatic dependent launch: nothing before the kernels in front have completed
  const int e = blockIdx.x;
  int first, count;
  event_hits(sp, e, first, count);
  for (int i = threadIdx.x; i < count; i += blockDim.x)
    staged[int64_t(e) * sp.max_hits + i] = make_hitc<T>(wires, n_wires, sp.hits[first + i], p, status);
}

// ---- explicit-box vote: one thread per box, hits broadcast from shared memory --------------------
template <class T>
__global__ void __launch_bounds__(128)
vote_boxes_kernel(HitSpan sp, const HitC<T>* __restrict__ staged, const double* __restrict__ lo,
                  const double* __restrict__ hi, int64_t n_boxes, uint16_t* __restrict__ votes) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  HitC<T>* sh = reinterpret_cast<HitC<T>*>(smem_raw);
  int first, count;
  event_hits(sp, 0, first, count);
  for (int i = threadIdx.x; i < count; i += blockDim.x) sh[i] = staged[i];
  __syncthreads();
  const int64_t b = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
  if (b >= n_boxes) return;
  const Iv<T> X = box_iv<T>(lo[5 * b + 0], hi[5 * b + 0]), Y = box_iv<T>(lo[5 * b + 1], hi[5 * b + 1]);
  Box3<T> bx = {box_iv<T>(lo[5 * b + 2], hi[5 * b + 2]), box_iv<T>(lo[5 * b + 3], hi[5 * b + 3]),
                box_iv<T>(lo[5 * b + 4], hi[5 * b + 4])};
  unsigned v = 0;
  for (int h = 0; h < count; ++h) {
    const HitC<T> c = sh[h];
    const XYInv<T> inv = xy_invariants(X, Y, c);
    v += hit_votes_general(bx, inv, hit_small(c), c.zref) ? 1u : 0u;
  }
  votes[b] = uint16_t(v);
}

// ---- diagnostics: f enclosure per (box, hit, sign) -----------------------------------------------
template <class T>
__global__ void residual_kernel(HitSpan sp, const HitC<T>* __restrict__ staged, const double* __restrict__ lo,
                                const double* __restrict__ hi, int64_t n_boxes, double* __restrict__ out) {
  const int n_hits = sp.n_hits_single;
  const int64_t t = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
  if (t >= n_boxes * n_hits) return;
  const int64_t b = t / n_hits;
  const int h = int(t - b * n_hits);
  const HitC<T> c = staged[h];
  const Iv<T> X = box_iv<T>(lo[5 * b + 0], hi[5 * b + 0]), Y = box_iv<T>(lo[5 * b + 1], hi[5 * b + 1]);
  Box3<T> bx = {box_iv<T>(lo[5 * b + 2], hi[5 * b + 2]), box_iv<T>(lo[5 * b + 3], hi[5 * b + 3]),
                box_iv<T>(lo[5 * b + 4], hi[5 * b + 4])};
  const XYInv<T> inv = xy_invariants(X, Y, c);
  for (int s = 0; s < 2; ++s) {
    Resid r = residual_general(bx, inv, hit_small(c), c.zref, s == 0 ? +1 : -1);
    double* o = out + (t * 2 + s) * 4;
    o[0] = r.flo; o[1] = r.fhi; o[2] = r.scale; o[3] = r.forced ? 1.0 : 0.0;
  }
}

// ---- primitives exposed for unit tests ---------------------------------------------------------
template <class T>
__global__ void prim_kernel(int op, const double* __restrict__ a, const double* __restrict__ b, int64_t n,
                            double* __restrict__ out) {
  const int64_t i = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
  if (i >= n) return;
  Iv<T> x = {T(a[2 * i]), T(a[2 * i + 1])}, y = {T(0), T(0)}, r = {T(0), T(0)};
  if (b) y = {T(b[2 * i]), T(b[2 * i + 1])};
  switch (op) {
    case 0: r = iadd(x, y); break;
    case 1: r = isub(x, y); break;
    case 2: r = imul(x, y); break;
    case 3: r = isqr(x); break;
    case 4: r = idiv_pos(x, y); break;
    case 5: r = isqrt(x); break;
    case 6: r = isin(x); break;
    case 7: r = icos(x); break;
    case 8: r = iatan2(x, y); break;
    case 9: r = irecip_pos(x); break;
    case 10: r = iscale(y.lo, x); break;
    // primitives of the dense fast path (ia_fast.cuh)
    case 11: r = prod_p(to_mr(x), y); break;                 // x >= 0 as (m, r), y any
    case 12: r = prod_u(to_mr(x), y); break;                 // x any class as (m, r), y any
    case 13: {                                               // x = D+ >= 0, y = u_d^2 in [1/4, 4]
      struct { T Dlo, Dhi, DloP, DhiP; } h = {x.lo, x.hi, Rnd<T>::fma_dn(-x.lo, Rnd<T>::pad_rel(), x.lo),
                                              Rnd<T>::fma_up(x.hi, Rnd<T>::pad_rel(), x.hi)};
      r = Dir<T>::d_over_sqrt(h, y);
      break;
    }
    case 14: r = sqr_u(x); break;
    case 15: { Iv<T> c; trig_small(x, r, c); break; }        // sin over x inside [-1/4, 1/4]
    case 16: { Iv<T> s; trig_small(x, s, r); break; }        // cos
    case 17: r = clamp_unit(x); break;
    case 18: { Iv<T> c; trig_medium(x, r, c); break; }       // sin over x inside (-1, 1) (double)
    case 19: { Iv<T> s; trig_medium(x, s, r); break; }       // cos
    default: break;
  }
  out[2 * i] = double(r.lo);
  out[2 * i + 1] = double(r.hi);
}

// ---- refinement ---------------------------------------------------------------------------------
// dense cell index -> box (S9): linear index ((((ix*ny+iy)*nR+iR)*nz+iz)*nl+il), lambda fastest
__global__ void gather_dense_kernel(GridDesc g, const int64_t* __restrict__ idx, const uint16_t* __restrict__ v,
                                    int k, int levels, ia_box* __restrict__ boxes) {
  pdl_wait();                 // programmatic dependent launch: nothing before the kernels in front have completed
  const int e = blockIdx.x, r = threadIdx.x;
  if (r >= k) return;
  int64_t c = idx[int64_t(e) * k + r];
  ia_box bx;
  for (int d = 4; d >= 0; --d) {
    const int kk = int(c % g.n[d]);
    c /= g.n[d];
    bx.lo[d] = cell_edge(g.lo[d], g.hi[d], g.w[d], kk, g.n[d]);
    bx.hi[d] = cell_edge(g.lo[d], g.hi[d], g.w[d], kk + 1, g.n[d]);
  }
  bx.votes = v[int64_t(e) * k + r];
  bx._pad[0] = bx._pad[1] = bx._pad[2] = 0;
  boxes[(int64_t(e) * levels + 0) * k + r] = bx;
}

// child c of a box: bit (4-d) of c set -> upper half [mid, hi], mid = 0.5*(lo+hi) rn (S9, G18)
__device__ __forceinline__ void child_axis(double lo, double hi, int upper, double& clo, double& chi) {
  const double mid = __dmul_rn(0.5, __dadd_rn(lo, hi));
  clo = upper ? mid : lo;
  chi = upper ? hi : mid;
}

// One refinement pass, stage 1: block (split, e, chunk) owns the children t = chunk*256 + thread of
// event e (rank t/32, child t%32); each thread computes its child from the parent on the fly and
// counts the votes of the hits [split*per_split, ...) - the hit range is split across blocks so
// that a single event still fills the chip; partial[e][split][t].
template <class T>
__global__ void __launch_bounds__(256)
vote_children_kernel(HitSpan sp, const HitC<T>* __restrict__ staged, const ia_box* __restrict__ boxes, int lev,
                     int levels, int k, int per_split, uint16_t* __restrict__ partial) {
  pdl_wait();                 // programmatic dependent launch: nothing before the kernels in front have completed
  extern __shared__ __align__(16) unsigned char smem_raw[];
  HitC<T>* sh = reinterpret_cast<HitC<T>*>(smem_raw);
  const int e = blockIdx.y, split = blockIdx.x;
  int first, count;
  event_hits(sp, e, first, count);
  const int h0 = split * per_split;
  int h1 = h0 + per_split;
  if (h1 > count) h1 = count;
  for (int i = h0 + threadIdx.x; i < h1; i += blockDim.x) sh[i - h0] = staged[int64_t(e) * sp.max_hits + i];
  __syncthreads();
  const int t = blockIdx.z * blockDim.x + threadIdx.x;
  if (t >= k * 32) return;
  const ia_box par = boxes[(int64_t(e) * levels + (lev - 1)) * k + (t >> 5)];
  const int c = t & 31;
  double lo[5], hi[5];
#pragma unroll
  for (int d = 0; d < 5; ++d) child_axis(par.lo[d], par.hi[d], (c >> (4 - d)) & 1, lo[d], hi[d]);
  const Iv<T> X = box_iv<T>(lo[0], hi[0]), Y = box_iv<T>(lo[1], hi[1]);
  Box3<T> bx = {box_iv<T>(lo[2], hi[2]), box_iv<T>(lo[3], hi[3]), box_iv<T>(lo[4], hi[4])};
  unsigned v = 0;
  for (int h = 0; h < h1 - h0; ++h) {
    const HitC<T> hc = sh[h];
    const XYInv<T> inv = xy_invariants(X, Y, hc);
    v += hit_votes_general(bx, inv, hit_small(hc), hc.zref) ? 1u : 0u;
  }
  partial[(int64_t(e) * gridDim.x + split) * (k * 32) + t] = uint16_t(v);
}

// stage 2: one block per event sums the partial counts, selects the top k of the 32k children
// (warp = one parent's 32 children: sort, then merge across warps) and writes their boxes.
__global__ void __launch_bounds__(1024)
select_children_kernel(const uint16_t* __restrict__ partial, int n_splits, int lev, int levels, int k,
                       ia_box* __restrict__ boxes) {
  pdl_wait();                 // programmatic dependent launch: nothing before the kernels in front have completed
  __shared__ u64 smem_keys[32 * 32];
  const int e = blockIdx.x, t = threadIdx.x, lane = t & 31, warp = t >> 5;
  unsigned v = 0;
  for (int s = 0; s < n_splits; ++s) v += partial[(int64_t(e) * n_splits + s) * (k * 32) + t];
  u64 mine = warp_sort_desc(make_key(v, t));
  mine = block_merge(mine, smem_keys);
  if (warp == 0 && lane < k) {
    const int child = int(key_index(mine));
    const ia_box par = boxes[(int64_t(e) * levels + (lev - 1)) * k + (child >> 5)];
    const int c = child & 31;
    ia_box bx;
#pragma unroll
    for (int d = 0; d < 5; ++d) child_axis(par.lo[d], par.hi[d], (c >> (4 - d)) & 1, bx.lo[d], bx.hi[d]);
    bx.votes = key_votes(mine);
    bx._pad[0] = bx._pad[1] = bx._pad[2] = 0;
    boxes[(int64_t(e) * levels + lev) * k + lane] = bx;
  }
}

// value = centre, error = half-width of the rank-0 box of the last pass (L94, G19); then the hull of the kept boxes of
// the last pass that share rank 0's vote count (G19: the paper keeps every cell at the maximum, L94)
__global__ void params_kernel(int n_events, int levels, int k, const ia_box* __restrict__ boxes,
                              double* __restrict__ params) {
  pdl_wait();                 // programmatic dependent launch: nothing before the kernels in front have completed
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n_events) return;
  const ia_box* last = boxes + (int64_t(e) * levels + (levels - 1)) * k;
  const ia_box b = last[0];
  double* out = params + int64_t(e) * IA_N_PARAMS;
  for (int d = 0; d < 5; ++d) {
    out[d] = __dmul_rn(0.5, __dadd_rn(b.lo[d], b.hi[d]));
    out[5 + d] = __dmul_rn(0.5, __dadd_rn(b.hi[d], -b.lo[d]));
    double hl = b.lo[d], hh = b.hi[d];
    for (int r = 1; r < k; ++r)
      if (last[r].votes == b.votes) { hl = fmin(hl, last[r].lo[d]); hh = fmax(hh, last[r].hi[d]); }
    out[10 + d] = hl;
    out[15 + d] = hh;
  }
}

template <class T> size_t staged_bytes(const HitSpan& sp) { return size_t(sp.n_events) * sp.max_hits * sizeof(HitC<T>); }

}  // namespace

#define IA_DISPATCH_PREC(ctx, CALL_D, CALL_F) \
  do {                                        \
    if ((ctx)->params.precision == 32) {      \
      CALL_F;                                 \
    } else {                                  \
      CALL_D;                                 \
    }                                         \
  } while (0)

cudaError_t launch_stage_hits(ia_ctx* ctx, const HitSpan& sp) {
  const bool f32 = ctx->params.precision == 32;
  cudaError_t err = scratch_reserve(ctx->staged, f32 ? staged_bytes<float>(sp) : staged_bytes<double>(sp));
  if (err != cudaSuccess) return err;
  if (sp.n_events <= 0 || sp.max_hits <= 0) return cudaSuccess;
  IA_DISPATCH_PREC(ctx,
    (err = launch_k(ctx, stage_hits_kernel<double>, dim3(sp.n_events), dim3(64), 0, sp, ctx->wires, ctx->n_wires, ctx->params,
                    static_cast<HitC<double>*>(ctx->staged.p), ctx->status)),
    (err = launch_k(ctx, stage_hits_kernel<float>, dim3(sp.n_events), dim3(64), 0, sp, ctx->wires, ctx->n_wires, ctx->params,
                    static_cast<HitC<float>*>(ctx->staged.p), ctx->status)));
  ctx->launches++;
  return err;
}

cudaError_t launch_vote_boxes(ia_ctx* ctx, const HitSpan& sp, const double* lo, const double* hi, int64_t n_boxes,
                              uint16_t* votes_out) {
  if (n_boxes <= 0) return cudaSuccess;
  const unsigned blocks = unsigned((n_boxes + 127) / 128);
  // up to IA_MAX_HITS staged hits (120 B each in double) exceed the 48 KB default of dynamic shared memory
  cudaError_t aerr = cudaSuccess;
  IA_DISPATCH_PREC(ctx,
    (aerr = cudaFuncSetAttribute(vote_boxes_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 int(sp.max_hits * sizeof(HitC<double>)))),
    (aerr = cudaFuncSetAttribute(vote_boxes_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 int(sp.max_hits * sizeof(HitC<float>)))));
  if (aerr != cudaSuccess) return aerr;
  IA_DISPATCH_PREC(ctx,
    (vote_boxes_kernel<double><<<blocks, 128, sp.max_hits * sizeof(HitC<double>), ctx->stream>>>(
        sp, static_cast<const HitC<double>*>(ctx->staged.p), lo, hi, n_boxes, votes_out)),
    (vote_boxes_kernel<float><<<blocks, 128, sp.max_hits * sizeof(HitC<float>), ctx->stream>>>(
        sp, static_cast<const HitC<float>*>(ctx->staged.p), lo, hi, n_boxes, votes_out)));
  ctx->launches++;
  return cudaGetLastError();
}

cudaError_t launch_residual(ia_ctx* ctx, const HitSpan& sp, const double* lo, const double* hi, int64_t n_boxes,
                            double* out) {
  const int64_t n = n_boxes * sp.n_hits_single;
  if (n <= 0) return cudaSuccess;
  const unsigned blocks = unsigned((n + 127) / 128);
  IA_DISPATCH_PREC(ctx,
    (residual_kernel<double><<<blocks, 128, 0, ctx->stream>>>(sp, static_cast<const HitC<double>*>(ctx->staged.p), lo, hi,
                                                              n_boxes, out)),
    (residual_kernel<float><<<blocks, 128, 0, ctx->stream>>>(sp, static_cast<const HitC<float>*>(ctx->staged.p), lo, hi,
                                                             n_boxes, out)));
  ctx->launches++;
  return cudaGetLastError();
}

cudaError_t launch_prim(ia_ctx* ctx, int op, int prec, const double* a, const double* b, int64_t n, double* out) {
  if (n <= 0) return cudaSuccess;
  const unsigned blocks = unsigned((n + 127) / 128);
  if (prec == 32) prim_kernel<float><<<blocks, 128, 0, ctx->stream>>>(op, a, b, n, out);
  else prim_kernel<double><<<blocks, 128, 0, ctx->stream>>>(op, a, b, n, out);
  ctx->launches++;
  return cudaGetLastError();
}

cudaError_t launch_gather_dense(ia_ctx* ctx, const GridDesc& g, const int64_t* idx, const uint16_t* v, int n_events,
                                int k, int levels, ia_box* boxes_out) {
  const cudaError_t err = launch_k(ctx, gather_dense_kernel, dim3(n_events), dim3(32), 0, g, idx, v, k, levels, boxes_out);
  ctx->launches++;
  return err;
}

cudaError_t launch_refine_level(ia_ctx* ctx, const HitSpan& sp, int lev, int levels, int k, ia_box* boxes_out) {
  int sm = 148;
  cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, ctx->device);
  const int threads = k * 32;
  int n_splits = 1;
  uint16_t* partial = nullptr;
  cudaError_t err;
  if (!(ctx->params.flags & IA_FLAG_GENERAL)) {
    // sign-specialised form, a4 shared by the children of an xy sub-cell (ia_vote_dense.cu); with IA_FLAG_RIGOROUS_PHI its
    // rigorous-Phi instantiation
    err = launch_vote_children_fast(ctx, sp, lev, levels, k, sm, boxes_out, &n_splits, &partial);
    if (err != cudaSuccess) return err;
  } else {
    // general form (IA_FLAG_GENERAL, alone or with the rigorous-Phi mode of IA_FLAG_RIGOROUS_PHI): split the hit range when there are too few events to fill the chip
    n_splits = (2 * sm + sp.n_events - 1) / sp.n_events;
    if (n_splits > sp.max_hits) n_splits = sp.max_hits;
    if (n_splits < 1) n_splits = 1;
    int per_split = (sp.max_hits + n_splits - 1) / n_splits;
    if (per_split < 1) per_split = 1;                   // no hits at all: one split that votes nothing
    n_splits = sp.max_hits > 0 ? (sp.max_hits + per_split - 1) / per_split : 1;
    err = scratch_reserve(ctx->partial, size_t(sp.n_events) * n_splits * k * 32 * sizeof(uint16_t));
    if (err != cudaSuccess) return err;
    partial = static_cast<uint16_t*>(ctx->partial.p);
    dim3 grid(n_splits, sp.n_events, (threads + 255) / 256);
    IA_DISPATCH_PREC(ctx,
      (err = cudaFuncSetAttribute(vote_children_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  int(per_split * sizeof(HitC<double>)))),
      (err = cudaFuncSetAttribute(vote_children_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                  int(per_split * sizeof(HitC<float>)))));
    if (err != cudaSuccess) return err;
    IA_DISPATCH_PREC(ctx,
      (err = launch_k(ctx, vote_children_kernel<double>, grid, dim3(256), per_split * sizeof(HitC<double>), sp,
                      static_cast<const HitC<double>*>(ctx->staged.p), boxes_out, lev, levels, k, per_split, partial)),
      (err = launch_k(ctx, vote_children_kernel<float>, grid, dim3(256), per_split * sizeof(HitC<float>), sp,
                      static_cast<const HitC<float>*>(ctx->staged.p), boxes_out, lev, levels, k, per_split, partial)));
    ctx->launches++;
    if (err != cudaSuccess) return err;
  }
  err = launch_k(ctx, select_children_kernel, dim3(sp.n_events), dim3(threads), 0, partial, n_splits, lev, levels, k, boxes_out);
  ctx->launches++;
  return err;
}

cudaError_t launch_params(ia_ctx* ctx, int n_events, int levels, int k, const ia_box* boxes, double* params_out) {
  const cudaError_t err = launch_k(ctx, params_kernel, dim3((n_events + 127) / 128), dim3(128), 0, n_events, levels, k, boxes, params_out);
  ctx->launches++;
  return err;
}

}  // namespace ia

// ---- FP64 pipe probe: what the chip sustains on independent double-precision chains ---------------
// mode 0: DFMA (round-to-nearest); mode 1: DADD.RM / DMUL.RP alternating (the interval mix);
// mode 2: DFMA.RM / DFMA.RP.  8 independent chains per thread, `iters` rounds of 8 instructions.
// modes 3, 4, 5: DFMA.RM / DFMA.RP on 1, 2, 4 chains per thread (same instruction count): how much
// instruction-level parallelism inside one warp the FP64 pipe needs.
namespace ia {
namespace {
template <int mode>
__global__ void __launch_bounds__(256) fp64_probe_kernel(int iters, double seed, double* __restrict__ sink) {
  double a[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) a[j] = seed + 1e-3 * (threadIdx.x + 8 * j);
  const double m = 1.0 - 1e-9, c = 1e-12;
  if (mode == 0) {
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int j = 0; j < 8; ++j) a[j] = __fma_rn(a[j], m, c);
    }
  } else if (mode == 1) {
    for (int i = 0; i < iters; i += 2) {
#pragma unroll
      for (int j = 0; j < 8; ++j) a[j] = __dadd_rd(a[j], c);
#pragma unroll
      for (int j = 0; j < 8; ++j) a[j] = __dmul_ru(a[j], m);
    }
  } else if (mode == 2) {
    for (int i = 0; i < iters; i += 2) {
#pragma unroll
      for (int j = 0; j < 8; ++j) a[j] = __fma_rd(a[j], m, c);
#pragma unroll
      for (int j = 0; j < 8; ++j) a[j] = __fma_ru(a[j], m, c);
    }
  } else if (mode == 6 || mode == 7) {
    // 8 DFMA.RM/RP chains with one independent non-FP64 instruction after every DFMA: mode 6 an integer
    // ALU-pipe operation (LOP3), mode 7 an FP32 FMA-pipe operation (FFMA).  Only the DFMAs are counted.
    unsigned u[8];
    float f[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) { u[j] = threadIdx.x * 2654435761u + j; f[j] = float(j) + 0.5f; }
    unsigned ku = unsigned(iters) | 0x10001u;
    float kf = 0.999f, kc = 1e-3f;
    asm volatile("" : "+r"(ku), "+f"(kf), "+f"(kc));     // in registers, not re-read from the constant bank
    for (int i = 0; i < iters; i += 2) {
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        a[j] = __fma_rd(a[j], m, c);
        if (mode == 6) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[j]) : "r"(ku), "r"(u[(j + 1) & 7]));
        else asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[j]) : "f"(kf), "f"(kc));
      }
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        a[j] = __fma_ru(a[j], m, c);
        if (mode == 6) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(u[j]) : "r"(ku), "r"(u[(j + 3) & 7]));
        else asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[j]) : "f"(kf), "f"(kc));
      }
    }
#pragma unroll
    for (int j = 0; j < 8; ++j) a[j] += double(u[j] & 1u) + double(f[j]) * 1e-30;
  } else if (mode == 10 || mode == 11) {
    // three register operands, one of them shared by consecutive instructions (the operand reuse cache):
    // mode 10 shares the multiplier among 4 consecutive DFMAs, mode 11 among 2
    double bb[8], cc[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) { bb[j] = 1.0 - 1e-9 * (threadIdx.x + j + 1); cc[j] = 1e-12 * (threadIdx.x + 3 * j + 1); }
    asm volatile("" : "+d"(bb[0]), "+d"(bb[1]), "+d"(bb[2]), "+d"(bb[3]), "+d"(bb[4]), "+d"(bb[5]), "+d"(bb[6]), "+d"(bb[7]));
    asm volatile("" : "+d"(cc[0]), "+d"(cc[1]), "+d"(cc[2]), "+d"(cc[3]), "+d"(cc[4]), "+d"(cc[5]), "+d"(cc[6]), "+d"(cc[7]));
    const int sh = mode == 10 ? 2 : 1;
    for (int i = 0; i < iters; i += 2) {
#pragma unroll
      for (int j = 0; j < 8; ++j) asm volatile("fma.rm.f64 %0, %1, %0, %2;" : "+d"(a[j]) : "d"(bb[j >> sh]), "d"(cc[j]));
#pragma unroll
      for (int j = 0; j < 8; ++j) asm volatile("fma.rp.f64 %0, %1, %0, %2;" : "+d"(a[j]) : "d"(bb[4 + (j >> sh)]), "d"(cc[(j + 1) & 7]));
    }
  } else if (mode == 8 || mode == 9) {
    // register operands: mode 8 DFMA.RM/RP with three distinct per-thread register operands (the probes above
    // multiply by and add uniform values), mode 9 DMUL.RM / DADD.RP with two - does operand fetch from the
    // register file hold the pipe below one instruction per two cycles?
    double bb[8], cc[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) { bb[j] = 1.0 - 1e-9 * (threadIdx.x + j + 1); cc[j] = 1e-12 * (threadIdx.x + 3 * j + 1); }
    asm volatile("" : "+d"(bb[0]), "+d"(bb[1]), "+d"(bb[2]), "+d"(bb[3]), "+d"(bb[4]), "+d"(bb[5]), "+d"(bb[6]), "+d"(bb[7]));
    asm volatile("" : "+d"(cc[0]), "+d"(cc[1]), "+d"(cc[2]), "+d"(cc[3]), "+d"(cc[4]), "+d"(cc[5]), "+d"(cc[6]), "+d"(cc[7]));
    for (int i = 0; i < iters; i += 2) {
      if (mode == 8) {
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = __fma_rd(a[j], bb[j], cc[(j + 1) & 7]);
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = __fma_ru(a[j], bb[(j + 3) & 7], cc[j]);
      } else {
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = __dmul_rd(a[j], bb[j]);
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = __dadd_ru(a[j], cc[j]);
      }
    }
  } else {
    // modes 3, 4, 5: the same number of DFMA.RM/RP per thread on 1, 2, 4 independent chains only
    const int nc = 1 << (mode - 3);
    for (int i = 0; i < iters; i += 2) {
      if (nc == 1) {
#pragma unroll
        for (int r = 0; r < 8; ++r) { a[0] = __fma_rd(a[0], m, c); a[0] = __fma_ru(a[0], m, c); }
      } else if (nc == 2) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
          a[0] = __fma_rd(a[0], m, c); a[1] = __fma_rd(a[1], m, c);
          a[0] = __fma_ru(a[0], m, c); a[1] = __fma_ru(a[1], m, c);
        }
      } else {
#pragma unroll
        for (int r = 0; r < 2; ++r) {
#pragma unroll
          for (int j = 0; j < 4; ++j) a[j] = __fma_rd(a[j], m, c);
#pragma unroll
          for (int j = 0; j < 4; ++j) a[j] = __fma_ru(a[j], m, c);
        }
      }
    }
  }
  double s = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) s += a[j];
  if (s == 12345.678) sink[0] = s;   // never true: keeps the chains alive
}
}  // namespace

cudaError_t launch_fp64_probe(ia_ctx* ctx, int mode, int iters, int blocks, double* sink) {
  switch (mode) {
#define IA_PROBE_CASE(M) case M: fp64_probe_kernel<M><<<blocks, 256, 0, ctx->stream>>>(iters, 1.0, sink); break;
    IA_PROBE_CASE(0) IA_PROBE_CASE(1) IA_PROBE_CASE(2) IA_PROBE_CASE(3) IA_PROBE_CASE(4) IA_PROBE_CASE(5)
    IA_PROBE_CASE(6) IA_PROBE_CASE(7) IA_PROBE_CASE(8) IA_PROBE_CASE(9) IA_PROBE_CASE(10) IA_PROBE_CASE(11)
#undef IA_PROBE_CASE
    default: return cudaErrorInvalidValue;
  }
  ctx->launches++;
  return cudaGetLastError();
}
}  // namespace ia
