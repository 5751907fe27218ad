// ia_vote_paper.cu - the paper's own vote configuration.
//
//   M1  voxel = 4-D interval xc x yc x R x z0 (L64); mid-point m = 0.5*(lo+hi) per axis.
//   M2  momentum fixed to its true value (L64), given as P = R sqrt(1 + lambda^2): |lambda| =
//       sqrt((P/R_m)^2 - 1); two accumulators for the two signs of lambda (L78); R_m > P: no vote.
//   M3  d_Ax of (A.5b) is a NUMBER: steps S2-S8 at the voxel's mid-point in round-to-nearest double
//       arithmetic (L82: "Their values are taken in the middle of the voxel").  Negative radicand or
//       NaN: that drift sign does not vote.
//   M4  tolerance: hull of d_Ax at d - tol (clamped at 0) and d + tol; tol = 0 is the paper's form.
//   M5  condition (4) L74-76 in interval arithmetic: 0 in (x_Ax-xc)^2 + (y_Ax-yc)^2 - (R + d_Ax)^2,
//       either drift sign, one count per hit.
// The point arithmetic keeps the association order of the interval form and is
// never contracted into FMAs (explicit __dmul_rn/__dadd_rn), so it differs from a plain host evaluation
// only through sin, cos and atan2.
//
// Block = one (xc, yc) cell: its threads compute once per hit what depends on (xc_m, yc_m, hit) only
// (the point values of S2, S3, S3' and the interval (x_Ax-xc)^2 + (y_Ax-yc)^2) into shared memory, then
// every thread walks (R, z0) voxels of the column, keeps the two vote counts in registers and stores
// two uint16 per voxel.  No atomics.
#include "ia_internal.h"
#include "ia_fast.cuh"

namespace ia {
namespace {

struct PHit {
  double Qlo, Qhi;                            // interval (x_Ax - X)^2 + (y_Ax - Y)^2
  double cA, sA, dphi, iQ, RA, iR, c2, s2;    // point values at (xc_m, yc_m)
  double Tn, T2, twoT, dlo, dhi, zref;
  int valid, _pad;
};

IA_DEV double mul(double a, double b) { return __dmul_rn(a, b); }
IA_DEV double add(double a, double b) { return __dadd_rn(a, b); }
IA_DEV double sub(double a, double b) { return __dadd_rn(a, -b); }

// per-hit scalars (round to nearest, unfused: the same operations as stage_hits_kernel) and the
// (xc_m, yc_m)-dependent point values of S2, S3, S3'
// (xr, yr): the reference point of this pass - ia_params' or, inside ia_track_paper, the one of reading F2d'
__device__ void make_phit(const double* __restrict__ wires, int n_wires, ia_hit h, const ia_params& p, double xr, double yr,
                          Iv<double> X, Iv<double> Y, int* status, PHit& o) {
  int w = h.wire;
  o.valid = (w >= 0 && w < n_wires && h.drift >= 0.0);
  if (!o.valid) {
    if (status) atomicOr(status, 1);
    w = 0;
    h.drift = 0.0;
  }
  const double x0 = wires[w], y0 = wires[n_wires + w], s = wires[2 * n_wires + w], co = wires[3 * n_wires + w];
  const double t = wires[4 * n_wires + w];
  const double zr = p.z_ref;
  const double xA = add(x0, mul(mul(zr, s), t));                       // (A.4d)
  const double yA = sub(y0, mul(mul(zr, co), t));                      // (A.4e)
  const double k0 = sub(mul(xr, yA), mul(yr, xA)), ky = sub(yr, yA), kx = sub(xA, xr);
  const double mx_ = mul(0.5, add(xr, xA)), my_ = mul(0.5, add(yr, yA));
  const double hx = mul(0.5, sub(xA, xr)), hy = mul(0.5, sub(yA, yr));
  const double h2 = add(mul(hx, hx), mul(hy, hy));
  o.Tn = t; o.T2 = mul(t, t); o.twoT = mul(2.0, t); o.zref = zr;
  o.dlo = fmax(sub(h.drift, p.tol), 0.0);                              // M4
  o.dhi = add(h.drift, p.tol);
  // M5, xy part: every variable occurs once
  const Iv<double> Q = iadd(isqr(isub(thin(xA), X)), isqr(isub(thin(yA), Y)));
  o.Qlo = Q.lo; o.Qhi = Q.hi;
  // S2, S3, S3' at the mid-point
  const double xc = mul(0.5, add(X.lo, X.hi)), yc = mul(0.5, add(Y.lo, Y.hi));
  const double A = sub(xA, xc), B = sub(yA, yc);
  const double Qp = add(mul(A, A), mul(B, B));
  o.cA = sub(mul(A, s), mul(B, co));
  o.sA = add(mul(A, co), mul(B, s));
  const double cr = add(add(k0, mul(ky, xc)), mul(kx, yc));
  const double dx = sub(xc, mx_), dy = sub(yc, my_);
  const double dt = sub(add(mul(dx, dx), mul(dy, dy)), h2);
  double dphi = atan2(cr, dt);
  // reading M6 (IA_FLAG_FULL_TURN): a counter-clockwise track of less than one turn emitted near the z axis has turned by
  // theta in [-m, 2 pi - m), m = 0.3 rad, past the point of its base circle closest to the axis when it reaches a point
  // P of the circle; phi_Ax - phi0 of (A.8d) = theta(wire point) - theta(reference point), right wherever the
  // reference point lies along the track (it moves between passes, L98).  theta(P) = the S3 angle with the reference
  // at the axis and the wire point at P; same operations, same order as the oracle's.
  if (p.flags & IA_FLAG_FULL_TURN) {
    auto theta = [&](double px, double py) {
      const double hx_ = mul(0.5, px), hy_ = mul(0.5, py);
      const double cr0 = add(mul(sub(0.0, py), xc), mul(px, yc));
      const double ex = sub(xc, hx_), ey = sub(yc, hy_);
      const double dt0 = sub(add(mul(ex, ex), mul(ey, ey)), add(mul(hx_, hx_), mul(hy_, hy_)));
      double th = atan2(cr0, dt0);
      if (th < -0.3) th = add(th, 6.283185307179586);
      return th;
    };
    dphi = sub(theta(xA, yA), theta(xr, yr));
  }
  o.dphi = dphi;
  o.iQ = __ddiv_rn(1.0, Qp);
  o.RA = __dsqrt_rn(Qp);
  o.iR = __ddiv_rn(1.0, o.RA);
  o.c2 = mul(sub(mul(o.cA, o.cA), mul(o.sA, o.sA)), o.iQ);
  o.s2 = mul(mul(2.0, mul(o.sA, o.cA)), o.iQ);
}

// sin and cos of e = Phi - Phi_Ax: Taylor forms of ia_fast.cuh inside [-1/4, 1/4] (error below 1 ulp),
// the library functions outside
IA_DEV void sincos_e(double e, double& se, double& ce) {
  if (fabs(e) < 0.25) {
    const double s = mul(e, e);
    se = Trig<double>::sin_small(e, s);
    ce = Trig<double>::cos_small(s);
  } else {
    se = sin(e);
    ce = cos(e);
  }
}

// S4-S8 at a point; D is the signed drift distance.  false: no d_Ax (M3)
IA_DEV bool dax_point(const PHit& h, double R, double Zr, double lam, double D, double& dax) {
  const double LR = mul(lam, R);
  const double zA = add(Zr, mul(LR, h.dphi));
  const double LD = mul(lam, D);
  const double P1 = -mul(add(mul(zA, h.sA), mul(LD, h.cA)), h.iQ);
  const double t1 = mul(LR, zA);
  const double t2 = mul(mul(mul(lam, zA), sub(R, mul(2.0, D))), h.c2);
  const double t3 = mul(add(mul(zA, zA), mul(D, add(h.RA, mul(mul(lam, lam), sub(add(R, h.RA), D))))), h.s2);
  const double P2 = mul(0.5, mul(add(sub(t1, t2), t3), h.iQ));
  const double e = add(mul(h.Tn, P1), mul(h.T2, P2));
  double se, ce;
  sincos_e(e, se, ce);
  double sinP = mul(add(mul(h.sA, ce), mul(h.cA, se)), h.iR);
  double cosP = mul(sub(mul(h.cA, ce), mul(h.sA, se)), h.iR);
  sinP = fmin(1.0, fmax(-1.0, sinP));
  cosP = fmin(1.0, fmax(-1.0, cosP));
  const double u2 = add(add(add(1.0, mul(h.twoT, mul(lam, sinP))), mul(h.T2, mul(lam, lam))), mul(h.T2, mul(cosP, cosP)));
  const double u = __dsqrt_rn(u2);
  const double dl = __ddiv_rn(D, u);
  const double z = sub(add(Zr, mul(LR, add(h.dphi, e))), mul(h.Tn, mul(dl, cosP)));
  const double Ld = mul(lam, dl);
  const double ct = sub(mul(z, h.cA), mul(Ld, h.sA));
  const double Rd = add(R, dl), Tz = mul(h.Tn, z), TLd = mul(h.Tn, Ld);
  const double rad = sub(sub(sub(mul(Rd, Rd), mul(h.twoT, ct)), mul(Tz, Tz)), mul(TLd, TLd));
  if (!(rad >= 0.0)) return false;
  dax = sub(__dsqrt_rn(rad), R);
  return true;
}

constexpr int PAPER_THREADS = 256;

// a fixed grid, or (centre != nullptr) a window of half-widths `half` around a fit that lives on the device:
// lo = value - half, hi = value + half, w = (hi - lo)/n - the operations of make_grid, done by every kernel
// that needs the grid, so that a pass can be enqueued before the previous one has produced its centre
IA_DEV GridDesc resolve_grid(const PaperGrid& pg) {
  GridDesc g = pg.g;
  if (pg.centre) {
#pragma unroll
    for (int d = 0; d < 4; ++d) {
      const double c = (d == 3 && pg.self) ? pg.self->z0_centre : pg.centre->value[d];
      g.lo[d] = sub(c, pg.half[d]);
      g.hi[d] = add(c, pg.half[d]);
      g.w[d] = __ddiv_rn(sub(g.hi[d], g.lo[d]), double(g.n[d]));
    }
  }
  return g;
}

// M3-M5 for one (voxel, hit, lambda): does either drift sign contain 0 ?
IA_DEV bool paper_hit_votes(const PHit& ph, Iv<double> R, double Rm, double Zr, double l, bool two_ends) {
  bool yes = false;
#pragma unroll
  for (int ds = 0; ds < 2; ++ds) {
    double a = 0.0, b;
    bool ok = dax_point(ph, Rm, Zr, l, ds == 0 ? ph.dlo : -ph.dlo, a);
    b = a;
    if (two_ends) ok = dax_point(ph, Rm, Zr, l, ds == 0 ? ph.dhi : -ph.dhi, b) && ok;
    const Iv<double> Dax = {fmin(a, b), fmax(a, b)};
    const Iv<double> S = isqr(iadd(R, Dax));
    const Iv<double> f = isub(Iv<double>{ph.Qlo, ph.Qhi}, S);
    yes = yes || (ok && !(f.lo > 0.0 || f.hi < 0.0));
  }
  return yes;
}

// M2: |lambda| at the mid radius from the fixed momentum; false if R_m > P
IA_DEV bool paper_lambda(double P, double Rm, double& lam) {
  const double q = __ddiv_rn(P, Rm);
  const double l2 = sub(mul(q, q), 1.0);
  lam = l2 >= 0.0 ? __dsqrt_rn(l2) : 0.0;
  return l2 >= 0.0;
}

// F2a, conditions (3a,b) L66-70: 0 in X^2 + Y^2 - (R + [-r_disk, r_disk])^2
IA_DEV bool disk_passes(Iv<double> X, Iv<double> Y, Iv<double> R, double r_disk) {
  const Iv<double> f = isub(iadd(isqr(X), isqr(Y)), isqr(iadd(R, Iv<double>{-r_disk, r_disk})));
  return !(f.lo > 0.0 || f.hi < 0.0);
}

__global__ void __launch_bounds__(PAPER_THREADS)
vote_paper_kernel(const ia_hit* __restrict__ hits, int n_hits, const uint8_t* __restrict__ hit_mask,
                  const double* __restrict__ wires, int n_wires, ia_params p, const ia_paper_fit* __restrict__ ref, double P,
                  double r_disk, PaperGrid pg, int signs, int* status, uint16_t* __restrict__ votes) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  PHit* sh = reinterpret_cast<PHit*>(smem_raw);
  const GridDesc g = resolve_grid(pg);
  const int ixy = blockIdx.x;
  const int ix = ixy / g.n[1], iy = ixy - ix * g.n[1];
  const Iv<double> X = {cell_edge(g.lo[0], g.hi[0], g.w[0], ix, g.n[0]), cell_edge(g.lo[0], g.hi[0], g.w[0], ix + 1, g.n[0])};
  const Iv<double> Y = {cell_edge(g.lo[1], g.hi[1], g.w[1], iy, g.n[1]), cell_edge(g.lo[1], g.hi[1], g.w[1], iy + 1, g.n[1])};
  // ref != nullptr: the reference point of this pass sits on the device (written by paper_ref_kernel just before)
  const double xr = ref ? ref->x_ref : p.x_ref, yr = ref ? ref->y_ref : p.y_ref;
  for (int h = threadIdx.x; h < n_hits; h += blockDim.x) {
    make_phit(wires, n_wires, hits[h], p, xr, yr, X, Y, status, sh[h]);
    if (hit_mask && !hit_mask[h]) sh[h].valid = 0;       // L96: only the selected hits are used
  }
  __syncthreads();
  const int nR = g.n[2], nz = g.n[3];
  const int64_t n_cells = g.cells;                       // nx*ny*nR*nz
  const bool two_ends = p.tol > 0.0;
  for (int j = threadIdx.x; j < nR * nz; j += blockDim.x) {
    const int iR = j / nz, iz = j - iR * nz;
    const Iv<double> R = {cell_edge(g.lo[2], g.hi[2], g.w[2], iR, nR), cell_edge(g.lo[2], g.hi[2], g.w[2], iR + 1, nR)};
    const double zlo = cell_edge(g.lo[3], g.hi[3], g.w[3], iz, nz), zhi = cell_edge(g.lo[3], g.hi[3], g.w[3], iz + 1, nz);
    const double Rm = mul(0.5, add(R.lo, R.hi)), zm = mul(0.5, add(zlo, zhi));
    double lam;
    bool live = paper_lambda(P, Rm, lam);
    if (live && r_disk >= 0.0) live = disk_passes(X, Y, R, r_disk);
    unsigned v[2] = {0u, 0u};
    if (live) {
      for (int h = 0; h < n_hits; ++h) {
        const PHit& ph = sh[h];
        if (!ph.valid) continue;
        const double Zr = sub(zm, ph.zref);
        // signs: bit 0 = the lambda >= 0 accumulator is wanted, bit 1 = the lambda < 0 one (a chain of
        // ia_track_paper needs one; the other is written as 0)
        if (signs & 1) v[0] += paper_hit_votes(ph, R, Rm, Zr, lam, two_ends) ? 1u : 0u;
        if (signs & 2) v[1] += paper_hit_votes(ph, R, Rm, Zr, -lam, two_ends) ? 1u : 0u;
      }
    }
    const int64_t cell = int64_t(ixy) * (nR * nz) + j;
    votes[cell] = uint16_t(v[0]);
    votes[n_cells + cell] = uint16_t(v[1]);
  }
}

// ---- F2b: selection of the maximum-vote voxels (L94, L121) -------------------------------------------
// Integer reductions only (atomicMax / atomicMin / atomicAdd on integers), so the result does not depend on
// the order in which blocks run.  acc: [0..1] vmax per accumulator, then for the chosen accumulator
// [2] count, [3..6] sum of cell indices per axis, [7..10] kmin, [11..14] kmax  (all unsigned long long)
__global__ void paper_init_kernel(unsigned long long* __restrict__ acc) {
  if (threadIdx.x < 16) acc[threadIdx.x] = (threadIdx.x >= 7 && threadIdx.x <= 10) ? ~0ull : 0ull;
}

__global__ void paper_max_kernel(const uint16_t* __restrict__ votes, int64_t n, unsigned long long* __restrict__ acc) {
  unsigned m0 = 0, m1 = 0;
  for (int64_t i = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; i < n; i += int64_t(gridDim.x) * blockDim.x) {
    m0 = max(m0, unsigned(votes[i]));
    m1 = max(m1, unsigned(votes[n + i]));
  }
  m0 = __reduce_max_sync(0xffffffffu, m0);
  m1 = __reduce_max_sync(0xffffffffu, m1);
  if ((threadIdx.x & 31) == 0) {
    atomicMax(&acc[0], (unsigned long long)m0);
    atomicMax(&acc[1], (unsigned long long)m1);
  }
}

// which: 0 = the accumulator with the larger maximum (equal maxima: lambda >= 0 wins), +1 / -1 = that accumulator
IA_DEV int pick_acc(const unsigned long long* acc, int which) { return which > 0 ? 0 : (which < 0 ? 1 : (acc[1] > acc[0] ? 1 : 0)); }

__global__ void paper_moments_kernel(const uint16_t* __restrict__ votes, int64_t n, GridDesc g, int which,
                                     unsigned long long* __restrict__ acc) {
  const int s = pick_acc(acc, which);
  const unsigned vmax = unsigned(acc[s]);
  const uint16_t* v = votes + int64_t(s) * n;
  // per-thread, then per-warp partial results; 13 atomics per warp at the end (a plateau can hold every voxel)
  unsigned long long cnt = 0, sum[4] = {0, 0, 0, 0};
  unsigned kmin[4] = {~0u, ~0u, ~0u, ~0u}, kmax[4] = {0, 0, 0, 0};
  for (int64_t i = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; i < n; i += int64_t(gridDim.x) * blockDim.x) {
    if (unsigned(v[i]) != vmax) continue;
    int64_t idx = i;
    ++cnt;
#pragma unroll
    for (int d = 3; d >= 0; --d) {
      const unsigned k = unsigned(idx % g.n[d]);
      idx /= g.n[d];
      sum[d] += k;
      kmin[d] = min(kmin[d], k);
      kmax[d] = max(kmax[d], k);
    }
  }
  const bool lead = (threadIdx.x & 31) == 0;
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    cnt += __shfl_down_sync(0xffffffffu, cnt, off);
#pragma unroll
    for (int d = 0; d < 4; ++d) sum[d] += __shfl_down_sync(0xffffffffu, sum[d], off);
  }
#pragma unroll
  for (int d = 0; d < 4; ++d) {
    kmin[d] = __reduce_min_sync(0xffffffffu, kmin[d]);
    kmax[d] = __reduce_max_sync(0xffffffffu, kmax[d]);
  }
  if (lead && cnt != 0) {
    atomicAdd(&acc[2], cnt);
#pragma unroll
    for (int d = 0; d < 4; ++d) {
      atomicAdd(&acc[3 + d], sum[d]);
      atomicMin(&acc[7 + d], (unsigned long long)kmin[d]);
      atomicMax(&acc[11 + d], (unsigned long long)kmax[d]);
    }
  }
}

__global__ void paper_fit_kernel(const unsigned long long* __restrict__ acc, PaperGrid pg, double P, int which,
                                 int keep_ref, double x_ref, double y_ref, ia_paper_fit* __restrict__ out) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const GridDesc g = resolve_grid(pg);
  const int s = pick_acc(acc, which);
  const unsigned long long cnt = acc[2];
  ia_paper_fit f;
  for (int d = 0; d < 4; ++d) {
    const double m = __ddiv_rn(double(2 * acc[3 + d] + cnt), double(2 * cnt));
    f.value[d] = add(g.lo[d], mul(m, g.w[d]));
    f.error[d] = mul(0.5, mul(double(acc[11 + d] - acc[7 + d] + 1), g.w[d]));
  }
  double lam;
  const bool has = paper_lambda(P, f.value[2], lam);
  f.lambda = has ? (s == 0 ? lam : -lam) : 0.0;
  f.lambda_sign = s == 0 ? 1 : -1;
  f.vmax = int32_t(acc[s]);
  f.n_sel = int64_t(cnt);
  // the reference point of the pass: written into the slot before the vote (ia_track_paper) or the caller's (ia_params)
  f.x_ref = keep_ref ? out->x_ref : x_ref;
  f.y_ref = keep_ref ? out->y_ref : y_ref;
  f.z0_centre = keep_ref ? out->z0_centre : 0.0;
  *out = f;
}

// ---- F2c: hit finding (L96): condition (4) on the interval value -/+ factor * error, per hit ---------------
__global__ void find_hits_paper_kernel(const ia_hit* __restrict__ hits, int n_hits, const double* __restrict__ wires, int n_wires,
                                       ia_params p, double P, const ia_paper_fit* __restrict__ fit, double factor, int* status,
                                       uint8_t* __restrict__ flags) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= n_hits) return;
  double lo[4], hi[4];
  for (int d = 0; d < 4; ++d) {
    const double e = mul(factor, fit->error[d]);
    lo[d] = sub(fit->value[d], e);
    hi[d] = add(fit->value[d], e);
  }
  PHit ph;
  make_phit(wires, n_wires, hits[h], p, fit->x_ref, fit->y_ref, Iv<double>{lo[0], hi[0]}, Iv<double>{lo[1], hi[1]}, status, ph);
  const Iv<double> R = {lo[2], hi[2]};
  const double Rm = mul(0.5, add(lo[2], hi[2])), zm = mul(0.5, add(lo[3], hi[3]));
  double lam;
  bool yes = false;
  if (ph.valid && paper_lambda(P, Rm, lam))
    yes = paper_hit_votes(ph, R, Rm, sub(zm, ph.zref), fit->lambda_sign >= 0 ? lam : -lam, p.tol > 0.0);
  flags[h] = yes ? 1 : 0;
}

}  // namespace

cudaError_t launch_vote_paper(ia_ctx* ctx, const ia_hit* hits, int n_hits, const uint8_t* hit_mask, double P, double r_disk,
                              const PaperGrid& pg, int signs, const ia_paper_fit* ref, uint16_t* votes_out) {
  const GridDesc& g = pg.g;
  const size_t smem = size_t(n_hits) * sizeof(PHit);
  cudaError_t err = cudaFuncSetAttribute(vote_paper_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem));
  if (err != cudaSuccess) return err;
  const int col = g.n[2] * g.n[3];
  int threads = PAPER_THREADS;
  if (col < threads) threads = (col + 31) / 32 * 32;
  vote_paper_kernel<<<unsigned(g.n[0] * g.n[1]), threads, smem, ctx->stream>>>(hits, n_hits, hit_mask, ctx->wires, ctx->n_wires,
                                                                              ctx->params, ref, P, r_disk, pg, signs, ctx->status,
                                                                              votes_out);
  ctx->launches++;
  return cudaGetLastError();
}

cudaError_t launch_select_max_paper(ia_ctx* ctx, const uint16_t* votes, const PaperGrid& pg, double P, int which,
                                    int keep_ref, ia_paper_fit* fit_out) {
  cudaError_t err = scratch_reserve(ctx->keys, 16 * sizeof(unsigned long long));
  if (err != cudaSuccess) return err;
  unsigned long long* acc = static_cast<unsigned long long*>(ctx->keys.p);
  paper_init_kernel<<<1, 32, 0, ctx->stream>>>(acc);
  const int64_t n = pg.g.cells;
  int blocks = int((n + 1023) / 1024);
  if (blocks > 1184) blocks = 1184;
  paper_max_kernel<<<blocks, 256, 0, ctx->stream>>>(votes, n, acc);
  paper_moments_kernel<<<blocks, 256, 0, ctx->stream>>>(votes, n, pg.g, which, acc);   // cell indices only: dims suffice
  paper_fit_kernel<<<1, 32, 0, ctx->stream>>>(acc, pg, P, which, keep_ref, ctx->params.x_ref, ctx->params.y_ref, fit_out);
  ctx->launches += 4;
  return cudaGetLastError();
}

cudaError_t launch_find_hits_paper(ia_ctx* ctx, const ia_hit* hits, int n_hits, double P, const ia_paper_fit* fit, double factor,
                                   uint8_t* flags_out) {
  if (n_hits <= 0) return cudaSuccess;
  find_hits_paper_kernel<<<(n_hits + 63) / 64, 64, 0, ctx->stream>>>(hits, n_hits, ctx->wires, ctx->n_wires, ctx->params, P, fit,
                                                                    factor, ctx->status, flags_out);
  ctx->launches++;
  return cudaGetLastError();
}

namespace {
// F2d' (L98): the reference point of the next pass = the z_ref-plane point (A.4d,e) of the wire of the selected hit
// (mask != 0) closest to the circle of the previous pass's fit; ties: lowest hit index; none selected: it stays.
// mode 0: copy the reference point of `prev` (or of ia_params when prev == nullptr) into next; 1: move it.
__global__ void paper_ref_kernel(const ia_hit* __restrict__ hits, int n_hits, const uint8_t* __restrict__ mask,
                                 const double* __restrict__ wires, int n_wires, ia_params p, const ia_paper_fit* __restrict__ prev,
                                 int mode, ia_paper_fit* __restrict__ next) {
  const double x_old = prev ? prev->x_ref : p.x_ref, y_old = prev ? prev->y_ref : p.y_ref;
  if (mode == 0) {
    if (threadIdx.x == 0) { next->x_ref = x_old; next->y_ref = y_old; next->z0_centre = prev ? prev->value[3] : 0.0; }
    return;
  }
  // one warp: every lane keeps the best of its hits (strict <, so the lowest index of equal distances), then a
  // shuffle reduction on (distance, index).  Distances are non-negative doubles: their bit patterns order like the values.
  unsigned long long bd = ~0ull;
  int bh = 0x7fffffff;
  double bx = x_old, by = y_old;
  for (int h = threadIdx.x; h < n_hits; h += 32) {
    if (mask && !mask[h]) continue;
    const int w = hits[h].wire;
    if (w < 0 || w >= n_wires) continue;
    const double x0 = wires[w], y0 = wires[n_wires + w], s = wires[2 * n_wires + w], co = wires[3 * n_wires + w], t = wires[4 * n_wires + w];
    const double xA = add(x0, mul(mul(p.z_ref, s), t)), yA = sub(y0, mul(mul(p.z_ref, co), t));       // (A.4d,e)
    const double dx = sub(xA, prev->value[0]), dy = sub(yA, prev->value[1]);
    const double d = fabs(sub(__dsqrt_rn(add(mul(dx, dx), mul(dy, dy))), prev->value[2]));
    const unsigned long long db = (unsigned long long)__double_as_longlong(d);
    if (db < bd) { bd = db; bh = h; bx = xA; by = yA; }
  }
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) {
    const unsigned long long od = __shfl_down_sync(0xffffffffu, bd, off);
    const int oh = __shfl_down_sync(0xffffffffu, bh, off);
    const double ox = __shfl_down_sync(0xffffffffu, bx, off), oy = __shfl_down_sync(0xffffffffu, by, off);
    if (od < bd || (od == bd && oh < bh)) { bd = od; bh = oh; bx = ox; by = oy; }
  }
  if (threadIdx.x == 0) {
    next->x_ref = bx;
    next->y_ref = by;
    // the previous z0 seen from the new point: z0 + (lambda R) (theta(new) - theta(old)), angles as in make_phit
    double z0c = prev->value[3];
    if (!(bx == x_old && by == y_old)) {
      const double xc = prev->value[0], yc = prev->value[1], two_pi = 6.283185307179586;
      double dth;
      if (p.flags & IA_FLAG_FULL_TURN) {
        auto theta = [&](double px, double py) {
          const double hx_ = mul(0.5, px), hy_ = mul(0.5, py);
          const double cr0 = add(mul(sub(0.0, py), xc), mul(px, yc));
          const double ex = sub(xc, hx_), ey = sub(yc, hy_);
          const double dt0 = sub(add(mul(ex, ex), mul(ey, ey)), add(mul(hx_, hx_), mul(hy_, hy_)));
          double th = atan2(cr0, dt0);
          if (th < -0.3) th = add(th, two_pi);
          return th;
        };
        dth = sub(theta(bx, by), theta(x_old, y_old));
      } else {
        dth = sub(atan2(sub(bx, xc), sub(yc, by)), atan2(sub(x_old, xc), sub(yc, y_old)));
        if (dth > 3.141592653589793) dth = sub(dth, two_pi);
        if (dth <= -3.141592653589793) dth = add(dth, two_pi);
      }
      z0c = add(prev->value[3], mul(mul(prev->lambda, prev->value[2]), dth));
    }
    next->z0_centre = z0c;
  }
}

__global__ void paper_sign_kernel(const ia_paper_fit* __restrict__ last, int32_t* __restrict__ sign_out) {
  if (threadIdx.x == 0) *sign_out = last[1].vmax > last[0].vmax ? -1 : 1;      // L121; ties: lambda >= 0
}
}  // namespace

cudaError_t launch_paper_ref(ia_ctx* ctx, const ia_hit* hits, int n_hits, const uint8_t* mask, const ia_paper_fit* prev, int move,
                             ia_paper_fit* next) {
  paper_ref_kernel<<<1, 32, 0, ctx->stream>>>(hits, n_hits, mask, ctx->wires, ctx->n_wires, ctx->params, prev, move, next);
  ctx->launches++;
  return cudaGetLastError();
}

cudaError_t launch_paper_sign(ia_ctx* ctx, const ia_paper_fit* last, int32_t* sign_out) {
  paper_sign_kernel<<<1, 32, 0, ctx->stream>>>(last, sign_out);
  ctx->launches++;
  return cudaGetLastError();
}

}  // namespace ia
