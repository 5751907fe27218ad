// ia_vote_dense.cu - steps a3-a6: the dense-grid vote kernel (layer B1, the hot loop).
//
// Condition (4): hit i votes for the cell iff 0 is in the interval extension of
// eq. (2) for either drift sign; votes[cell] = number of such hits.  A block owns one (xc, yc) cell
// of one event and a slice of that cell's (R, z0, lambda) column.  Its threads first compute, once
// per hit, everything of the residual that depends on (xc, yc, hit) only (a4: S2, S3, S3' of
// the atan2, the square root and the two divisions) into shared memory; every thread
// then walks its cells, reads the hits by shared-memory broadcast, keeps its vote count in a
// register and writes one uint16 per cell.  No atomics, no inter-thread traffic in the loop.
#include <algorithm>
#include <cmath>

#include "ia_internal.h"
#include "ia_fastq.cuh"

namespace ia {

namespace {

constexpr int GEN_THREADS = 128;
constexpr int GEN_CELLS_PER_THREAD = 8;

template <class T> struct HitShared {
  XYInv<T> inv;
  HitS<T> hs;
};

// general form: no assumption on signs; serves any grid
template <class T>
__global__ void __launch_bounds__(GEN_THREADS)
vote_dense_general_kernel(HitSpan sp, const HitC<T>* __restrict__ staged, GridDesc g, int chunks_per_col,
                          uint16_t* __restrict__ votes) {
  pdl_wait();                 // programmatic dependent launch: nothing before the kernels in front have completed
  extern __shared__ __align__(16) unsigned char smem_raw[];
  HitShared<T>* sh = reinterpret_cast<HitShared<T>*>(smem_raw);
  const int e = blockIdx.y;
  const int64_t bid = blockIdx.x;
  const int64_t ixy = bid / chunks_per_col;
  const int chunk = int(bid - ixy * chunks_per_col);
  const int ixl = int(ixy / g.n[1]), iy = int(ixy - int64_t(ixl) * g.n[1]);
  const int ix = g.ix0 + ixl;                                   // ixy counts inside the slab, ix in the full grid
  int count;
  if (sp.offsets) {
    count = sp.offsets[e + 1] - sp.offsets[e];
    if (count > sp.max_hits) count = sp.max_hits;
    if (count < 0) count = 0;
  } else {
    count = sp.n_hits_single;
  }
  const Iv<T> X = box_iv<T>(cell_edge(g.lo[0], g.hi[0], g.w[0], ix, g.n[0]), cell_edge(g.lo[0], g.hi[0], g.w[0], ix + 1, g.n[0]));
  const Iv<T> Y = box_iv<T>(cell_edge(g.lo[1], g.hi[1], g.w[1], iy, g.n[1]), cell_edge(g.lo[1], g.hi[1], g.w[1], iy + 1, g.n[1]));
  T zref = T(0);
  for (int h = threadIdx.x; h < count; h += blockDim.x) {
    const HitC<T> c = staged[int64_t(e) * sp.max_hits + h];
    sh[h].inv = xy_invariants(X, Y, c);
    sh[h].hs = hit_small(c);
  }
  if (count > 0) zref = staged[int64_t(e) * sp.max_hits].zref;
  __syncthreads();
  const int64_t col0 = int64_t(chunk) * (GEN_THREADS * GEN_CELLS_PER_THREAD);
  uint16_t* out = votes + int64_t(e) * g.cells + ixy * g.col_cells;
  for (int it = 0; it < GEN_CELLS_PER_THREAD; ++it) {
    const int64_t j = col0 + int64_t(it) * GEN_THREADS + threadIdx.x;
    if (j >= g.col_cells) break;
    const int il = int(j % g.n[4]);
    const int64_t q = j / g.n[4];
    const int iz = int(q % g.n[3]), iR = int(q / g.n[3]);
    Box3<T> bx;
    bx.R = box_iv<T>(cell_edge(g.lo[2], g.hi[2], g.w[2], iR, g.n[2]), cell_edge(g.lo[2], g.hi[2], g.w[2], iR + 1, g.n[2]));
    bx.Z = box_iv<T>(cell_edge(g.lo[3], g.hi[3], g.w[3], iz, g.n[3]), cell_edge(g.lo[3], g.hi[3], g.w[3], iz + 1, g.n[3]));
    bx.L = box_iv<T>(cell_edge(g.lo[4], g.hi[4], g.w[4], il, g.n[4]), cell_edge(g.lo[4], g.hi[4], g.w[4], il + 1, g.n[4]));
    unsigned v = 0;
    for (int h = 0; h < count; ++h) v += hit_votes_general(bx, sh[h].inv, sh[h].hs, zref) ? 1u : 0u;
    out[j] = uint16_t(v);
  }
}


// ---- fast form ------------------------------------------------------------------------------------
// Block = (event, xy cell, tile of FAST_THREADS (R, lambda) pairs, tile of FAST_ZT z0 cells).
// Thread = one (R, lambda) pair; loops over the hits (outer) and its FAST_ZT z0 cells (inner), so
// that everything depending on (R, lambda, hit, drift sign) is computed once per FAST_ZT cells.
// Vote counts: 8 bytes packed in one 64-bit register (hits per event <= 255 on this path).
#ifndef IA_FAST_THREADS
#define IA_FAST_THREADS 256
#endif
#ifndef IA_FAST_MIN_BLOCKS
#define IA_FAST_MIN_BLOCKS 2
#endif
constexpr int FAST_THREADS = IA_FAST_THREADS;
constexpr int FAST_MIN_BLOCKS = IA_FAST_MIN_BLOCKS;
#ifndef IA_FAST_ZT
#define IA_FAST_ZT 16
#endif
constexpr int FAST_ZT = IA_FAST_ZT;                      // 8 or 16: z0 cells per thread (vote bits + filter bits share 32 bits)
static_assert(FAST_ZT == 8 || FAST_ZT == 16, "FAST_ZT");

template <class T> struct __align__(16) ZTab {
  Iv<T> z[2][FAST_ZT];        // [0]: z0 - z_ref, [1]: its negation
  T zeta, _pad;               // largest |z0 - z_ref| of the tile (prefilter)
};

template <class T> __device__ __noinline__ bool general_votes_norm(const HitF<T>& h, int va, Iv<T> R, Iv<T> Zeff, Iv<T> L, int rig = 0) {
  XYInv<T> v;
  v.Q = h.Q; v.cA = h.cA; v.sA = h.sA[va]; v.dphi = h.dphi[va]; v.iQ = h.iQ; v.RA = h.RA; v.iR = h.iR; v.c2 = h.c2;
  v.s2 = h.s2[va];
  v.forced = 0;
  HitS<T> hs = {h.Tabs, h.Dlo, h.Dhi, 1, rig};
  Box3<T> bx = {R, Zeff, L};
  return hit_votes_general(bx, v, hs, T(0));
}

// one hit, one thread: both drift signs over the thread's z0 cells; returns the vote mask (bit i = z0 cell i)
// (float: bit FAST_ZT + i set = cell i is too close to call in this form, see Filter in ia_fast.cuh)
template <int SS, class T>
IA_DEV unsigned fast_hit(const HitF<T>& h, unsigned h_addr, int va, const PairC<T>& p, const Iv<T>* zt, int nz_tile) {
  const HitP<T> hp = hit_prepare(h, va, p);
  const Pass2<T> pc2 = pass_prepare2(h, p, hp);
  const HitLds<T> hl = {h_addr};
  unsigned bits = 0;
#pragma unroll 1
  for (int i = 0; i < nz_tile; ++i) {
    const unsigned r = pass_vote_q<SS, T>(hl, va, pc2, p, hp, zt[i]);
    bits |= Filter<T>::on ? ((r & 1u) | ((r & 2u) << (FAST_ZT - 1))) << i : r << i;
  }
  return bits;
}

// float: the cells the fast form could not decide are re-taken in the general form (which does the oracle's arithmetic)
template <class T>
IA_DEV unsigned settle(unsigned bits, const HitF<T>& h, int va, Iv<T> R, Iv<T> L, const Iv<T>* zt, int rig = 0) {
  if (Filter<T>::on) {
    unsigned amb = bits >> FAST_ZT;
    bits &= (1u << FAST_ZT) - 1u;
    while (amb) {
      const int i = __ffs(amb) - 1;
      amb &= amb - 1;
      bits = (bits & ~(1u << i)) | (general_votes_norm(h, va, R, zt[i], L, rig) ? 1u << i : 0u);
    }
  }
  return bits;
}

// the same with the sign class as a run-time value (one compiled body, ia_fastq.cuh)
// RIG: rigorous-Phi mode (IA_FLAG_RIGOROUS_PHI); cells whose evaluation leaves the fast form's domain there (bit 2 of the result)
// are re-taken in the general form at once
template <class T, bool RIG = false>
IA_DEV unsigned fast_hit_rt(const HitF<T>& h, unsigned h_addr, int ss, int va, const PairC<T>& p, const Iv<T>* zt, int nz_tile) {
  const HitP<T> hp = hit_prepare(h, va, p);
  const Pass2<T> pc2 = pass_prepare2(h, p, hp);
  const HitLds<T> hl = {h_addr};
  const MR<T> sAm = ss < 0 ? mr_neg(h.sAm[va]) : h.sAm[va], s2m = ss < 0 ? mr_neg(h.s2m[va]) : h.s2m[va];
  const Iv<T> sAabs = ss < 0 ? ineg(h.sA[va]) : h.sA[va], sA2abs = ss < 0 ? ineg(h.sA2[va]) : h.sA2[va];
  unsigned bits = 0;
#pragma unroll 1
  for (int i = 0; i < nz_tile; ++i) {
    unsigned r = pass_vote_qr<RIG, T>(hl, ss, va, pc2, p, hp, zt[i], sAm, s2m, sAabs, sA2abs);
    if (RIG && (r & 4u)) r = general_votes_norm(h, va, p.R, zt[i], p.L, 1) ? 1u : 0u;
    bits |= Filter<T>::on ? ((r & 1u) | ((r & 2u) << (FAST_ZT - 1))) << i : (r & 1u) << i;
  }
  return bits;
}

// 8 vote bits -> 8 packed byte counters (bit k -> byte k).  Four bits at a time: in k + 7j, k,j < 4,
// no two partial products meet, so nothing carries.
IA_DEV unsigned long long spread8(unsigned bits) {
  const unsigned lo = ((bits & 0xfu) * 0x00204081u) & 0x01010101u;
  const unsigned hi = (((bits >> 4) & 0xfu) * 0x00204081u) & 0x01010101u;
  return ((unsigned long long)hi << 32) | lo;
}

// RT: the sign class of a hit as a run-time value in one compiled body (coarse grids, where all three
// classes are live on every SM and three bodies overflow the instruction cache) or as a template
// argument of three bodies (fine grids: 6 % faster there).  Same arithmetic, same results.
// SPLIT: the hit range is divided over blockIdx.z (small launches only; a separate instantiation so that the
// main path keeps its code: with the split as a run-time case C1 and C3 ran 0.5-0.9 % slower).
template <class T, bool RT, bool SPLIT, bool RIG = false>
__global__ void __launch_bounds__(FAST_THREADS, FAST_MIN_BLOCKS)
vote_dense_fast_kernel(HitSpan sp, const HitC<T>* __restrict__ staged, GridDesc g, int tiles_p, int tiles_z, int zt,
                       int per_split, int prefilter, uint16_t* __restrict__ votes) {
  pdl_wait();                 // programmatic dependent launch: nothing before the kernels in front have completed
  extern __shared__ __align__(16) unsigned char smem_raw[];
  ZTab<T>* ztab = reinterpret_cast<ZTab<T>*>(smem_raw);
  HitF<T>* sh = reinterpret_cast<HitF<T>*>(smem_raw + sizeof(ZTab<T>));
  const int e = blockIdx.y;
  int64_t bid = blockIdx.x;
  const int tz = int(bid % tiles_z); bid /= tiles_z;
  const int tp = int(bid % tiles_p); bid /= tiles_p;
  const int64_t ixy = bid;
  const int ixl = int(ixy / g.n[1]), iy = int(ixy - int64_t(ixl) * g.n[1]);
  const int ix = g.ix0 + ixl;                                   // ixy counts inside the slab, ix in the full grid
  int count;
  if (sp.offsets) {
    count = sp.offsets[e + 1] - sp.offsets[e];
    if (count > sp.max_hits) count = sp.max_hits;
    if (count < 0) count = 0;
  } else {
    count = sp.n_hits_single;
  }
  const int nR = g.n[2], nz = g.n[3], nL = g.n[4];
  const Iv<T> X = box_iv<T>(cell_edge(g.lo[0], g.hi[0], g.w[0], ix, g.n[0]), cell_edge(g.lo[0], g.hi[0], g.w[0], ix + 1, g.n[0]));
  const Iv<T> Y = box_iv<T>(cell_edge(g.lo[1], g.hi[1], g.w[1], iy, g.n[1]), cell_edge(g.lo[1], g.hi[1], g.w[1], iy + 1, g.n[1]));
  const T Rlo_min = Rnd<T>::from_dn(g.lo[2]);
  const T Lmag = mx(fabs(Rnd<T>::from_dn(g.lo[4])), fabs(Rnd<T>::from_up(g.hi[4])));
  T zref = T(0);
  if (count > 0) zref = staged[int64_t(e) * sp.max_hits].zref;
  // small launches split the hit range over blockIdx.z (a single event on a coarse grid would otherwise leave every
  // thread a serial chain of all its hits): block z votes the hits [z*per_split, (z+1)*per_split) into its own
  // partial accumulator votes + z*(n_events*cells); sum_partial_votes_kernel adds them up - no atomics
  const int h_begin = SPLIT ? blockIdx.z * per_split : 0;
  const int h_end = SPLIT ? ((h_begin + per_split < count) ? h_begin + per_split : count) : count;
  if (SPLIT) {
    votes += int64_t(blockIdx.z) * (int64_t(gridDim.y) * g.cells);
    sh -= h_begin;                                      // sh[h] for h in [h_begin, h_end)
  }
  for (int h = h_begin + threadIdx.x; h < h_end; h += blockDim.x) {
    const HitC<T> c = staged[int64_t(e) * sp.max_hits + h];
    make_hitf(xy_invariants(X, Y, c), hit_small(c), Rlo_min, Lmag, sh[h]);
  }
  const int iz0 = tz * zt;                              // zt <= FAST_ZT z0 cells per block (launcher's choice)
  const int nz_tile = (nz - iz0) < zt ? (nz - iz0) : zt;
  if (threadIdx.x < FAST_ZT) {
    const int iz = iz0 + (threadIdx.x < nz_tile ? threadIdx.x : nz_tile - 1);
    const Iv<T> Z = box_iv<T>(cell_edge(g.lo[3], g.hi[3], g.w[3], iz, nz), cell_edge(g.lo[3], g.hi[3], g.w[3], iz + 1, nz));
    const Iv<T> Zr = isub(Z, thin(zref));
    ztab->z[0][threadIdx.x] = Zr;
    ztab->z[1][threadIdx.x] = ineg(Zr);
    // (threads beyond nz_tile repeat the last cell, so the maximum over all FAST_ZT lanes is the tile's)
    T zm = mx(fabs(Zr.lo), fabs(Zr.hi));
#pragma unroll
    for (int off = FAST_ZT / 2; off > 0; off >>= 1) zm = mx(zm, __shfl_xor_sync((1u << FAST_ZT) - 1u, zm, off));
    if (threadIdx.x == 0) ztab->zeta = zm;
  }
  __syncthreads();
  // shared-window address of (virtual) record 0: the conversion is applied to a record that exists, sh[h_begin], and
  // the shift is taken in unsigned arithmetic afterwards - in the SPLIT case sh itself may point below the window, where
  // cvta.to.shared is undefined; every address formed from sh_addr is sh_addr + h*sizeof(HitF) with h >= h_begin
  const unsigned sh_addr = hit_address(sh + h_begin) - unsigned(h_begin) * unsigned(sizeof(HitF<T>));
  // pair enumeration: R fastest, then the lambda index within its half, then the half - a warp's lambda cells share a
  // sign, and along R the sign of z_A = (z0 - z_ref) + lambda R dphi is the same for every lane of most warps, which
  // pass_vote_q uses (round 2: C4 1.2226 -> 1.2080 s; the stores of a warp are then strided, 2 bytes per cell in 1.2 s)
  const int n_pairs = nR * nL;
  const int hl = (nL % 2 == 0) ? nL / 2 : nL;
  int p = tp * FAST_THREADS + threadIdx.x;
  const bool live = p < n_pairs;
  if (!live) p = n_pairs - 1;
  const int iR = p % nR;
  const int rest = p / nR;
  const int il_in = rest % hl, half = rest / hl;
  const int iL = half * hl + il_in;
  const Iv<T> R = box_iv<T>(cell_edge(g.lo[2], g.hi[2], g.w[2], iR, nR), cell_edge(g.lo[2], g.hi[2], g.w[2], iR + 1, nR));
  const Iv<T> Lraw = box_iv<T>(cell_edge(g.lo[4], g.hi[4], g.w[4], iL, nL), cell_edge(g.lo[4], g.hi[4], g.w[4], iL + 1, nL));
  const int lcls = cls_of(Lraw);
  const bool allP = __all_sync(0xffffffffu, lcls == CLS_P), allN = __all_sync(0xffffffffu, lcls == CLS_N);
  const bool a = !allP && allN;                       // S_a: flip lambda, z0 - z_ref and T for this warp
  const bool warp_fast = allP || allN;
  PairC<T> pr;
  pr.L = a ? ineg(Lraw) : Lraw;
  pr.R = R;
  pr.Lm = to_mr(pr.L);
  pr.LRm = to_mr(warp_fast ? mul_pp(pr.L, R) : imul(pr.L, R));
  pr.L2 = warp_fast ? mul_pp(pr.L, pr.L) : isqr(pr.L);
  unsigned long long acc[FAST_ZT / 8];
#pragma unroll
  for (int j = 0; j < FAST_ZT / 8; ++j) acc[j] = 0;
  const int va = a ? 1 : 0;
  for (int h = h_begin; h < h_end; ++h) {
    const HitF<T>& hf = sh[h];
    const int kind = hf.kind[va];
    if (kind == HIT_SKIP) continue;
    if (kind == HIT_FORCED) {
#pragma unroll
      for (int j = 0; j < FAST_ZT / 8; ++j) acc[j] += 0x0101010101010101ull;
      continue;
    }
    const Iv<T>* zt = ztab->z[hf.zflip];
    if (kind != HIT_GENERAL && warp_fast) {
      // IA_FLAG_PREFILTER: a crude enclosure over the whole z0 tile excludes this hit for every lane -> nobody votes
      // (not in the rigorous-Phi mode: the bound is built on the series value of Phi - Phi_Ax)
      if (!RIG && prefilter && __all_sync(0xffffffffu, crude_excludes(hf, pr, ztab->zeta))) continue;
      unsigned bits;
      if (RT) bits = fast_hit_rt<T, RIG>(hf, sh_addr + unsigned(h) * unsigned(sizeof(HitF<T>)), kind == HIT_FAST_P ? 1 : (kind == HIT_FAST_N ? -1 : 0), va, pr, zt, nz_tile);
      else if (kind == HIT_FAST_P) bits = fast_hit<1, T>(hf, sh_addr + unsigned(h) * unsigned(sizeof(HitF<T>)), va, pr, zt, nz_tile);
      else if (kind == HIT_FAST_N) bits = fast_hit<-1, T>(hf, sh_addr + unsigned(h) * unsigned(sizeof(HitF<T>)), va, pr, zt, nz_tile);
      else bits = fast_hit<0, T>(hf, sh_addr + unsigned(h) * unsigned(sizeof(HitF<T>)), va, pr, zt, nz_tile);
      bits = settle(bits, hf, va, R, pr.L, zt, RIG ? 1 : 0);
#pragma unroll
      for (int j = 0; j < FAST_ZT / 8; ++j) acc[j] += spread8((bits >> (8 * j)) & 0xffu);
    } else {
      unsigned bits = 0;
      for (int i = 0; i < nz_tile; ++i) bits |= (general_votes_norm(hf, va, R, zt[i], pr.L, RIG ? 1 : 0) ? 1u : 0u) << i;
#pragma unroll
      for (int j = 0; j < FAST_ZT / 8; ++j) acc[j] += spread8((bits >> (8 * j)) & 0xffu);
    }
  }
  if (live) {
    uint16_t* out = votes + int64_t(e) * g.cells + ixy * g.col_cells + (int64_t(iR) * nz + iz0) * nL + iL;
#pragma unroll
    for (int i = 0; i < FAST_ZT; ++i)
      if (i < nz_tile) out[int64_t(i) * nL] = uint16_t((acc[i >> 3] >> (8 * (i & 7))) & 0xffu);
  }
}

// partial accumulators of a hit-split launch -> the accumulator (deterministic, no atomics)
__global__ void sum_partial_votes_kernel(const uint16_t* __restrict__ partial, int n_splits, int64_t n, uint16_t* __restrict__ votes) {
  pdl_wait();                 // programmatic dependent launch: nothing before the kernels in front have completed
  for (int64_t i = int64_t(blockIdx.x) * blockDim.x + threadIdx.x; i < n; i += int64_t(gridDim.x) * blockDim.x) {
    unsigned v = 0;
    for (int s = 0; s < n_splits; ++s) v += partial[int64_t(s) * n + i];
    votes[i] = uint16_t(v);
  }
}

// ---- refinement children, sign-specialised form ------------------------------------------------------
// One refinement pass votes the 32 children of each of the k kept boxes (a8-a9).  The 32 children of a
// parent are 4 (xc, yc) sub-cells x 4 (R, lambda) pairs x 2 z0 halves: a4 is computed once per (parent,
// xy sub-cell, hit) into shared memory (the general children kernel recomputes it in every child: 8 x),
// a thread owns one (parent, xy sub-cell, pair) and votes its two z0 children with the one-body fast
// form.  Block = (hit split, event), k*16 threads; the hit range is split so that the records of a split
// fit CHILD_SMEM bytes and a single event still fills the chip; partial[e][split][rank*32 + c].
// A warp holds two parents and four xy sub-cells, so the class of a hit is a per-lane value: the warp
// takes the body of the class all its lanes share, else the universal one (valid for every class).
// records per block (measured on C3, 1,024 events, K = 8: 20 KB 27.6 ms, 37 KB 27.03, 48 KB 27.02, 74 KB 27.25, 96 KB 27.8, 148 KB 29.5)
#ifndef IA_CHILD_SMEM
#define IA_CHILD_SMEM (48 * 1024)
#endif
constexpr int CHILD_SMEM = IA_CHILD_SMEM;
template <class T> struct ZTab2 { Iv<T> z[2][2]; };           // [negated][z half]

__device__ __forceinline__ void child_half(double lo, double hi, int upper, double& clo, double& chi) {
  const double mid = __dmul_rn(0.5, __dadd_rn(lo, hi));       // S9, G18: same midpoint as select_children_kernel
  clo = upper ? mid : lo;
  chi = upper ? hi : mid;
}

// RIG: rigorous-Phi mode (IA_FLAG_RIGOROUS_PHI): the verification loop of pass_vote_qr, as in the dense kernel
template <class T, bool RIG = false>
__global__ void __launch_bounds__(512, 1)
vote_children_fast_kernel(HitSpan sp, const HitC<T>* __restrict__ staged, const ia_box* __restrict__ boxes, int lev,
                          int levels, int k, int per_split, uint16_t* __restrict__ partial) {
  pdl_wait();                 // programmatic dependent launch: nothing before the kernels in front have completed
  extern __shared__ __align__(16) unsigned char smem_raw[];
  ZTab2<T>* ztab = reinterpret_cast<ZTab2<T>*>(smem_raw);
  HitF<T>* rec = reinterpret_cast<HitF<T>*>(smem_raw + size_t(k) * sizeof(ZTab2<T>));
  const int e = blockIdx.y, split = blockIdx.x;
  int count;
  if (sp.offsets) {
    count = sp.offsets[e + 1] - sp.offsets[e];
    if (count > sp.max_hits) count = sp.max_hits;
    if (count < 0) count = 0;
  } else {
    count = sp.n_hits_single;
  }
  const int h0 = split * per_split;
  int nh = count - h0;
  if (nh > per_split) nh = per_split;
  if (nh < 0) nh = 0;
  const ia_box* par = boxes + (int64_t(e) * levels + (lev - 1)) * k;
  const HitC<T>* hits = staged + int64_t(e) * sp.max_hits + h0;
  T zref = T(0);
  if (count > 0) zref = staged[int64_t(e) * sp.max_hits].zref;
  // a4 per (parent, xy sub-cell, hit)
  for (int i = threadIdx.x; i < k * 4 * nh; i += blockDim.x) {
    const int h = i % nh, rx = i / nh, xy = rx & 3, r = rx >> 2;
    double xl, xh, yl, yh;
    child_half(par[r].lo[0], par[r].hi[0], (xy >> 1) & 1, xl, xh);
    child_half(par[r].lo[1], par[r].hi[1], xy & 1, yl, yh);
    const T Rlo_min = Rnd<T>::from_dn(par[r].lo[2]);
    const T Lmag = mx(fabs(Rnd<T>::from_dn(par[r].lo[4])), fabs(Rnd<T>::from_up(par[r].hi[4])));
    const HitC<T> c = hits[h];
    make_hitf(xy_invariants(box_iv<T>(xl, xh), box_iv<T>(yl, yh), c), hit_small(c), Rlo_min, Lmag, rec[rx * per_split + h]);
  }
  for (int i = threadIdx.x; i < k * 2; i += blockDim.x) {
    double zl, zh;
    child_half(par[i >> 1].lo[3], par[i >> 1].hi[3], i & 1, zl, zh);
    const Iv<T> Zr = isub(box_iv<T>(zl, zh), thin(zref));
    ztab[i >> 1].z[0][i & 1] = Zr;
    ztab[i >> 1].z[1][i & 1] = ineg(Zr);
  }
  __syncthreads();
  const bool live = int(threadIdx.x) < k * 16;
  const int t = live ? threadIdx.x : k * 16 - 1;
  const int r = t >> 4, xy = (t >> 2) & 3, rb = (t >> 1) & 1, lb = t & 1;
  double rl, rh, ll, lh;
  child_half(par[r].lo[2], par[r].hi[2], rb, rl, rh);
  child_half(par[r].lo[4], par[r].hi[4], lb, ll, lh);
  const Iv<T> R = box_iv<T>(rl, rh), Lraw = box_iv<T>(ll, lh);
  const int lcls = cls_of(Lraw);
  const bool warp_fast = __all_sync(0xffffffffu, lcls != CLS_M);
  const bool a = lcls == CLS_N;                       // S_a for this lane: flip lambda, z0 - z_ref and T
  const int va = a ? 1 : 0;
  PairC<T> pr;
  pr.L = a ? ineg(Lraw) : Lraw;
  pr.R = R;
  pr.Lm = to_mr(pr.L);
  pr.LRm = to_mr(lcls != CLS_M ? mul_pp(pr.L, R) : imul(pr.L, R));
  pr.L2 = lcls != CLS_M ? mul_pp(pr.L, pr.L) : isqr(pr.L);
  unsigned v0 = 0, v1 = 0;
  const HitF<T>* myrec = rec + (r * 4 + xy) * per_split;
  const unsigned my_addr = hit_address(myrec);          // after the barrier above
  for (int h = 0; h < nh; ++h) {
    const HitF<T>& hf = myrec[h];
    const int kind = hf.kind[va];
    const bool need = kind >= HIT_FAST_P;
    const Iv<T>* zt = ztab[r].z[hf.zflip];
    if (kind == HIT_FORCED) { v0 += 1; v1 += 1; }
    if (!warp_fast || __any_sync(0xffffffffu, kind == HIT_GENERAL)) {
      if (need) {
        v0 += general_votes_norm(hf, va, R, zt[0], pr.L, RIG ? 1 : 0) ? 1u : 0u;
        v1 += general_votes_norm(hf, va, R, zt[1], pr.L, RIG ? 1 : 0) ? 1u : 0u;
      }
    } else {
      const bool allP = __all_sync(0xffffffffu, kind == HIT_FAST_P || !need);
      const bool allN = __all_sync(0xffffffffu, kind == HIT_FAST_N || !need);
      // lanes that do not need the hit (forced, skipped) run along on their record and drop the result
      unsigned bits = fast_hit_rt<T, RIG>(hf, my_addr + unsigned(h) * unsigned(sizeof(HitF<T>)), allP ? 1 : (allN ? -1 : 0), va, pr, zt, 2);
      if (need) {
        bits = settle(bits, hf, va, R, pr.L, zt, RIG ? 1 : 0);
        v0 += bits & 1u; v1 += (bits >> 1) & 1u;
      }
    }
  }
  if (live) {
    uint16_t* out = partial + (int64_t(e) * gridDim.x + split) * (k * 32) + r * 32 + ((xy << 3) | (rb << 2) | lb);
    out[0] = uint16_t(v0);
    out[2] = uint16_t(v1);
  }
}

// ---- diagnostics: the f enclosures of the sign-specialised form, per (box, hit, drift sign) -------------------
// What the dense fast kernel computes for the cell [lo, hi] (one-body variant: same arithmetic as the three-body one),
// next to residual_kernel's general form: out[(box*n_hits + hit)*2 + sign][4] = f.lo, f.hi, scale (R_Ax^2.hi), form
// (0: fast form; 1: forced vote, G15; 2: this (box, hit) takes the general form - guards, lambda straddling 0 - whose
// enclosure is written instead; 3: invalid hit).
template <class T>
__global__ void residual_fast_kernel(HitSpan sp, const HitC<T>* __restrict__ staged, const double* __restrict__ lo,
                                     const double* __restrict__ hi, int64_t n_boxes, double* __restrict__ out) {
  const int n_hits = sp.n_hits_single;
  const int64_t t = int64_t(blockIdx.x) * blockDim.x + threadIdx.x;
  if (t >= n_boxes * n_hits) return;
  const int64_t b = t / n_hits;
  const HitC<T> c = staged[int(t - b * n_hits)];
  const Iv<T> X = box_iv<T>(lo[5 * b + 0], hi[5 * b + 0]), Y = box_iv<T>(lo[5 * b + 1], hi[5 * b + 1]);
  const Iv<T> R = box_iv<T>(lo[5 * b + 2], hi[5 * b + 2]), Z = box_iv<T>(lo[5 * b + 3], hi[5 * b + 3]);
  const Iv<T> Lraw = box_iv<T>(lo[5 * b + 4], hi[5 * b + 4]);
  const XYInv<T> inv = xy_invariants(X, Y, c);
  HitF<T> hf;
  make_hitf(inv, hit_small(c), R.lo, mx(fabs(Lraw.lo), fabs(Lraw.hi)), hf);
  const int lcls = cls_of(Lraw);
  const int va = lcls == CLS_N ? 1 : 0;
  const int kind = hf.kind[va];
  double* o = out + t * 8;
  if (kind == HIT_SKIP || kind == HIT_FORCED || kind == HIT_GENERAL || lcls == CLS_M) {
    const Box3<T> bx = {R, Z, Lraw};
    for (int s = 0; s < 2; ++s) {
      const Resid r = residual_general(bx, inv, hit_small(c), c.zref, s == 0 ? +1 : -1);
      o[4 * s] = r.flo; o[4 * s + 1] = r.fhi; o[4 * s + 2] = r.scale;
      o[4 * s + 3] = kind == HIT_SKIP ? 3.0 : (r.forced ? 1.0 : 2.0);
    }
    return;
  }
  PairC<T> pr;
  pr.L = va ? ineg(Lraw) : Lraw;
  pr.R = R;
  pr.Lm = to_mr(pr.L);
  pr.LRm = to_mr(mul_pp(pr.L, R));
  pr.L2 = mul_pp(pr.L, pr.L);
  const HitP<T> hp = hit_prepare(hf, va, pr);
  const Pass2<T> pc2 = pass_prepare2(hf, pr, hp);
  const int ss = kind == HIT_FAST_P ? 1 : (kind == HIT_FAST_N ? -1 : 0);
  const MR<T> sAm = ss < 0 ? mr_neg(hf.sAm[va]) : hf.sAm[va], s2m = ss < 0 ? mr_neg(hf.s2m[va]) : hf.s2m[va];
  const Iv<T> sAabs = ss < 0 ? ineg(hf.sA[va]) : hf.sA[va], sA2abs = ss < 0 ? ineg(hf.sA2[va]) : hf.sA2[va];
  const Iv<T> Zr = isub(Z, thin(c.zref));
  Iv<T> f[2];
  pass_vote_qr<false, T>(HitDirect<T>{hf}, ss, va, pc2, pr, hp, hf.zflip ? ineg(Zr) : Zr, sAm, s2m, sAabs, sA2abs, f);
  for (int s = 0; s < 2; ++s) { o[4 * s] = f[s].lo; o[4 * s + 1] = f[s].hi; o[4 * s + 2] = hf.Q.hi; o[4 * s + 3] = 0.0; }
}

}  // namespace

cudaError_t launch_residual_fast(ia_ctx* ctx, const HitSpan& sp, const double* lo, const double* hi, int64_t n_boxes,
                                 double* out) {
  const int64_t n = n_boxes * sp.n_hits_single;
  if (n <= 0) return cudaSuccess;
  const unsigned blocks = unsigned((n + 63) / 64);
  if (ctx->params.precision == 32)
    residual_fast_kernel<float><<<blocks, 64, 0, ctx->stream>>>(sp, static_cast<const HitC<float>*>(ctx->staged.p), lo, hi, n_boxes, out);
  else
    residual_fast_kernel<double><<<blocks, 64, 0, ctx->stream>>>(sp, static_cast<const HitC<double>*>(ctx->staged.p), lo, hi, n_boxes, out);
  ctx->launches++;
  return cudaGetLastError();
}

template <class T>
static cudaError_t launch_fast(ia_ctx* ctx, const HitSpan& sp, const GridDesc& g, uint16_t* votes_out) {
  const int n_pairs = g.n[2] * g.n[4];
  int threads = FAST_THREADS;
  if (n_pairs < threads) threads = (n_pairs + 31) / 32 * 32;
  const int tiles_p = (n_pairs + FAST_THREADS - 1) / FAST_THREADS;
  // z0 cells per block: FAST_ZT amortises the per-(pair, hit) terms best; small launches (one event on a
  // coarse grid) take fewer so that the chip still gets about 8 blocks per SM
  int n_sm = 148;
  cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, ctx->device);
  int zt = FAST_ZT;
  {
    const int64_t base = int64_t(g.nx_run) * g.n[1] * ((n_pairs + FAST_THREADS - 1) / FAST_THREADS) * sp.n_events;
    while (zt > 1 && base * ((g.n[3] + zt - 1) / zt) < int64_t(8) * n_sm) zt >>= 1;
  }
  const int tiles_z = (g.n[3] + zt - 1) / zt;
  const int64_t nxy = int64_t(g.nx_run) * g.n[1];
  const int64_t blocks = nxy * tiles_p * tiles_z;
  if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
  // still too few warps to hide the latency of a thread's serial chain over its hits (one event on a coarse grid):
  // split the hits over blockIdx.z, up to 8 ways, aiming at 32 warps per SM
  int n_splits = 1;
  {
    const int64_t warps = blocks * sp.n_events * ((threads + 31) / 32);
    const int64_t want = int64_t(32) * n_sm;
    if (warps < want / 2) n_splits = int(std::min<int64_t>(8, (want + warps - 1) / warps));
    if (n_splits > sp.max_hits) n_splits = sp.max_hits > 0 ? sp.max_hits : 1;
  }
  const int per_split = (sp.max_hits + n_splits - 1) / (n_splits > 0 ? n_splits : 1);
  n_splits = per_split > 0 ? (sp.max_hits + per_split - 1) / per_split : 1;
  const size_t smem = sizeof(ZTab<T>) + size_t(per_split) * sizeof(HitF<T>);
  uint16_t* target = votes_out;
  const int64_t n_acc = int64_t(sp.n_events) * g.cells;
  cudaError_t err;
  if (n_splits > 1) {
    err = scratch_reserve(ctx->partial, size_t(n_splits) * n_acc * sizeof(uint16_t));
    if (err != cudaSuccess) return err;
    target = static_cast<uint16_t*>(ctx->partial.p);
  }
  // coarse = an xy cell is wider than half the chamber radius: the classes of s_Ax, c_Ax then vary from
  // hit to hit inside every block (measured: C3's 8^5 start grid runs 28 % faster with the one-body form,
  // C1's 32^5 grid about the same, C4's 64^5 grid 0.7 % slower)
  const double wxy = std::fmin((g.hi[0] - g.lo[0]) / g.n[0], (g.hi[1] - g.lo[1]) / g.n[1]);
  const bool coarse = (ctx->params.flags & IA_FLAG_ONE_BODY) ? true : ((ctx->params.flags & IA_FLAG_THREE_BODY) ? false : wxy > 0.5 * ctx->max_wire_r);
  dim3 grid((unsigned)blocks, (unsigned)sp.n_events, (unsigned)n_splits);
  const HitC<T>* staged = static_cast<const HitC<T>*>(ctx->staged.p);
#define IA_LAUNCH_FAST(RT_, SPLIT_, RIG_)                                                                                    \
  do {                                                                                                                       \
    err = cudaFuncSetAttribute(vote_dense_fast_kernel<T, RT_, SPLIT_, RIG_>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem)); \
    if (err != cudaSuccess) return err;                                                                                      \
    err = launch_k(ctx, vote_dense_fast_kernel<T, RT_, SPLIT_, RIG_>, grid, dim3(threads), smem, sp, staged, g, tiles_p, tiles_z, zt, \
                   per_split, (ctx->params.flags & IA_FLAG_PREFILTER) ? 1 : 0, target);                                                     \
  } while (0)
  if (ctx->params.flags & IA_FLAG_RIGOROUS_PHI) {
    // rigorous Phi: the one-body variant carries the verification loop (any grid)
    if (n_splits > 1) IA_LAUNCH_FAST(true, true, true); else IA_LAUNCH_FAST(true, false, true);
  } else if (n_splits > 1) {
    if (coarse) IA_LAUNCH_FAST(true, true, false); else IA_LAUNCH_FAST(false, true, false);
  } else {
    if (coarse) IA_LAUNCH_FAST(true, false, false); else IA_LAUNCH_FAST(false, false, false);
  }
#undef IA_LAUNCH_FAST
  ctx->launches++;
  if (err != cudaSuccess || n_splits == 1) return err;
  int sum_blocks = int((n_acc + 1023) / 1024);
  if (sum_blocks > 8 * n_sm) sum_blocks = 8 * n_sm;
  err = launch_k(ctx, sum_partial_votes_kernel, dim3(sum_blocks), dim3(256), 0, target, n_splits, n_acc, votes_out);
  ctx->launches++;
  return err;
}

template <class T>
static cudaError_t launch_general(ia_ctx* ctx, const HitSpan& sp, const GridDesc& g, uint16_t* votes_out) {
  const int per_block = GEN_THREADS * GEN_CELLS_PER_THREAD;
  const int chunks = int((g.col_cells + per_block - 1) / per_block);
  const int64_t nxy = int64_t(g.nx_run) * g.n[1];
  dim3 grid((unsigned)(nxy * chunks), (unsigned)sp.n_events);
  const size_t smem = size_t(sp.max_hits) * sizeof(HitShared<T>);
  cudaError_t err = cudaFuncSetAttribute(vote_dense_general_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem));
  if (err != cudaSuccess) return err;
  err = launch_k(ctx, vote_dense_general_kernel<T>, grid, dim3(GEN_THREADS), smem, sp, static_cast<const HitC<T>*>(ctx->staged.p), g, chunks,
                 votes_out);
  ctx->launches++;
  return err;
}

template <class T>
static cudaError_t launch_children_fast_t(ia_ctx* ctx, const HitSpan& sp, int lev, int levels, int k, int n_sm,
                                          ia_box* boxes, int* n_splits_out, uint16_t** partial_out) {
  int per_split = int(CHILD_SMEM / (size_t(k) * 4 * sizeof(HitF<T>)));
  if (per_split < 1) per_split = 1;
  // few events: split further so that about two blocks per SM exist
  const int want = (2 * n_sm + sp.n_events - 1) / sp.n_events;
  if (want > 1) {
    const int ps = (sp.max_hits + want - 1) / want;
    if (ps < per_split) per_split = ps < 1 ? 1 : ps;
  }
  if (per_split > sp.max_hits) per_split = sp.max_hits;
  if (per_split < 1) per_split = 1;                     // no hits at all: one split that votes nothing
  const int n_splits = sp.max_hits > 0 ? (sp.max_hits + per_split - 1) / per_split : 1;
  cudaError_t err = scratch_reserve(ctx->partial, size_t(sp.n_events) * n_splits * k * 32 * sizeof(uint16_t));
  if (err != cudaSuccess) return err;
  uint16_t* partial = static_cast<uint16_t*>(ctx->partial.p);
  const size_t smem = size_t(k) * sizeof(ZTab2<T>) + size_t(k) * 4 * per_split * sizeof(HitF<T>);
  const int threads = (k * 16 + 31) / 32 * 32;
  dim3 grid(n_splits, sp.n_events);
  const HitC<T>* staged = static_cast<const HitC<T>*>(ctx->staged.p);
  if (ctx->params.flags & IA_FLAG_RIGOROUS_PHI) {
    err = cudaFuncSetAttribute(vote_children_fast_kernel<T, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem));
    if (err != cudaSuccess) return err;
    err = launch_k(ctx, vote_children_fast_kernel<T, true>, grid, dim3(threads), smem, sp, staged, boxes, lev, levels, k, per_split, partial);
  } else {
    err = cudaFuncSetAttribute(vote_children_fast_kernel<T, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem));
    if (err != cudaSuccess) return err;
    err = launch_k(ctx, vote_children_fast_kernel<T, false>, grid, dim3(threads), smem, sp, staged, boxes, lev, levels, k, per_split, partial);
  }
  ctx->launches++;
  *n_splits_out = n_splits;
  *partial_out = partial;
  return err;
}

cudaError_t launch_vote_children_fast(ia_ctx* ctx, const HitSpan& sp, int lev, int levels, int k, int n_sm, ia_box* boxes,
                                      int* n_splits_out, uint16_t** partial_out) {
  if (ctx->params.precision == 32) return launch_children_fast_t<float>(ctx, sp, lev, levels, k, n_sm, boxes, n_splits_out, partial_out);
  return launch_children_fast_t<double>(ctx, sp, lev, levels, k, n_sm, boxes, n_splits_out, partial_out);
}

cudaError_t launch_vote_dense(ia_ctx* ctx, const HitSpan& sp, const GridDesc& g, uint16_t* votes_out) {
  // the fast form packs vote counts in bytes and keeps one HitF per hit in shared memory
  // bit 4 (rigorous Phi): sign-specialised too since round 2 (one-body variant with the verification loop); bits 0 + 4
  // together keep the general form
  const bool fast = !(ctx->params.flags & IA_FLAG_GENERAL) && sp.max_hits <= 255;
  if (ctx->params.precision == 32)
    return fast ? launch_fast<float>(ctx, sp, g, votes_out) : launch_general<float>(ctx, sp, g, votes_out);
  return fast ? launch_fast<double>(ctx, sp, g, votes_out) : launch_general<double>(ctx, sp, g, votes_out);
}

}  // namespace ia
