// ia_vote_dense.cu - steps a3-a6: the dense-grid vote kernel (layer B1, the hot loop).
//
// Condition (4): hit i votes for the cell iff 0 is in the interval extension of
// eq. (2) for either drift sign; votes[cell] = number of such hits.  A block owns one (xc, yc) cell
// of one event and a slice of that cell's (R, z0, lambda) column.  Its threads first compute, once
// per hit, everything of the residual that depends on (xc, yc, hit) only (a4: S2, S3, S3' of
// the atan2, the square root and the two divisions) into shared memory; every thread
// then walks its cells, reads the hits by shared-memory broadcast, keeps its vote count in a
// register and writes one uint16 per cell.  No atomics, no inter-thread traffic in the loop.
#include "ia_internal.h"
#include "ia_residual.cuh"

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
  extern __shared__ __align__(16) unsigned char smem_raw[];
  HitShared<T>* sh = reinterpret_cast<HitShared<T>*>(smem_raw);
  const int e = blockIdx.y;
  const int64_t bid = blockIdx.x;
  const int64_t ixy = bid / chunks_per_col;
  const int chunk = int(bid - ixy * chunks_per_col);
  const int ix = int(ixy / g.n[1]), iy = int(ixy - int64_t(ix) * g.n[1]);
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

}  // namespace

cudaError_t launch_vote_dense(ia_ctx* ctx, const HitSpan& sp, const GridDesc& g, uint16_t* votes_out) {
  const int per_block = GEN_THREADS * GEN_CELLS_PER_THREAD;
  const int chunks = int((g.col_cells + per_block - 1) / per_block);
  const int64_t nxy = int64_t(g.n[0]) * g.n[1];
  dim3 grid((unsigned)(nxy * chunks), (unsigned)sp.n_events);
  cudaError_t err;
  if (ctx->params.precision == 32) {
    const size_t smem = size_t(sp.max_hits) * sizeof(HitShared<float>);
    err = cudaFuncSetAttribute(vote_dense_general_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem));
    if (err != cudaSuccess) return err;
    vote_dense_general_kernel<float><<<grid, GEN_THREADS, smem, ctx->stream>>>(
        sp, static_cast<const HitC<float>*>(ctx->staged.p), g, chunks, votes_out);
  } else {
    const size_t smem = size_t(sp.max_hits) * sizeof(HitShared<double>);
    err = cudaFuncSetAttribute(vote_dense_general_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem));
    if (err != cudaSuccess) return err;
    vote_dense_general_kernel<double><<<grid, GEN_THREADS, smem, ctx->stream>>>(
        sp, static_cast<const HitC<double>*>(ctx->staged.p), g, chunks, votes_out);
  }
  ctx->launches++;
  return cudaGetLastError();
}

}  // namespace ia
