// ia_topk.cu - step a7: the K best cells of a vote accumulator (G16).
//
// Pass 1 (topk_partial): the accumulator is cut into one contiguous range per warp; each warp streams
// its range with 16-byte loads (8 votes per lane) and keeps a sorted top-32 in its lanes
// (ia_topk.cuh).  After the first few chunks the entry bar is high, so the common case per 256
// votes is one compare per lane and one warp vote - the pass is HBM-bound.  Warps are merged per
// block through shared memory.  Pass 2 (topk_final): the per-block lists of an event are merged and
// the first k entries written out.  Ties on votes are broken by index ascending, carried in the key.
#include "ia_internal.h"
#include "ia_topk.cuh"

namespace ia {

namespace {

constexpr int TOPK_THREADS = 256;

__device__ __forceinline__ u64 best_of_8(const uint4 q, int64_t idx0) {
  // the best key among 8 consecutive votes: highest votes, then lowest index
  unsigned w[4] = {q.x, q.y, q.z, q.w};
  u64 best = 0;
#pragma unroll
  for (int i = 3; i >= 0; --i) {
    u64 kb = make_key(w[i] >> 16, idx0 + 2 * i + 1);
    u64 ka = make_key(w[i] & 0xffffu, idx0 + 2 * i);
    best = umax64(best, umax64(ka, kb));
  }
  return best;
}

// grid (blocks_per_event, n_events); votes of event e at votes + e*n
__global__ void __launch_bounds__(TOPK_THREADS)
topk_partial(const uint16_t* __restrict__ votes, int64_t n, int k, int64_t per_warp, u64* __restrict__ partial,
             int64_t* __restrict__ idx_out, uint16_t* __restrict__ votes_out, int write_final) {
  __shared__ u64 smem_keys[(TOPK_THREADS / 32) * 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int e = blockIdx.y;
  const uint16_t* v = votes + int64_t(e) * n;
  const int64_t gw = int64_t(blockIdx.x) * (TOPK_THREADS / 32) + warp;
  int64_t beg = gw * per_warp, end = beg + per_warp;
  if (end > n) end = n;
  u64 mine = 0, kth = 0;
  int64_t i = beg;
  const bool aligned = ((reinterpret_cast<uintptr_t>(v + beg) & 15) == 0);
  if (aligned) {
    for (; i + 256 <= end; i += 256) {
      const int64_t idx0 = i + 8 * lane;
      const uint4 q = *reinterpret_cast<const uint4*>(v + idx0);
      if (__any_sync(0xffffffffu, best_of_8(q, idx0) > kth)) {
        unsigned w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          unsigned vv = (j & 1) ? (w[j >> 1] >> 16) : (w[j >> 1] & 0xffffu);
          warp_offer(mine, kth, make_key(vv, idx0 + j), k);
        }
      }
    }
  }
  for (; i < end; i += 32) {
    const int64_t idx = i + lane;
    u64 cand = idx < end ? make_key(v[idx], idx) : 0;
    warp_offer(mine, kth, cand, k);
  }
  mine = block_merge(mine, smem_keys);
  if (warp == 0) {
    if (write_final) {
      if (lane < k) {
        idx_out[int64_t(e) * k + lane] = key_index(mine);
        votes_out[int64_t(e) * k + lane] = key_votes(mine);
      }
    } else {
      partial[(int64_t(e) * gridDim.x + blockIdx.x) * 32 + lane] = mine;
    }
  }
}

// grid (n_events); merges n_lists lists of 32 keys
__global__ void __launch_bounds__(TOPK_THREADS)
topk_final(const u64* __restrict__ partial, int n_lists, int k, int64_t* __restrict__ idx_out,
           uint16_t* __restrict__ votes_out) {
  __shared__ u64 smem_keys[(TOPK_THREADS / 32) * 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int e = blockIdx.x;
  const u64* p = partial + int64_t(e) * n_lists * 32;
  u64 mine = 0;
  for (int l = warp; l < n_lists; l += TOPK_THREADS / 32) mine = warp_merge_desc(mine, p[l * 32 + lane]);
  mine = block_merge(mine, smem_keys);
  if (warp == 0 && lane < k) {
    idx_out[int64_t(e) * k + lane] = key_index(mine);
    votes_out[int64_t(e) * k + lane] = key_votes(mine);
  }
}

}  // namespace

cudaError_t launch_topk(ia_ctx* ctx, const uint16_t* votes, int64_t n, int n_events, int k, int64_t* idx_out,
                        uint16_t* votes_out) {
  // ranges per warp: multiples of 256 votes so that the 16-byte path stays aligned
  int sm = 148;
  cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, ctx->device);
  const int warps_per_block = TOPK_THREADS / 32;
  int64_t want_blocks = (int64_t(sm) * 8 + n_events - 1) / n_events;          // fill the chip across events
  int64_t max_blocks = (n + 256 * warps_per_block - 1) / (256 * warps_per_block);
  int64_t blocks = want_blocks < max_blocks ? want_blocks : max_blocks;
  if (blocks < 1) blocks = 1;
  int64_t per_warp = (n + blocks * warps_per_block - 1) / (blocks * warps_per_block);
  per_warp = (per_warp + 255) / 256 * 256;
  blocks = (n + per_warp * warps_per_block - 1) / (per_warp * warps_per_block);
  const int write_final = blocks == 1;
  u64* partial = nullptr;
  if (!write_final) {
    cudaError_t err = scratch_reserve(ctx->keys, size_t(n_events) * blocks * 32 * sizeof(u64));
    if (err != cudaSuccess) return err;
    partial = static_cast<u64*>(ctx->keys.p);
  }
  dim3 grid((unsigned)blocks, (unsigned)n_events);
  topk_partial<<<grid, TOPK_THREADS, 0, ctx->stream>>>(votes, n, k, per_warp, partial, idx_out, votes_out, write_final);
  ctx->launches++;
  cudaError_t err = cudaGetLastError();
  if (err != cudaSuccess || write_final) return err;
  topk_final<<<n_events, TOPK_THREADS, 0, ctx->stream>>>(partial, int(blocks), k, idx_out, votes_out);
  ctx->launches++;
  return cudaGetLastError();
}

}  // namespace ia
