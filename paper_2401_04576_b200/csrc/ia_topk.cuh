// ia_topk.cuh - warp-level top-K primitives (layer B2).
//
// Selection order ("cells where the maximum of votes ... are found"; G16):
// votes descending, linear index ascending.  Both are packed in one 64-bit key
//     key = votes << 48 | (2^48-1 - index)
// so that "larger key = better" is a total order, shuffles and merges are exact and the result does
// not depend on the order in which candidates are seen.  A warp keeps its running top-32 as one key
// per lane, sorted descending by lane; key 0 means "empty".
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ia {

typedef unsigned long long u64;

__device__ __forceinline__ u64 make_key(unsigned votes, int64_t idx) {
  return (u64(votes) << 48) | (0xFFFFFFFFFFFFull - u64(idx));
}
__device__ __forceinline__ int64_t key_index(u64 k) { return int64_t(0xFFFFFFFFFFFFull - (k & 0xFFFFFFFFFFFFull)); }
__device__ __forceinline__ uint16_t key_votes(u64 k) { return uint16_t(k >> 48); }
__device__ __forceinline__ u64 umax64(u64 a, u64 b) { return a > b ? a : b; }
__device__ __forceinline__ u64 umin64(u64 a, u64 b) { return a < b ? a : b; }

// bitonic sort of 32 keys (one per lane), descending by lane
__device__ __forceinline__ u64 warp_sort_desc(u64 x) {
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int k = 2; k <= 32; k <<= 1) {
#pragma unroll
    for (int j = k >> 1; j > 0; j >>= 1) {
      u64 y = __shfl_xor_sync(0xffffffffu, x, j);
      bool desc = (lane & k) == 0;       // direction of the length-k run this lane is in
      bool lower = (lane & j) == 0;      // lower lane of the compared pair
      x = (desc == lower) ? umax64(x, y) : umin64(x, y);
    }
  }
  return x;
}

// mine, other: each sorted descending by lane.  Returns the 32 largest of the 64, sorted descending.
__device__ __forceinline__ u64 warp_merge_desc(u64 mine, u64 other) {
  const int lane = threadIdx.x & 31;
  u64 rev = __shfl_sync(0xffffffffu, other, 31 - lane);
  u64 x = umax64(mine, rev);            // bitonic, holds the top 32 of the union
#pragma unroll
  for (int j = 16; j > 0; j >>= 1) {
    u64 y = __shfl_xor_sync(0xffffffffu, x, j);
    x = ((lane & j) == 0) ? umax64(x, y) : umin64(x, y);
  }
  return x;
}

// offer one candidate per lane to the running list; kth = key held by lane k-1 (the entry bar)
__device__ __forceinline__ void warp_offer(u64& mine, u64& kth, u64 cand, int k) {
  if (__any_sync(0xffffffffu, cand > kth)) {
    mine = warp_merge_desc(mine, warp_sort_desc(cand));
    kth = __shfl_sync(0xffffffffu, mine, k - 1);
  }
}

// insert ONE key x (the same value in every lane, x > kth) into the sorted list: the entries greater than x are the
// lanes [0, pos); x goes to lane pos, the rest moves down one lane, the last entry drops out.  One ballot and one
// 64-bit shuffle instead of a 32-key sort and a merge - the common case of a chunk that beats the entry bar is one
// or two such keys.
__device__ __forceinline__ void warp_insert(u64& mine, u64& kth, u64 x, int k) {
  const int lane = threadIdx.x & 31;
  const int pos = __popc(__ballot_sync(0xffffffffu, mine > x));
  const u64 up = __shfl_up_sync(0xffffffffu, mine, 1);
  if (lane == pos) mine = x;
  else if (lane > pos) mine = up;
  kth = __shfl_sync(0xffffffffu, mine, k - 1);
}

// offer the 8 consecutive votes of every lane (packed in q, first index idx0 per lane).  Few lanes with something above
// the bar: their keys are inserted one at a time, lowest lane first, each lane walking its votes in index order and
// skipping what the rising bar has overtaken.  Many lanes (a warp's first chunks, a plateau): eight sort-and-merge rounds.
__device__ __forceinline__ void warp_offer_8(u64& mine, u64& kth, const uint4 q, int64_t idx0, bool lane_may, int k) {
  const int lane = threadIdx.x & 31;
  const unsigned may = __ballot_sync(0xffffffffu, lane_may);
  if (may == 0u) return;
  if (__popc(may) > 8) {
    const unsigned w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      const unsigned vv = (j & 1) ? (w[j >> 1] >> 16) : (w[j >> 1] & 0xffffu);
      warp_offer(mine, kth, make_key(vv, idx0 + j), k);
    }
    return;
  }
  const u64 lo = (u64(q.y) << 32) | q.x, hi = (u64(q.w) << 32) | q.z;
  int j = 0;
  u64 c = 0;
  auto next = [&]() {
    c = 0;
    while (j < 8) {
      const unsigned vv = unsigned(((j < 4 ? lo : hi) >> (16 * (j & 3))) & 0xffffu);
      const u64 kk = make_key(vv, idx0 + j);
      ++j;
      if (kk > kth) { c = kk; break; }
    }
  };
  if (lane_may) next();
  unsigned m;
  while ((m = __ballot_sync(0xffffffffu, c != 0)) != 0u) {
    const int src = __ffs(m) - 1;
    const u64 x = __shfl_sync(0xffffffffu, c, src);
    if (x > kth) warp_insert(mine, kth, x, k);
    if (lane == src) next();
  }
}

// block-level merge: every warp deposits its list in shared memory (nwarps*32 keys), warp 0 folds
// them together and returns the block's list in its lanes (other warps return garbage)
__device__ __forceinline__ u64 block_merge(u64 mine, u64* smem_keys) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = (blockDim.x + 31) >> 5;
  smem_keys[warp * 32 + lane] = mine;
  __syncthreads();
  if (warp == 0) {
    for (int w = 1; w < nwarps; ++w) mine = warp_merge_desc(mine, smem_keys[w * 32 + lane]);
  }
  return mine;
}

}  // namespace ia
