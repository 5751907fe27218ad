// ia_topk.cu - step a7: the K best cells of a vote accumulator (G16).
//
// Pass 1 (topk_partial): the accumulator is read as one stream of 256-vote chunks (16 bytes per lane) dealt
// round-robin to the warps in groups of eight; each warp keeps a sorted top-32 in its lanes (ia_topk.cuh).
// After the first few chunks the entry bar is high, so the common case per 256 votes is three packed
// maxima, one compare per lane and one warp vote - the pass is HBM-bound.  Warps are merged per
// block through shared memory.  Pass 2 (topk_final): the per-block lists of an event are merged and
// the first k entries written out.  Ties on votes are broken by index ascending, carried in the key.
#include <cstdio>
#include <mutex>

#include "ia_internal.h"
#include "ia_topk.cuh"

namespace ia {

namespace {

constexpr int TOPK_THREADS = 256;

// an upper bound of every key among 8 consecutive votes starting at idx0: their largest vote with the smallest index
__device__ __forceinline__ u64 bound_of_8(const uint4 q, int64_t idx0) {
  const unsigned m = __vmaxu2(__vmaxu2(q.x, q.y), __vmaxu2(q.z, q.w));
  return make_key(max(m >> 16, m & 0xffffu), idx0);
}

#ifndef IA_TOPK_UNROLL
#define IA_TOPK_UNROLL 8
#endif
#ifndef IA_TOPK_BLOCKS_PER_SM
#define IA_TOPK_BLOCKS_PER_SM 2
#endif
constexpr int TOPK_UNROLL = IA_TOPK_UNROLL;      // 16-byte loads in flight per lane (large accumulators; small ones take 1)

// grid (blocks_per_event, n_events); votes of event e at votes + e*n.
// The accumulator is read as a stream: chunk c = 256 votes = one 16-byte load per lane; a warp takes TOPK_UNROLL
// consecutive chunks, consecutive warps consecutive groups, so the warps in flight read one contiguous window of the
// accumulator (DRAM pages are read whole; one private range per warp, as in round 1, had every warp on a page of its
// own and reached 37 % of the HBM rate).  All loads of a group are issued before the first is looked at.
template <int U>
__global__ void __launch_bounds__(TOPK_THREADS)
topk_partial(const uint16_t* __restrict__ votes, int64_t n, int k, int64_t idx_base, u64* __restrict__ partial,
             int64_t* __restrict__ idx_out, uint16_t* __restrict__ votes_out, u64* __restrict__ keys_out, int write_final) {
  pdl_wait();                 // programmatic dependent launch: nothing before the kernels in front have completed
  __shared__ u64 smem_keys[(TOPK_THREADS / 32) * 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int e = blockIdx.y;
  const uint16_t* v = votes + int64_t(e) * n;
  const int64_t gw = int64_t(blockIdx.x) * (TOPK_THREADS / 32) + warp;
  const int64_t n_warps = int64_t(gridDim.x) * (TOPK_THREADS / 32);
  // [0, head): votes before the first 16-byte boundary; then n_chunks aligned chunks; then the tail
  int64_t head = int64_t((16 - (reinterpret_cast<uintptr_t>(v) & 15)) & 15) >> 1;
  if (head > n) head = n;
  const int64_t n_chunks = (n - head) / 256;
  const uint16_t* va = v + head;
  u64 mine = 0, kth = 0;
  if (gw == 0) {
    for (int64_t i = 0; i < head; i += 32) {
      const int64_t idx = i + lane;
      warp_offer(mine, kth, idx < head ? make_key(v[idx], idx_base + idx) : 0, k);
    }
  }
  for (int64_t c0 = gw * U; c0 < n_chunks; c0 += n_warps * U) {
    uint4 q[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      q[u] = make_uint4(0u, 0u, 0u, 0u);
      if (c0 + u < n_chunks) q[u] = __ldcs(reinterpret_cast<const uint4*>(va + (c0 + u) * 256 + 8 * lane));
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (c0 + u >= n_chunks) break;
      const int64_t idx0 = idx_base + head + (c0 + u) * 256 + 8 * lane;
      warp_offer_8(mine, kth, q[u], idx0, bound_of_8(q[u], idx0) > kth, k);
    }
  }
  if (gw == n_warps - 1) {
    for (int64_t i = head + n_chunks * 256; i < n; i += 32) {
      const int64_t idx = i + lane;
      warp_offer(mine, kth, idx < n ? make_key(v[idx], idx_base + idx) : 0, k);
    }
  }
  mine = block_merge(mine, smem_keys);
  if (warp == 0) {
    if (write_final) {
      if (keys_out) {
        keys_out[int64_t(e) * 32 + lane] = lane < k ? mine : 0;       // only the first k of a list are exact
      } else if (lane < k) {
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
           uint16_t* __restrict__ votes_out, u64* __restrict__ keys_out) {
  pdl_wait();                 // programmatic dependent launch: nothing before the kernels in front have completed
  __shared__ u64 smem_keys[(TOPK_THREADS / 32) * 32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int e = blockIdx.x;
  const u64* p = partial + int64_t(e) * n_lists * 32;
  u64 mine = 0;
  for (int l = warp; l < n_lists; l += TOPK_THREADS / 32) mine = warp_merge_desc(mine, p[l * 32 + lane]);
  mine = block_merge(mine, smem_keys);
  if (warp == 0) {
    if (keys_out) {
      keys_out[int64_t(e) * 32 + lane] = lane < k ? mine : 0;
    } else if (lane < k) {
      idx_out[int64_t(e) * k + lane] = key_index(mine);
      votes_out[int64_t(e) * k + lane] = key_votes(mine);
    }
  }
}

}  // namespace

cudaError_t launch_topk(ia_ctx* ctx, const uint16_t* votes, int64_t n, int n_events, int k, int64_t* idx_out,
                        uint16_t* votes_out, int64_t idx_base, unsigned long long* keys_out) {
  // 2 blocks per SM over all events, never more than there are groups of chunks (measured on the 2.1 GB accumulator of
  // C4, loads in flight per lane x blocks per SM: 4x8 0.468 ms, 8x4 0.402, 8x2 0.404, 8x3 0.388, 16x2 0.407, 8x1 0.552;
  // on random votes 8x2 is the fastest, 0.396 ms = 5.4 TB/s)
  int sm = 148;
  cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, ctx->device);
  // a chunk whose votes beat the entry bar costs a warp some microseconds (eight sort-and-merge rounds), and every
  // warp's first chunk does: small accumulators (the start grid of a refinement) take one chunk per warp and turn
  const int64_t n_chunks = (n + 255) / 256;
  const int64_t want_blocks = (int64_t(sm) * IA_TOPK_BLOCKS_PER_SM + n_events - 1) / n_events;     // fill the chip across events
  const int unroll = n_chunks >= want_blocks * (TOPK_THREADS / 32) * TOPK_UNROLL ? TOPK_UNROLL : 1;
  const int64_t per_block = int64_t(256) * unroll * (TOPK_THREADS / 32);
  const int64_t max_blocks = (n + per_block - 1) / per_block;
  int64_t blocks = want_blocks < max_blocks ? want_blocks : max_blocks;
  if (blocks < 1) blocks = 1;
  const int write_final = blocks == 1;
  u64* partial = nullptr;
  if (!write_final) {
    cudaError_t err = scratch_reserve(ctx->keys, size_t(n_events) * blocks * 32 * sizeof(u64));
    if (err != cudaSuccess) return err;
    partial = static_cast<u64*>(ctx->keys.p);
  }
  dim3 grid((unsigned)blocks, (unsigned)n_events);
  cudaError_t err;
  if (unroll == 1)
    err = launch_k(ctx, topk_partial<1>, grid, dim3(TOPK_THREADS), 0, votes, n, k, idx_base, partial, idx_out, votes_out, keys_out, write_final);
  else
    err = launch_k(ctx, topk_partial<TOPK_UNROLL>, grid, dim3(TOPK_THREADS), 0, votes, n, k, idx_base, partial, idx_out, votes_out, keys_out,
                   write_final);
  ctx->launches++;
  if (err != cudaSuccess || write_final) return err;
  err = launch_k(ctx, topk_final, dim3(n_events), dim3(TOPK_THREADS), 0, partial, int(blocks), k, idx_out, votes_out, keys_out);
  ctx->launches++;
  return err;
}

// key lists of several accumulators (the slabs of a split vote, gathered from their GPUs) -> the k best of their union
cudaError_t launch_merge_keys(ia_ctx* ctx, const unsigned long long* keys, int n_lists, int k, int64_t* idx_out,
                              uint16_t* votes_out) {
  const cudaError_t err = launch_k(ctx, topk_final, dim3(1), dim3(TOPK_THREADS), 0, keys, n_lists, k, idx_out, votes_out, nullptr);
  ctx->launches++;
  return err;
}

// ---- ia_topk_static: the same two passes with the per-block lists in a fixed array of the device image -----------
// (include/ia.h says who needs this and why).  Everything that concerns the array is in this file: its definition,
// the one place that asks the runtime for its device address, and the launches that are given that address.
namespace {

// One sorted 32-key list per block of the first pass.  256 KB on every GPU that loads this module, until process exit.
static __device__ __align__(256) u64 static_lists[size_t(IA_TOPK_STATIC_LISTS) * 32];

// In host code `static_lists` is only the runtime's handle for the symbol - not an address a kernel could use.  The
// address on a given device is what cudaGetSymbolAddress returns while that device is current; it is looked up once per
// device and kept here.
constexpr int STATIC_MAX_DEVICES = 64;
std::mutex static_mu;
u64* static_lists_on[STATIC_MAX_DEVICES] = {};
thread_local char static_msg[320] = "";

struct CurrentDevice {          // make `dev` current for the scope, restore the caller's device afterwards
  int prev = -1;
  cudaError_t err = cudaSuccess;
  explicit CurrentDevice(int dev) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev);
  }
  ~CurrentDevice() {
    int cur = -1;
    if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
  }
};

// set-up, once per device, with that device current
cudaError_t static_lists_address(int device, u64** out) {
  std::lock_guard<std::mutex> lock(static_mu);
  if (!static_lists_on[device]) {
    u64* p = nullptr;
    const cudaError_t err = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), static_lists);
    if (err != cudaSuccess) return err;
    if (!p) return cudaErrorInvalidSymbol;
    static_lists_on[device] = p;
  }
  *out = static_lists_on[device];
  return cudaSuccess;
}

int static_fail(int code, const char* fmt, long long a = 0, long long b = 0) {
  std::snprintf(static_msg, sizeof(static_msg), fmt, a, b);
  return code;
}

int static_fail_cuda(const char* what, cudaError_t err) {
  std::snprintf(static_msg, sizeof(static_msg), "ia_topk_static: %s failed: %s", what, cudaGetErrorString(err));
  cudaGetLastError();           // a launch-configuration error is sticky until read
  return IA_ERR_CUDA;
}

}  // namespace

}  // namespace ia

extern "C" {

int ia_topk_static(int device, void* cuda_stream, const uint16_t* votes_dev, int64_t n_cells, int k, int64_t* idx_out_dev,
                   uint16_t* votes_out_dev) {
  using namespace ia;
  static_msg[0] = 0;
  if (!votes_dev || !idx_out_dev || !votes_out_dev)
    return static_fail(IA_ERR_ARG, "ia_topk_static: votes_dev, idx_out_dev and votes_out_dev must be device pointers, not NULL");
  if (n_cells <= 0 || k <= 0 || k > n_cells)
    return static_fail(IA_ERR_ARG, "ia_topk_static: needs n_cells >= 1 and 1 <= k <= n_cells (got n_cells = %lld, k = %lld)",
                       (long long)n_cells, (long long)k);
  if (k > IA_MAX_K)
    return static_fail(IA_ERR_CAPACITY, "ia_topk_static: k = %lld is beyond IA_MAX_K = %lld (one key per lane of a warp)",
                       (long long)k, (long long)IA_MAX_K);
  if (n_cells > IA_TOPK_STATIC_MAX_CELLS)
    return static_fail(IA_ERR_CAPACITY, "ia_topk_static: n_cells = %lld is beyond IA_TOPK_STATIC_MAX_CELLS = %lld",
                       (long long)n_cells, (long long)IA_TOPK_STATIC_MAX_CELLS);
  int n_dev = 0;
  cudaError_t err = cudaGetDeviceCount(&n_dev);
  if (err != cudaSuccess) return static_fail_cuda("cudaGetDeviceCount", err);
  if (device < 0 || device >= n_dev)
    return static_fail(IA_ERR_ARG, "ia_topk_static: device %lld does not exist (%lld visible)", (long long)device, (long long)n_dev);
  if (device >= STATIC_MAX_DEVICES)
    return static_fail(IA_ERR_CAPACITY, "ia_topk_static: device %lld is beyond the %lld devices the address table holds",
                       (long long)device, (long long)STATIC_MAX_DEVICES);
  CurrentDevice cur(device);
  if (cur.err != cudaSuccess) return static_fail_cuda("cudaSetDevice", cur.err);
  u64* lists = nullptr;
  if ((err = static_lists_address(device, &lists)) != cudaSuccess) return static_fail_cuda("cudaGetSymbolAddress(static_lists)", err);
  // the grid of launch_topk for one accumulator: two blocks per SM, never more than there are groups of chunks -
  // and never more lists than the array holds
  int sm = 148;
  if ((err = cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess)
    return static_fail_cuda("cudaDeviceGetAttribute", err);
  const int64_t n_chunks = (n_cells + 255) / 256;
  int64_t want_blocks = int64_t(sm) * IA_TOPK_BLOCKS_PER_SM;
  if (want_blocks > IA_TOPK_STATIC_LISTS) want_blocks = IA_TOPK_STATIC_LISTS;
  const int unroll = n_chunks >= want_blocks * (TOPK_THREADS / 32) * TOPK_UNROLL ? TOPK_UNROLL : 1;
  const int64_t per_block = int64_t(256) * unroll * (TOPK_THREADS / 32);
  const int64_t max_blocks = (n_cells + per_block - 1) / per_block;
  int64_t blocks = want_blocks < max_blocks ? want_blocks : max_blocks;
  if (blocks < 1) blocks = 1;              // 1 <= blocks <= IA_TOPK_STATIC_LISTS from here on
  const int write_final = blocks == 1;      // one block: its list is the answer, the array is not touched
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  const dim3 grid((unsigned)blocks, 1u);
  u64* no_keys = nullptr;
  if (unroll == 1)
    topk_partial<1><<<grid, TOPK_THREADS, 0, stream>>>(votes_dev, n_cells, k, int64_t(0), lists, idx_out_dev, votes_out_dev, no_keys,
                                                      write_final);
  else
    topk_partial<TOPK_UNROLL><<<grid, TOPK_THREADS, 0, stream>>>(votes_dev, n_cells, k, int64_t(0), lists, idx_out_dev, votes_out_dev,
                                                                no_keys, write_final);
  if ((err = cudaGetLastError()) != cudaSuccess) return static_fail_cuda("launch of the first pass", err);
  if (write_final) return IA_OK;
  topk_final<<<1, TOPK_THREADS, 0, stream>>>(lists, int(blocks), k, idx_out_dev, votes_out_dev, no_keys);
  if ((err = cudaGetLastError()) != cudaSuccess) return static_fail_cuda("launch of the merge pass", err);
  return IA_OK;
}

const char* ia_topk_static_error(void) { return ia::static_msg; }

}  // extern "C"
