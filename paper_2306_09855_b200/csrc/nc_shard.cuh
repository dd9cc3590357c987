// nc_shard.cuh -- one shard of a network per context (nc_set_shard; "future work is required to extend the
// algorithm to employing multiple GPUs"; owner-computes generation with redundant random numbers for the
// rules whose target is drawn; reading S1 in include/nc.h).  A sharded context runs every connect call in full into
// staging blocks with the ordinary generators -- so every rule, node arrays, value arrays and the autapse / multapse
// flags need nothing special -- and then keeps the connections whose target it owns, in order:
//   owned_count_kernel : owned connections per tile of kOwnTile staged positions
//   [device-wide exclusive scan; the host reads the total and reserves blocks by Eq. 1]
//   owned_copy_kernel  : ordered compaction of the owned connections into the storage blocks
// No data-path collective: ranks do not exchange connections, they skip what they do not own.
#pragma once

#include "nc_common.cuh"

namespace nc {

constexpr int kOwnThreads = 256, kOwnItems = 16;
constexpr int kOwnTile = kOwnThreads * kOwnItems;

struct ShardFilterParams {
  BlockMap stage;      // the full projection, creation order, positions 0 .. n - 1
  BlockMap store;      // the context's storage blocks
  uint64_t n;          // staged connections
  uint64_t pos0;       // first creation position the owned ones take in the storage
  uint32_t first, count;        // owned node ids: first .. first + count - 1
  uint32_t* tile_count;         // [ceil(n / kOwnTile)]
  const uint32_t* tile_offset;  // exclusive scan of tile_count
};

__device__ __forceinline__ bool owned(const ShardFilterParams& p, uint32_t t) { return t - p.first < p.count; }

// A warp owns kOwnItems * 32 consecutive positions of the tile and walks them 32 at a time (lane = position, so loads and
// the compacted stores are coalesced); the order of the kept connections is the order of the positions.
__device__ __forceinline__ uint32_t owned_mask_of_chunk(const ShardFilterParams& p, uint64_t pos) {
  bool o = false;
  if (pos < p.n) o = owned(p, *tgt_ptr(p.stage, locate(p.stage, pos)));
  return __ballot_sync(0xffffffffu, o);
}

__global__ void __launch_bounds__(kOwnThreads) owned_count_kernel(const __grid_constant__ ShardFilterParams p) {
  __shared__ uint32_t warp_sum[kOwnThreads / 32];
  const uint32_t warp = threadIdx.x >> 5, lane = lane_id();
  const uint64_t base = (uint64_t)blockIdx.x * kOwnTile + (uint64_t)warp * (kOwnItems * 32) + lane;
  uint32_t c = 0;
#pragma unroll 4
  for (int i = 0; i < kOwnItems; ++i) c += __popc(owned_mask_of_chunk(p, base + (uint64_t)i * 32));
  if (lane == 0) warp_sum[warp] = c;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t tot = 0;
#pragma unroll
    for (int w = 0; w < kOwnThreads / 32; ++w) tot += warp_sum[w];
    p.tile_count[blockIdx.x] = tot;
  }
}

__global__ void __launch_bounds__(kOwnThreads) owned_copy_kernel(const __grid_constant__ ShardFilterParams p) {
  __shared__ uint32_t warp_sum[kOwnThreads / 32];
  const uint32_t warp = threadIdx.x >> 5, lane = lane_id();
  const uint64_t base = (uint64_t)blockIdx.x * kOwnTile + (uint64_t)warp * (kOwnItems * 32) + lane;
  uint32_t masks[kOwnItems];
  uint32_t c = 0;
#pragma unroll
  for (int i = 0; i < kOwnItems; ++i) {
    masks[i] = owned_mask_of_chunk(p, base + (uint64_t)i * 32);
    c += __popc(masks[i]);
  }
  if (lane == 0) warp_sum[warp] = c;
  __syncthreads();
  uint32_t before = 0;
  for (uint32_t w = 0; w < warp; ++w) before += warp_sum[w];
  uint64_t out = p.pos0 + p.tile_offset[blockIdx.x] + before;
#pragma unroll
  for (int i = 0; i < kOwnItems; ++i) {
    const uint32_t m = masks[i];
    if (m & (1u << lane)) {
      const BlockAddr a = locate(p.stage, base + (uint64_t)i * 32), b = locate(p.store, out + __popc(m & lanemask_lt()));
      *src_ptr(p.store, b) = *src_ptr(p.stage, a);
      *tgt_ptr(p.store, b) = *tgt_ptr(p.stage, a);
      *w_ptr(p.store, b) = *w_ptr(p.stage, a);
      *d_ptr(p.store, b) = *d_ptr(p.stage, a);
    }
    out += __popc(m);
  }
}

// How many owned connections precede staged position q[k] (the first staged position of a projection): one warp per query
// (a tile's scanned offset plus the owned positions of that tile before q[k]).
__global__ void __launch_bounds__(256) owned_before_kernel(const __grid_constant__ ShardFilterParams p, const uint64_t* __restrict__ q,
                                                          uint32_t n_q, uint64_t* __restrict__ out) {
  const uint32_t k = blockIdx.x * 8u + (threadIdx.x >> 5), lane = lane_id();
  if (k >= n_q) return;
  const uint64_t pos = q[k];
  const uint64_t tile = pos / kOwnTile, tile0 = tile * kOwnTile;
  uint32_t c = 0;
  for (uint64_t x = tile0 + lane; x < pos; x += 32) c += owned(p, *tgt_ptr(p.stage, locate(p.stage, x))) ? 1u : 0u;
  c = __reduce_add_sync(0xffffffffu, c);
  if (lane == 0) out[k] = (pos < p.n ? (uint64_t)p.tile_offset[tile] : (uint64_t)p.tile_offset[(p.n - 1) / kOwnTile] + p.tile_count[(p.n - 1) / kOwnTile]) + (pos < p.n ? c : 0u);
}

}  // namespace nc
