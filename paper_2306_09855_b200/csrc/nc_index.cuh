// nc_index.cuh -- index construction over the sorted keys (steps a12-a15 of DESIGN.md):
// group heads (source or delay differs from the previous connection), their device-wide exclusive scan,
// compaction into group_start / group_delay, per-source offsets src_offsets and p_i of Eq. 14, G_i and
// the degree histograms.  Also a generic device-wide exclusive scan used by pairwise_bernoulli.
#pragma once

#include "nc_common.cuh"

namespace nc {

// ---------------------------------------------------------------------------------------------
// Device-wide exclusive scan of a u32 array (reduce -> scan of partials -> downsweep).
// ---------------------------------------------------------------------------------------------
constexpr int kScanThreads = 256;
constexpr int kScanItems = 16;
constexpr int kScanChunk = kScanThreads * kScanItems;

// CTA-wide exclusive scan of one value per thread (THREADS threads; every thread calls it); total = the sum over the CTA.
template <int THREADS>
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* warp_tmp /*[THREADS / 32]*/, uint32_t& total) {
  uint32_t inc = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
    if (lane_id() >= (uint32_t)d) inc += t;
  }
  __syncthreads();  // protect warp_tmp against a previous use
  if (lane_id() == 31) warp_tmp[threadIdx.x >> 5] = inc;
  __syncthreads();
  uint32_t base = 0, tot = 0;
#pragma unroll
  for (uint32_t w = 0; w < THREADS / 32; ++w) {
    const uint32_t t = warp_tmp[w];
    if (w < (threadIdx.x >> 5)) base += t;
    tot += t;
  }
  total = tot;
  return base + inc - v;
}

__global__ void __launch_bounds__(kScanThreads) scan_reduce_kernel(const uint32_t* __restrict__ in, uint64_t n,
                                                                  uint32_t* __restrict__ partial) {
  __shared__ uint32_t warp_tmp[kScanThreads / 32];
  const uint64_t base = (uint64_t)blockIdx.x * kScanChunk;
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    const uint64_t idx = base + (uint64_t)i * kScanThreads + threadIdx.x;
    if (idx < n) s += in[idx];
  }
  s = __reduce_add_sync(0xffffffffu, s);
  if (lane_id() == 0) warp_tmp[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t t = 0;
#pragma unroll
    for (int w = 0; w < kScanThreads / 32; ++w) t += warp_tmp[w];
    partial[blockIdx.x] = t;
  }
}

// single CTA: exclusive scan of the partials in place, grand total (64-bit) to *total
__global__ void __launch_bounds__(kScanThreads) scan_partials_kernel(uint32_t* __restrict__ partial, uint64_t n_partial,
                                                                    uint64_t* __restrict__ total) {
  __shared__ uint32_t warp_tmp[kScanThreads / 32];
  uint64_t run = 0;
  for (uint64_t base = 0; base < n_partial; base += kScanThreads) {
    const uint64_t idx = base + threadIdx.x;
    const uint32_t v = idx < n_partial ? partial[idx] : 0u;
    uint32_t tot;
    const uint32_t ex = block_exclusive_scan<256>(v, warp_tmp, tot);
    if (idx < n_partial) partial[idx] = (uint32_t)run + ex;
    run += tot;
  }
  if (threadIdx.x == 0) *total = run;
}

__global__ void __launch_bounds__(kScanThreads) scan_downsweep_kernel(const uint32_t* __restrict__ in, uint64_t n,
                                                                     const uint32_t* __restrict__ partial,
                                                                     uint32_t* __restrict__ out) {
  __shared__ uint32_t warp_tmp[kScanThreads / 32];
  const uint64_t base = (uint64_t)blockIdx.x * kScanChunk + (uint64_t)threadIdx.x * kScanItems;
  uint32_t v[kScanItems];
  uint32_t s = 0;
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    v[i] = (base + i < n) ? in[base + i] : 0u;
    s += v[i];
  }
  uint32_t tot;
  uint32_t ex = block_exclusive_scan<256>(s, warp_tmp, tot) + partial[blockIdx.x];
#pragma unroll
  for (int i = 0; i < kScanItems; ++i) {
    if (base + i < n) out[base + i] = ex;
    ex += v[i];
  }
}

// ---------------------------------------------------------------------------------------------
// Group heads.  Position j is a head iff j == 0 or key[j] != key[j-1] (the key packs source and delay).
// ---------------------------------------------------------------------------------------------
constexpr int kHeadThreads = 256;
constexpr int kHeadItems = 8;
constexpr int kHeadTile = kHeadThreads * kHeadItems;

// Where the sorted (source, delay) keys come from: the packed key array of the pairs sort, or the final
// source / delay arrays written by the record-carrying sort (packed here with a fixed 16-bit delay field).
template <typename K>
struct PackedKeys {
  using KeyT = K;
  const K* k;
  uint32_t delay_bits;
  __device__ __forceinline__ K operator[](uint64_t j) const { return k[j]; }
  // keys of positions base .. base+7 (0 beyond n)
  __device__ __forceinline__ void load8(uint64_t base, uint32_t n, K (&out)[8]) const {
#pragma unroll
    for (int i = 0; i < 8; ++i) out[i] = base + i < n ? k[base + i] : (K)0;
  }
};
struct SoAKeys {
  using KeyT = uint64_t;
  const uint32_t* src;  // 256-byte aligned arrays
  const uint16_t* dly;
  uint32_t delay_bits;  // always 16
  __device__ __forceinline__ uint64_t operator[](uint64_t j) const { return ((uint64_t)src[j] << 16) | dly[j]; }
  // base % 8 == 0: two 128-bit loads of sources and one of delays
  __device__ __forceinline__ void load8(uint64_t base, uint32_t n, uint64_t (&out)[8]) const {
    if (base + 8 <= n) {
      const uint4 s0 = *reinterpret_cast<const uint4*>(src + base);
      const uint4 s1 = *reinterpret_cast<const uint4*>(src + base + 4);
      const uint4 d = *reinterpret_cast<const uint4*>(dly + base);
      out[0] = ((uint64_t)s0.x << 16) | (d.x & 0xffffu);
      out[1] = ((uint64_t)s0.y << 16) | (d.x >> 16);
      out[2] = ((uint64_t)s0.z << 16) | (d.y & 0xffffu);
      out[3] = ((uint64_t)s0.w << 16) | (d.y >> 16);
      out[4] = ((uint64_t)s1.x << 16) | (d.z & 0xffffu);
      out[5] = ((uint64_t)s1.y << 16) | (d.z >> 16);
      out[6] = ((uint64_t)s1.z << 16) | (d.w & 0xffffu);
      out[7] = ((uint64_t)s1.w << 16) | (d.w >> 16);
    } else {
#pragma unroll
      for (int i = 0; i < 8; ++i) out[i] = base + i < n ? (*this)[base + i] : 0ull;
    }
  }
};

// The organised connections inside their storage blocks (COPASS organisation, nc_copass.cuh): position j is entry
// j % B of block j / B; source and delay arrays as in the creation-order layout.
struct BlockKeys {
  using KeyT = uint64_t;
  BlockMap map;
  uint32_t delay_bits;  // always 16
  __device__ __forceinline__ uint64_t operator[](uint64_t j) const {
    const BlockAddr a = locate(map, j);
    return ((uint64_t)*src_ptr(map, a) << 16) | *d_ptr(map, a);
  }
  // base % 8 == 0; when B % 8 == 0 the eight positions sit in one block, 16-byte aligned
  __device__ __forceinline__ void load8(uint64_t base, uint32_t n, uint64_t (&out)[8]) const {
    if (base + 8 <= n && (map.B & 7) == 0) {
      const BlockAddr a = locate(map, base);
      const uint32_t* src = src_ptr(map, a);
      const uint4 s0 = *reinterpret_cast<const uint4*>(src);
      const uint4 s1 = *reinterpret_cast<const uint4*>(src + 4);
      const uint4 d = *reinterpret_cast<const uint4*>(d_ptr(map, a));
      out[0] = ((uint64_t)s0.x << 16) | (d.x & 0xffffu);
      out[1] = ((uint64_t)s0.y << 16) | (d.x >> 16);
      out[2] = ((uint64_t)s0.z << 16) | (d.y & 0xffffu);
      out[3] = ((uint64_t)s0.w << 16) | (d.y >> 16);
      out[4] = ((uint64_t)s1.x << 16) | (d.z & 0xffffu);
      out[5] = ((uint64_t)s1.y << 16) | (d.z >> 16);
      out[6] = ((uint64_t)s1.z << 16) | (d.w & 0xffffu);
      out[7] = ((uint64_t)s1.w << 16) | (d.w >> 16);
    } else {
#pragma unroll
      for (int i = 0; i < 8; ++i) out[i] = base + i < n ? (*this)[base + i] : 0ull;
    }
  }
};

// The 8 keys of a thread plus the key just before them: from the lane below, or (lane 0) from memory.
template <typename Keys>
__device__ __forceinline__ void load_keys_and_prev(const Keys& keys, uint64_t base, uint32_t n,
                                                   typename Keys::KeyT (&k)[8], typename Keys::KeyT& prev) {
  using KeyT = typename Keys::KeyT;
  static_assert(kHeadItems == 8, "load8 handles 8 positions");
#pragma unroll
  for (int i = 0; i < 8; ++i) k[i] = (KeyT)0;
  if (base < n) keys.load8(base, n, k);
  const KeyT up = __shfl_up_sync(0xffffffffu, k[7], 1);
  prev = up;
  if (lane_id() == 0) prev = (base > 0 && base < n) ? keys[base - 1] : (KeyT)0;
}

template <typename Keys>
__global__ void __launch_bounds__(kHeadThreads) head_count_kernel(const Keys keys, uint32_t n,
                                                                 uint32_t* __restrict__ tile_heads) {
  using KeyT = typename Keys::KeyT;
  __shared__ uint32_t warp_tmp[kHeadThreads / 32];
  const uint64_t base = (uint64_t)blockIdx.x * kHeadTile + (uint64_t)threadIdx.x * kHeadItems;
  KeyT k[kHeadItems], prev;
  load_keys_and_prev(keys, base, n, k, prev);
  uint32_t c = 0;
#pragma unroll
  for (int i = 0; i < kHeadItems; ++i) {
    const uint64_t j = base + i;
    if (j < n) c += (j == 0 || k[i] != prev) ? 1u : 0u;
    prev = k[i];
  }
  c = __reduce_add_sync(0xffffffffu, c);
  if (lane_id() == 0) warp_tmp[threadIdx.x >> 5] = c;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t t = 0;
#pragma unroll
    for (int w = 0; w < kHeadThreads / 32; ++w) t += warp_tmp[w];
    tile_heads[blockIdx.x] = t;
  }
}

struct IndexOut {
  uint32_t* src_offsets;  // [n_nodes + 1]
  uint32_t* group_ptr;    // [n_nodes + 1]
  uint32_t* group_start;  // [total_groups]
  uint16_t* group_delay;  // [total_groups]
  uint32_t n_nodes;
};

// One thread per kHeadItems consecutive sorted positions.  A head at position j gets group number
// g = (heads before j); if it is also the first connection of its source s, then for every node s' in
// (previous source, s] (the ones in between have no outgoing connection, Q9):
//   src_offsets[s'] = j  and  group_ptr[s'] = g   -- exactly exclusive_scan(out_degree) and Eq. 14.
template <typename Keys>
__global__ void __launch_bounds__(kHeadThreads) index_scatter_kernel(const Keys keys, uint32_t n,
                                                                    const uint32_t* __restrict__ tile_head_off,
                                                                    const uint64_t* __restrict__ total_groups,
                                                                    const __grid_constant__ IndexOut out) {
  using KeyT = typename Keys::KeyT;
  const uint32_t delay_bits = keys.delay_bits;
  __shared__ uint32_t warp_tmp[kHeadThreads / 32];
  const uint64_t base = (uint64_t)blockIdx.x * kHeadTile + (uint64_t)threadIdx.x * kHeadItems;
  KeyT k[kHeadItems];
  KeyT prev0;
  uint32_t flags = 0, c = 0;
  load_keys_and_prev(keys, base, n, k, prev0);
  {
    KeyT prev = prev0;
#pragma unroll
    for (int i = 0; i < kHeadItems; ++i) {
      const uint64_t j = base + i;
      if (j < n && (j == 0 || k[i] != prev)) {
        flags |= 1u << i;
        ++c;
      }
      prev = k[i];
    }
  }
  uint32_t tot;
  uint32_t g = block_exclusive_scan<256>(c, warp_tmp, tot) + tile_head_off[blockIdx.x];
  if (base >= n) return;
  const uint32_t dmask = (1u << delay_bits) - 1u;
  KeyT prev = prev0;
#pragma unroll
  for (int i = 0; i < kHeadItems; ++i) {
    const uint64_t j = base + i;
    if (j < n) {
      if (flags & (1u << i)) {
        const uint32_t s = (uint32_t)(k[i] >> delay_bits);
        out.group_start[g] = (uint32_t)j;
        out.group_delay[g] = (uint16_t)((uint32_t)k[i] & dmask);
        const bool first_of_source = (j == 0) || (uint32_t)(prev >> delay_bits) != s;
        if (first_of_source) {
          const uint32_t lo = (j == 0) ? 0u : (uint32_t)(prev >> delay_bits) + 1u;
          for (uint32_t node = lo; node <= s; ++node) {
            out.src_offsets[node] = (uint32_t)j;
            out.group_ptr[node] = g;
          }
        }
        ++g;
      }
      if (j == (uint64_t)n - 1) {  // nodes after the last source, and the closing entries
        const uint32_t s = (uint32_t)(k[i] >> delay_bits);
        const uint32_t tg = (uint32_t)(*total_groups);
        for (uint64_t node = (uint64_t)s + 1; node <= out.n_nodes; ++node) {
          out.src_offsets[node] = n;
          out.group_ptr[node] = tg;
        }
      }
      prev = k[i];
    }
  }
}

// The same step over the final source / delay arrays of the record-carrying sort, written for the common case:
// 128-bit loads, 32-bit compares, and all per-head work behind a find-first-set loop over the (sparse) head mask --
// heads are a few percent of the connections, so the kernel is a streaming read.
__global__ void __launch_bounds__(kHeadThreads) index_scatter_soa_kernel(const uint32_t* __restrict__ src,
                                                                        const uint16_t* __restrict__ dly, uint32_t n,
                                                                        const uint32_t* __restrict__ tile_head_off,
                                                                        const uint64_t* __restrict__ total_groups,
                                                                        const __grid_constant__ IndexOut out) {
  __shared__ uint32_t warp_tmp[kHeadThreads / 32];
  const uint32_t base = blockIdx.x * (uint32_t)kHeadTile + threadIdx.x * 8u;  // n < 2^32 and tiles are 2048 wide
  const bool in_range = base < n && (uint64_t)blockIdx.x * kHeadTile + threadIdx.x * 8u < n;
  uint32_t s[9], d[9];  // [0] = the connection just before this thread's eight
#pragma unroll
  for (int i = 0; i < 9; ++i) s[i] = d[i] = 0;
  uint32_t cnt = 0;  // how many of the eight exist
  if (in_range) {
    if (n - base >= 8u) {
      const uint4 s0 = *reinterpret_cast<const uint4*>(src + base);
      const uint4 s1 = *reinterpret_cast<const uint4*>(src + base + 4);
      const uint4 dd = *reinterpret_cast<const uint4*>(dly + base);
      s[1] = s0.x; s[2] = s0.y; s[3] = s0.z; s[4] = s0.w; s[5] = s1.x; s[6] = s1.y; s[7] = s1.z; s[8] = s1.w;
      d[1] = dd.x & 0xffffu; d[2] = dd.x >> 16; d[3] = dd.y & 0xffffu; d[4] = dd.y >> 16;
      d[5] = dd.z & 0xffffu; d[6] = dd.z >> 16; d[7] = dd.w & 0xffffu; d[8] = dd.w >> 16;
      cnt = 8;
    } else {
      cnt = n - base;
#pragma unroll
      for (int i = 0; i < 8; ++i)
        if ((uint32_t)i < cnt) {
          s[i + 1] = src[base + i];
          d[i + 1] = dly[base + i];
        }
    }
  }
  // the predecessor: last element of the lane below, or (lane 0) from memory
  const uint32_t up_s = __shfl_up_sync(0xffffffffu, s[8], 1), up_d = __shfl_up_sync(0xffffffffu, d[8], 1);
  s[0] = up_s;
  d[0] = up_d;
  if (lane_id() == 0 && in_range && base > 0) {
    s[0] = src[base - 1];
    d[0] = dly[base - 1];
  }
  uint32_t heads = 0, first_of_source = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const bool new_s = s[i + 1] != s[i];
    if (new_s | (d[i + 1] != d[i])) heads |= 1u << i;
    if (new_s) first_of_source |= 1u << i;
  }
  if (base == 0) {  // position 0 is a head and the first connection of its source
    heads |= 1u;
    first_of_source |= 1u;
  }
  const uint32_t live = cnt >= 8 ? 0xffu : ((1u << cnt) - 1u);
  heads &= live;
  first_of_source &= live;
  uint32_t tot;
  uint32_t g = block_exclusive_scan<256>(__popc(heads), warp_tmp, tot) + tile_head_off[blockIdx.x];
  uint32_t m = heads;
  while (m) {
    const int i = __ffs(m) - 1;
    m &= m - 1;
    const uint32_t j = base + i;
    // heads are ~1 % of the positions: their keys are re-read (cache hits) instead of selected out of the registers
    const uint32_t si = __ldg(src + j), di = __ldg(dly + j), sp = j ? __ldg(src + j - 1) : 0u;
    out.group_start[g] = j;
    out.group_delay[g] = (uint16_t)di;
    if (first_of_source & (1u << i)) {
      const uint32_t lo = j == 0 ? 0u : sp + 1u;  // nodes in between have no outgoing connection (Q9)
      for (uint32_t node = lo; node <= si; ++node) {
        out.src_offsets[node] = j;
        out.group_ptr[node] = g;
      }
    }
    ++g;
  }
  if (cnt > 0 && base + cnt == n) {  // nodes after the last source, and the closing entries
    uint32_t sl = s[1];
#pragma unroll
    for (int q = 1; q < 8; ++q)
      if (cnt == (uint32_t)q + 1) sl = s[q + 1];
    const uint32_t tg = (uint32_t)(*total_groups);
    for (uint64_t node = (uint64_t)sl + 1; node <= out.n_nodes; ++node) {
      out.src_offsets[node] = n;
      out.group_ptr[node] = tg;
    }
  }
}


// ---------------------------------------------------------------------------------------------
// The whole index in ONE read of the final source / delay arrays (NC_INDEX_FUSED=1; needs group arrays sized from the
// analytic bound; measured slower than the two streaming reads, see build_index_from_sorted): a tile of kFusedTile positions keeps its keys in registers, counts its heads, chains the
// count to the tiles before it with a decoupled look-back (one status word per tile: a warp polls 32 predecessors per
// load), and writes group_start / group_delay / src_offsets / group_ptr with the keys it still holds.  Replaces
// head_count_kernel + the three scan kernels + index_scatter_soa_kernel (two reads of the keys).
//   status word: bits 0..31 heads | bit 32 = aggregate of this tile published | bit 33 = inclusive prefix published
// Tiles are handed out by a ticket so that a tile only ever waits on tiles that already run.
// ---------------------------------------------------------------------------------------------
constexpr int kFusedChunks = 2;  // chunks of 8 consecutive positions per thread
constexpr int kFusedThreads = 1024;  // one CTA per SM: 148 tiles in flight, so a look-back walks at most 5 polls of 32
constexpr int kFusedTile = kFusedThreads * 8 * kFusedChunks;
constexpr uint64_t kStatAggregate = 1ull << 32, kStatInclusive = 2ull << 32;

__global__ void __launch_bounds__(kFusedThreads) index_fused_kernel(const uint32_t* __restrict__ src,
                                                                  const uint16_t* __restrict__ dly, uint32_t n,
                                                                  uint64_t* __restrict__ status, uint32_t* __restrict__ ticket,
                                                                  uint64_t* __restrict__ total_groups,
                                                                  uint32_t* __restrict__ error_flag,
                                                                  const __grid_constant__ IndexOut out) {
  __shared__ uint32_t warp_tmp[kFusedThreads / 32];
  __shared__ uint32_t sh_tile, sh_prefix;
  if (threadIdx.x == 0) sh_tile = atomicAdd(ticket, 1u);
  __syncthreads();
  const uint32_t tile = sh_tile;
  uint32_t s[kFusedChunks][9], d[kFusedChunks][9], cnt[kFusedChunks], heads[kFusedChunks], first_src[kFusedChunks];
  uint32_t my_heads = 0;
#pragma unroll
  for (int c = 0; c < kFusedChunks; ++c) {
    // chunk c of the tile: thread t owns positions tile * kFusedTile + c * 8 * kFusedThreads + t * 8 .. + 7
    const uint64_t base64 = (uint64_t)tile * kFusedTile + (uint64_t)c * (kFusedThreads * 8) + threadIdx.x * 8u;
    const uint32_t base = (uint32_t)base64;
    const bool in_range = base64 < n;
#pragma unroll
    for (int i = 0; i < 9; ++i) s[c][i] = d[c][i] = 0;
    cnt[c] = 0;
    if (in_range) {
      if (n - base >= 8u) {
        const uint4 s0 = *reinterpret_cast<const uint4*>(src + base);
        const uint4 s1 = *reinterpret_cast<const uint4*>(src + base + 4);
        const uint4 dd = *reinterpret_cast<const uint4*>(dly + base);
        s[c][1] = s0.x; s[c][2] = s0.y; s[c][3] = s0.z; s[c][4] = s0.w; s[c][5] = s1.x; s[c][6] = s1.y; s[c][7] = s1.z; s[c][8] = s1.w;
        d[c][1] = dd.x & 0xffffu; d[c][2] = dd.x >> 16; d[c][3] = dd.y & 0xffffu; d[c][4] = dd.y >> 16;
        d[c][5] = dd.z & 0xffffu; d[c][6] = dd.z >> 16; d[c][7] = dd.w & 0xffffu; d[c][8] = dd.w >> 16;
        cnt[c] = 8;
      } else {
        cnt[c] = n - base;
#pragma unroll
        for (int i = 0; i < 8; ++i)
          if ((uint32_t)i < cnt[c]) {
            s[c][i + 1] = src[base + i];
            d[c][i + 1] = dly[base + i];
          }
      }
    }
    const uint32_t up_s = __shfl_up_sync(0xffffffffu, s[c][8], 1), up_d = __shfl_up_sync(0xffffffffu, d[c][8], 1);
    s[c][0] = up_s;
    d[c][0] = up_d;
    if (lane_id() == 0 && in_range && base > 0) {
      s[c][0] = src[base - 1];
      d[c][0] = dly[base - 1];
    }
    uint32_t h = 0, f = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const bool new_s = s[c][i + 1] != s[c][i];
      if (new_s | (d[c][i + 1] != d[c][i])) h |= 1u << i;
      if (new_s) f |= 1u << i;
    }
    if (in_range && base == 0) {  // position 0 is a head and the first connection of its source
      h |= 1u;
      f |= 1u;
    }
    const uint32_t live = cnt[c] >= 8 ? 0xffu : ((1u << cnt[c]) - 1u);
    heads[c] = h & live;
    first_src[c] = f & live;
    my_heads += __popc(heads[c]);
  }
  // exclusive scan in POSITION order: chunk 0 of every thread precedes chunk 1 of any thread
  uint32_t tot0, tot1;
  const uint32_t ex0 = block_exclusive_scan<kFusedThreads>(__popc(heads[0]), warp_tmp, tot0);
  const uint32_t ex1 = block_exclusive_scan<kFusedThreads>(__popc(heads[1]), warp_tmp, tot1) + tot0;
  const uint32_t tile_total = tot0 + tot1;
  static_assert(kFusedChunks == 2, "the scan above is written for two chunks");
  (void)my_heads;

  // ---- chain the tile's head count to the tiles before it ----
  if (threadIdx.x < 32) {
    uint64_t* my_status = status + tile;
    uint32_t excl = 0;
    if (tile == 0) {
      if (threadIdx.x == 0) st_relaxed_u64(my_status, kStatInclusive | tile_total);
    } else {
      if (threadIdx.x == 0) st_relaxed_u64(my_status, kStatAggregate | tile_total);
      int64_t t = (int64_t)tile - 1;
      uint32_t spins = 0;
      while (true) {
        const int64_t mine = t - (int64_t)lane_id();
        const uint64_t w = mine >= 0 ? ld_relaxed_u64(status + mine) : kStatInclusive;  // before tile 0: prefix 0
        const uint32_t ready = __ballot_sync(0xffffffffu, (w >> 32) != 0);
        const uint32_t incl = __ballot_sync(0xffffffffu, (w >> 33) != 0);
        // usable: the run of ready predecessors starting at lane 0, up to and including the first inclusive one
        const uint32_t run = __ffs(~ready) - 1;  // 32 when all are ready (ffs(0) = 0 -> wraps to 0xffffffff: handled below)
        uint32_t usable = ready == 0xffffffffu ? 32u : run;
        const uint32_t first_incl = incl ? (uint32_t)__ffs(incl) - 1u : 32u;
        const bool done = first_incl < usable;
        if (done) usable = first_incl + 1;
        uint32_t v = lane_id() < usable ? (uint32_t)w : 0u;
        v = __reduce_add_sync(0xffffffffu, v);
        excl += v;
        if (done) break;
        t -= usable;
        if (usable == 0) {
          if (++spins > (1u << 22)) {  // a predecessor is lost: report instead of hanging the device
            if (lane_id() == 0) *error_flag = 1u;
            break;
          }
          __nanosleep(20);
        }
      }
      if (threadIdx.x == 0) st_relaxed_u64(my_status, kStatInclusive | (uint64_t)(excl + tile_total));
    }
    if (threadIdx.x == 0) sh_prefix = excl;
  }
  __syncthreads();
  const uint32_t prefix = sh_prefix;
  const uint64_t tile_end = (uint64_t)tile * kFusedTile + kFusedTile;
  if (threadIdx.x == 0 && tile_end >= n && (uint64_t)tile * kFusedTile < n) *total_groups = (uint64_t)prefix + tile_total;

#pragma unroll
  for (int c = 0; c < kFusedChunks; ++c) {
    const uint32_t base = tile * (uint32_t)kFusedTile + (uint32_t)c * (kFusedThreads * 8) + threadIdx.x * 8u;
    uint32_t g = prefix + (c == 0 ? ex0 : ex1);
    uint32_t m = heads[c];
    while (m) {
      const int i = __ffs(m) - 1;
      m &= m - 1;
      const uint32_t j = base + i;
      uint32_t si = s[c][1], di = d[c][1], sp = s[c][0];
#pragma unroll
      for (int q = 1; q < 8; ++q)
        if (i == q) {
          si = s[c][q + 1];
          di = d[c][q + 1];
          sp = s[c][q];
        }
      out.group_start[g] = j;
      out.group_delay[g] = (uint16_t)di;
      if (first_src[c] & (1u << i)) {
        const uint32_t lo = j == 0 ? 0u : sp + 1u;  // nodes in between have no outgoing connection (Q9)
        for (uint32_t node = lo; node <= si; ++node) {
          out.src_offsets[node] = j;
          out.group_ptr[node] = g;
        }
      }
      ++g;
    }
    if (cnt[c] > 0 && base + cnt[c] == n) {  // nodes after the last source, and the closing entries
      uint32_t sl = s[c][1];
#pragma unroll
      for (int q = 1; q < 8; ++q)
        if (cnt[c] == (uint32_t)q + 1) sl = s[c][q + 1];
      const uint32_t tg = prefix + tile_total;  // this is the last tile: its inclusive prefix is the number of groups
      for (uint64_t node = (uint64_t)sl + 1; node <= out.n_nodes; ++node) {
        out.src_offsets[node] = n;
        out.group_ptr[node] = tg;
      }
    }
  }
}

// G_i = p_{i+1} - p_i and out_degree_i = src_offsets_{i+1} - src_offsets_i, plus the maximum out-degree.
__global__ void __launch_bounds__(256) index_finish_kernel(const uint32_t* __restrict__ src_offsets,
                                                          const uint32_t* __restrict__ group_ptr, uint32_t n_nodes,
                                                          uint32_t* __restrict__ out_degree,
                                                          uint32_t* __restrict__ group_count,
                                                          uint32_t* __restrict__ max_out_degree) {
  const uint32_t s = blockIdx.x * 256u + threadIdx.x;
  uint32_t deg = 0;
  if (s < n_nodes) {
    deg = src_offsets[s + 1] - src_offsets[s];
    out_degree[s] = deg;
    group_count[s] = group_ptr[s + 1] - group_ptr[s];
  }
  deg = __reduce_max_sync(0xffffffffu, deg);
  if (lane_id() == 0 && deg) atomicMax(max_out_degree, deg);
}

// ---------------------------------------------------------------------------------------------
// Degree histograms over the storage blocks (creation order; usable before nc_finalize).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) degree_count_kernel(const __grid_constant__ BlockMap map, uint64_t n, int kind,
                                                          uint32_t* __restrict__ degree) {
  const uint64_t stride = (uint64_t)gridDim.x * 256u;
  for (uint64_t pos = (uint64_t)blockIdx.x * 256u + threadIdx.x; pos < n; pos += stride) {
    const BlockAddr a = locate(map, pos);
    const uint32_t node = kind == 0 ? *tgt_ptr(map, a) : *src_ptr(map, a);
    atomicAdd(degree + node, 1u);
  }
}

__global__ void __launch_bounds__(256) max_u32_kernel(const uint32_t* __restrict__ v, uint32_t n, uint32_t* __restrict__ out) {
  uint32_t m = 0;
  for (uint64_t i = (uint64_t)blockIdx.x * 256u + threadIdx.x; i < n; i += (uint64_t)gridDim.x * 256u) m = max(m, v[i]);
  m = __reduce_max_sync(0xffffffffu, m);
  if (lane_id() == 0 && m) atomicMax(out, m);
}

// ---------------------------------------------------------------------------------------------
// Receptor port and synaptic group are constants of a projection: they are kept per projection and an
// entry of either view is resolved through its creation position (binary search over the projections' first
// positions).  perm == NULL and perm_off == 0: the creation-order view (position = entry); perm != NULL: the flat
// organised view; perm_off != 0: the organised view inside the storage blocks (creation positions at perm_off).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) attribute_lookup_kernel(const __grid_constant__ BlockMap map, const uint32_t* __restrict__ perm,
                                                              uint64_t perm_off, uint64_t first, uint64_t count,
                                                              const uint32_t* __restrict__ proj_first, uint32_t n_proj,
                                                              const uint16_t* __restrict__ proj_attr,
                                                              uint8_t* __restrict__ port, uint8_t* __restrict__ group) {
  for (uint64_t j = (uint64_t)blockIdx.x * 256u + threadIdx.x; j < count; j += (uint64_t)gridDim.x * 256u) {
    uint32_t pos = (uint32_t)(first + j);
    if (perm) {
      pos = perm[first + j];
    } else if (perm_off) {
      const BlockAddr a = locate(map, first + j);
      pos = reinterpret_cast<const uint32_t*>(a.base + perm_off)[a.slot];
    }
    uint32_t lo = 0, hi = n_proj;  // last projection with proj_first <= pos (empty projections share their start
    while (hi - lo > 1) {          // with the next one and are skipped by taking the last)
      const uint32_t mid = (lo + hi) >> 1;
      if (proj_first[mid] <= pos) lo = mid; else hi = mid;
    }
    const uint16_t a = proj_attr[lo];
    if (port) port[j] = (uint8_t)(a & 0xffu);
    if (group) group[j] = (uint8_t)(a >> 8);
  }
}

}  // namespace nc
