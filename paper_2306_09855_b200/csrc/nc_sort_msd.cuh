// nc_sort_msd.cuh -- bucket-first organisation (NC_FLAG_SORT_BUCKETS): the same stable sort by (source, delay) as
// nc_sort_split.cuh (reading D10: ties keep creation order), arranged so that all digit passes but the first
// run inside the 126 MB L2 instead of through HBM.
//
//   pass A   one stable scatter of all connections (built from the storage blocks, as in the first pass of the default path)
//            into <= 256 BUCKETS of consecutive source ids, bucket(source) = min(umulhi(source, mul), 255) with
//            mul = floor(2^40 / N_nodes): ~N_nodes / 256 sources and ~n / 256 connections per bucket (configs[2]: 302 sources,
//            12 - 31 MB of records).  The host waits for the 256 bucket sizes (1 KB) while this scatter runs.
//   pass B   every bucket is then an independent small sort on the key RELATIVE to the bucket's first key (configs[2]: 15
//            bits = 8 + 7).  Two in-bucket passes (the configs[2] shape): ONE persistent kernel, bucket_sort_kernel, whose CTAs
//            take count and scatter items of the buckets off a ticket counter; bucket i keeps its intermediate records in slot
//            i mod 4, written with L2::evict_last and read back by the second pass.  Any other number of passes, or a bucket
//            above 64 MB: per bucket and pass seg_count_scan_kernel + scatter_pass_kernel (MODE 2 / 3), the buckets round-robin
//            over 2 - 3 CUDA streams with one slot each.  Either way the last pass writes the final arrays at the bucket's place.
//            HBM traffic per connection if the slots never left the L2: 14 + 16 + 1 (pass A) and 16 + 1 + 18 (pass B) = 66 B
//            instead of 102 B for three whole-array passes.
//
// MEASURED (B200, configs[2], profiles/r02_buckets.md): it loses.  Organisation takes 8.5 ms against 6.7 ms for the default
// path.  tests/cuda/membench.cu, section `ring`, shows that the MEMORY SYSTEM gains from the arrangement (two passes as plain
// copies: 3.43 ms whole-array, 2.29 ms with the intermediate in L2 slots), but a tile of scatter_pass_kernel costs 8.8 us of
// SM time with its records in the L2 and 7.9 us with them in HBM: the pass is bound by the SM's shared-memory pipe (ranking and
// staging, ~2 cycles per record per SM, the same with 16 or 36 warps per SM) at almost exactly the rate the HBM write pattern
// allows, so taking the HBM away does not make it faster.  Kept selectable and parity-tested as the evidence for that.
#pragma once

#include "nc_common.cuh"
#include "nc_sort_split.cuh"

namespace nc {

// ---------------------------------------------------------------------------------------------
// pass A counts: bucket of every connection straight from the storage blocks
// ---------------------------------------------------------------------------------------------
template <bool VEC>
__global__ void __launch_bounds__(kCountThreads) msd_tile_count_first_kernel(const __grid_constant__ BlockMap map, uint32_t n,
                                                                            uint32_t tile_size, uint32_t mul,
                                                                            uint16_t* __restrict__ counts) {
  __shared__ uint32_t hist[kRadix];
  hist[threadIdx.x] = 0;
  __syncthreads();
  auto bucket = [&](uint32_t s) { return min(__umulhi(s, mul), (uint32_t)kRadix - 1u); };
  const uint64_t tile0 = (uint64_t)blockIdx.x * tile_size;
  const uint32_t valid = (uint32_t)min((uint64_t)tile_size, (uint64_t)n - tile0);
  if (VEC) {
    for (uint32_t e = threadIdx.x * 4; e < valid; e += kCountThreads * 4) {
      const uint64_t pos = tile0 + e;
      if (e + 3 < valid) {
        const uint4 s4 = *reinterpret_cast<const uint4*>(src_ptr(map, locate(map, pos)));
        atomicAdd(&hist[bucket(s4.x)], 1u);
        atomicAdd(&hist[bucket(s4.y)], 1u);
        atomicAdd(&hist[bucket(s4.z)], 1u);
        atomicAdd(&hist[bucket(s4.w)], 1u);
      } else {
        for (uint32_t q = e; q < valid; ++q) atomicAdd(&hist[bucket(*src_ptr(map, locate(map, tile0 + q)))], 1u);
      }
    }
  } else {
    for (uint32_t e = threadIdx.x; e < valid; e += kCountThreads)
      atomicAdd(&hist[bucket(*src_ptr(map, locate(map, tile0 + e)))], 1u);
  }
  __syncthreads();
  counts[(uint64_t)blockIdx.x * kRadix + threadIdx.x] = (uint16_t)hist[threadIdx.x];
}

// ---------------------------------------------------------------------------------------------
// pass B counts + scan of ONE bucket.  CTA c counts the digits (one byte per record, any alignment) of the kSegChunkTiles
// tiles of chunk c -> counts[tile][256], chunk_base[c][256] = the chunk's totals.  The last CTA to finish turns the totals into
// the exclusive scan in (digit, chunk) order = first output position, relative to the bucket, of every chunk's run of every
// digit; scatter_pass_kernel adds the counts of the tiles before its own inside the chunk.  `done` is zero on entry and on exit.
// ---------------------------------------------------------------------------------------------
constexpr int kSegThreads = 1024;
constexpr int kSegScanSegs = kSegThreads / kRadix;

__global__ void __launch_bounds__(kSegThreads) seg_count_scan_kernel(const uint8_t* __restrict__ dig, uint32_t n, uint32_t tile_size,
                                                                    uint16_t* __restrict__ counts, uint32_t* chunk_base,
                                                                    uint32_t* done) {
  __shared__ uint32_t hist[kSegChunkTiles][kRadix];
  __shared__ uint32_t seg_tot[kSegScanSegs][kRadix];
  __shared__ uint32_t warp_tot[kRadix / 32];
  __shared__ uint32_t is_last;
  for (uint32_t i = threadIdx.x; i < kSegChunkTiles * kRadix; i += kSegThreads) (&hist[0][0])[i] = 0;
  __syncthreads();
  const uint32_t chunk = blockIdx.x, n_chunks = gridDim.x;
  const uint64_t c0 = (uint64_t)chunk * kSegChunkTiles * tile_size;
  const uint32_t len = (uint32_t)min((uint64_t)kSegChunkTiles * tile_size, (uint64_t)n - c0);
  {
    // aligned 16-byte words covering [a0, a0 + len); bytes outside it are skipped (they belong to the same allocation)
    const uintptr_t a0 = reinterpret_cast<uintptr_t>(dig + c0), a1 = a0 + len;
    const uintptr_t v0 = a0 & ~(uintptr_t)15;
    for (uintptr_t v = v0 + (uintptr_t)threadIdx.x * 16; v < a1; v += (uintptr_t)kSegThreads * 16) {
      const uint4 q = *reinterpret_cast<const uint4*>(v);
      const uint32_t w[4] = {q.x, q.y, q.z, q.w};
      const bool inside = v >= a0 && v + 16 <= a1;
      const uint32_t first_tile = (uint32_t)((v < a0 ? 0 : v - a0) / tile_size);
      const bool one_tile = inside && (uint32_t)((v + 15 - a0) / tile_size) == first_tile;
      if (one_tile) {
        uint32_t* h = hist[first_tile];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          atomicAdd(&h[w[j] & 0xffu], 1u);
          atomicAdd(&h[(w[j] >> 8) & 0xffu], 1u);
          atomicAdd(&h[(w[j] >> 16) & 0xffu], 1u);
          atomicAdd(&h[w[j] >> 24], 1u);
        }
      } else {
#pragma unroll
        for (int b = 0; b < 16; ++b) {
          const uintptr_t a = v + b;
          if (a >= a0 && a < a1) atomicAdd(&hist[(uint32_t)((a - a0) / tile_size)][(w[b >> 2] >> ((b & 3) * 8)) & 0xffu], 1u);
        }
      }
    }
  }
  __syncthreads();
  const uint32_t d = threadIdx.x & (kRadix - 1), seg = threadIdx.x / kRadix;
#pragma unroll
  for (uint32_t k = seg; k < kSegChunkTiles; k += kSegScanSegs)
    counts[((uint64_t)chunk * kSegChunkTiles + k) * kRadix + d] = (uint16_t)hist[k][d];
  if (seg == 0) {
    uint32_t tot = 0;
#pragma unroll
    for (uint32_t k = 0; k < kSegChunkTiles; ++k) tot += hist[k][d];
    chunk_base[(uint64_t)chunk * kRadix + d] = tot;
  }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) is_last = atomicAdd(done, 1u) == n_chunks - 1u ? 1u : 0u;
  __syncthreads();
  if (!is_last) return;
  __threadfence();

  // ---- the last CTA: exclusive scan of the chunk totals in (digit, chunk) order, thread (seg, digit) owns a run of chunks ----
  const uint32_t per_seg = (n_chunks + kSegScanSegs - 1) / kSegScanSegs;
  const uint32_t k0 = min(seg * per_seg, n_chunks), k1 = min(k0 + per_seg, n_chunks);
  uint32_t total = 0;
#pragma unroll 8
  for (uint32_t k = k0; k < k1; ++k) total += __ldcg(chunk_base + (uint64_t)k * kRadix + d);
  seg_tot[seg][d] = total;
  __syncthreads();
  uint32_t digit_total = 0, before = 0;
#pragma unroll
  for (int g = 0; g < kSegScanSegs; ++g) {
    const uint32_t v = seg_tot[g][d];
    digit_total += v;
    if ((uint32_t)g < seg) before += v;
  }
  uint32_t inc = digit_total;
#pragma unroll
  for (int s = 1; s < 32; s <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, inc, s);
    if (lane_id() >= (uint32_t)s) inc += t;
  }
  if (seg == 0 && lane_id() == 31) warp_tot[d >> 5] = inc;
  __syncthreads();
  uint32_t run = inc - digit_total + before;
  for (uint32_t w = 0; w < (d >> 5); ++w) run += warp_tot[w];
#pragma unroll 8
  for (uint32_t k = k0; k < k1; ++k) {
    const uint32_t v = __ldcg(chunk_base + (uint64_t)k * kRadix + d);
    chunk_base[(uint64_t)k * kRadix + d] = run;
    run += v;
  }
  if (threadIdx.x == 0) *done = 0u;
}

// ---------------------------------------------------------------------------------------------
// pass B as ONE persistent kernel (two in-bucket digit passes, the configs[2] shape).  Per-bucket launches leave the device
// idle between the dependent kernels of a bucket (count -> scatter -> count -> scatter, each a single wave); here resident
// CTAs take ITEMS off one ticket counter, in an order that puts a full round of other work between an item and what it
// waits for:
//   round r = [count 1 of bucket r] [scatter 1 of bucket r-1] [count 2 of bucket r-2] [scatter 2 of bucket r-3]
// (count = the digits of one chunk of kSegChunkTiles tiles, the last chunk to finish scans the chunk totals; scatter = one
// tile).  An item waits (thread 0 polls a per-bucket counter) only for items with smaller tickets, which CTAs already
// running hold, so the kernel cannot deadlock whatever share of the device it gets.  Bucket i uses intermediate slot
// i mod kBsSlots: four slots are in use at any time, and they stay in the L2.
// ---------------------------------------------------------------------------------------------
constexpr int kBsSlots = 4;
#ifndef NC_BS_WARPS
#define NC_BS_WARPS 8
#define NC_BS_ITEMS 16
#define NC_BS_CTAS 2
#endif
constexpr int kBsWarps = NC_BS_WARPS, kBsItems = NC_BS_ITEMS, kBsCtas = NC_BS_CTAS;
constexpr int kBsThreads = kBsWarps * 32;
constexpr uint32_t kBsTile = kBsThreads * kBsItems;
enum BsSync : int { kBsCount1 = 0, kBsReady1 = 1, kBsTiles1 = 2, kBsCount2 = 3, kBsReady2 = 4, kBsTiles2 = 5, kBsSyncWords = 8 };

struct BucketSortParams {
  const uint4* recs;       // pass A's output, all buckets
  const uint8_t* dig;      // and the first in-bucket digit of every record
  uint4* slot[kBsSlots];
  uint8_t* slot_dig[kBsSlots];
  uint16_t* counts[2][kBsSlots];      // per pass and slot: [tiles][256]
  uint32_t* chunk_base[2][kBsSlots];  //                    [chunks][256]
  uint32_t *out_src, *out_tgt;
  float* out_w;
  uint16_t* out_d;
  uint32_t* out_perm;
  const uint32_t* bstart;       // [nb] the non-empty buckets: first position,
  const uint32_t* bsize;        // [nb] connections,
  const uint32_t* bkey;         // [nb] smallest key
  const uint32_t* round_first;  // [nb + 4] ticket of the first item of every round
  uint32_t* sync;               // [nb][kBsSyncWords], zero on entry
  uint32_t* ticket;             // zero on entry
  uint32_t nb, n_items, delay_bits;
  uint32_t shift[2], bits[2];
  unsigned long long* prof;  // debug (NC_BUCKET_DEBUG): [grid][8] cycles of thread 0: blocked waits, scatter 1, scatter 2, count, items ...
};

__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void wait_at_least(const uint32_t* p, uint32_t want) {
  uint32_t spins = 0;
  while (ld_acquire_u32(p) < want) {
    __nanosleep(spins < 16 ? 100 : 500);
    if (++spins > (1u << 24)) __trap();  // ~8 s: never hang the device
  }
}

// digits of one chunk -> counts[tile][256], chunk_base[chunk][256] = chunk totals; returns through smem whether this CTA was
// the last of the bucket's chunks, in which case it turns the totals into their exclusive scan in (digit, chunk) order
__device__ __forceinline__ void bucket_count_chunk(const uint8_t* dig, uint32_t n, uint32_t chunk, uint32_t n_chunks,
                                                   uint16_t* counts, uint32_t* chunk_base, uint32_t* done_counter,
                                                   uint32_t* ready_flag, uint32_t* hist /* smem [kSegChunkTiles][256] */,
                                                   uint32_t* scratch /* smem [16] */) {
  constexpr uint32_t kTile = kBsTile;
  for (uint32_t i = threadIdx.x; i < kSegChunkTiles * kRadix; i += kBsThreads) hist[i] = 0;
  __syncthreads();
  const uint64_t c0 = (uint64_t)chunk * kSegChunkTiles * kTile;
  const uint32_t len = (uint32_t)min((uint64_t)kSegChunkTiles * kTile, (uint64_t)n - c0);
  {
    const uintptr_t a0 = reinterpret_cast<uintptr_t>(dig + c0), a1 = a0 + len;
    const uintptr_t v0 = a0 & ~(uintptr_t)15;
    for (uintptr_t v = v0 + (uintptr_t)threadIdx.x * 16; v < a1; v += (uintptr_t)kBsThreads * 16) {
      const uint4 q = __ldcg(reinterpret_cast<const uint4*>(v));
      const uint32_t w[4] = {q.x, q.y, q.z, q.w};
      const bool inside = v >= a0 && v + 16 <= a1;
      const uint32_t first_tile = (uint32_t)((v < a0 ? 0 : v - a0) / kTile);
      if (inside && (uint32_t)((v + 15 - a0) / kTile) == first_tile) {
        uint32_t* h = hist + first_tile * kRadix;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          atomicAdd(&h[w[j] & 0xffu], 1u);
          atomicAdd(&h[(w[j] >> 8) & 0xffu], 1u);
          atomicAdd(&h[(w[j] >> 16) & 0xffu], 1u);
          atomicAdd(&h[w[j] >> 24], 1u);
        }
      } else {
#pragma unroll
        for (int b = 0; b < 16; ++b) {
          const uintptr_t a = v + b;
          if (a >= a0 && a < a1) atomicAdd(&hist[(uint32_t)((a - a0) / kTile) * kRadix + ((w[b >> 2] >> ((b & 3) * 8)) & 0xffu)], 1u);
        }
      }
    }
  }
  __syncthreads();
  const uint32_t d = threadIdx.x;
  const bool digit_thread = threadIdx.x < (uint32_t)kRadix;  // whole warps
  if (digit_thread) {
    uint32_t tot = 0;
#pragma unroll
    for (uint32_t k = 0; k < kSegChunkTiles; ++k) {
      const uint32_t v = hist[k * kRadix + d];
      __stcg(counts + ((uint64_t)chunk * kSegChunkTiles + k) * kRadix + d, (uint16_t)v);
      tot += v;
    }
    __stcg(chunk_base + (uint64_t)chunk * kRadix + d, tot);
  }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) scratch[8] = atomicAdd(done_counter, 1u) == n_chunks - 1u ? 1u : 0u;
  __syncthreads();
  if (!scratch[8]) return;
  __threadfence();
  uint32_t total = 0, inc = 0;
  if (digit_thread) {
#pragma unroll 8
    for (uint32_t k = 0; k < n_chunks; ++k) total += __ldcg(chunk_base + (uint64_t)k * kRadix + d);
    inc = total;
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, s);
      if (lane_id() >= (uint32_t)s) inc += t;
    }
    if (lane_id() == 31) scratch[d >> 5] = inc;
  }
  __syncthreads();
  if (digit_thread) {
    uint32_t run = inc - total;
    for (uint32_t w = 0; w < (d >> 5); ++w) run += scratch[w];
#pragma unroll 8
    for (uint32_t k = 0; k < n_chunks; ++k) {
      const uint32_t v = __ldcg(chunk_base + (uint64_t)k * kRadix + d);
      __stcg(chunk_base + (uint64_t)k * kRadix + d, run);
      run += v;
    }
  }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) atomicExch(ready_flag, 1u);
}

template <bool ATOMIC_RANK>
__global__ void __launch_bounds__(kBsThreads, kBsCtas) bucket_sort_kernel(const __grid_constant__ BucketSortParams p) {
  using Smem = ScatterSmem<kBsWarps, kBsItems, false>;
  constexpr uint32_t kTile = Smem::kTile;
  static_assert(kTile == kBsTile && kSegChunkTiles * kRadix * 4 <= sizeof(Smem::recs), "the count histograms live in the record staging");
  constexpr uint32_t kNone = 0xffffffffu;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);
  __shared__ ScatterParams sp;
  // the item being worked on and the one claimed ahead of it: segment (0 count 1, 1 scatter 1, 2 count 2, 3 scatter 2; kNone = no
  // more work), bucket, index in the segment, whether everything it waits for had happened when it was claimed
  __shared__ uint32_t items[2][4];
  __shared__ uint32_t scratch[16];
  __shared__ uint32_t s_bsize[kRadix], s_round_first[kRadix + 4];  // the tables thread 0 walks for every item (nb <= 256)
  for (uint32_t i = threadIdx.x; i < p.nb; i += kBsThreads) s_bsize[i] = __ldg(p.bsize + i);
  for (uint32_t i = threadIdx.x; i < p.nb + 4; i += kBsThreads) s_round_first[i] = __ldg(p.round_first + i);
  __syncthreads();
  // thread 0 only
  uint32_t round = 0;            // tickets only grow
  uint32_t* pending = nullptr;   // counter of finished tiles to bump for the previous scatter item, once its stores are done

  auto tiles_of = [&](uint32_t b) { return (s_bsize[b] + kTile - 1) / kTile; };
  // what an item waits for: always items with smaller tickets
  auto deps = [&](uint32_t seg, uint32_t b, bool block) -> bool {
    uint32_t* sy = p.sync + (uint64_t)b * kBsSyncWords;
    const uint32_t* addr[2];
    uint32_t want[2], k = 0;
    if (b >= (uint32_t)kBsSlots && seg <= 1) {
      // the bucket that had this slot: its scatter 1 is done with the pass-1 offsets, its scatter 2 with the records
      const uint32_t pb = b - kBsSlots;
      addr[k] = p.sync + (uint64_t)pb * kBsSyncWords + (seg == 0 ? kBsTiles1 : kBsTiles2);
      want[k++] = tiles_of(pb);
    }
    if (seg == 1) addr[k] = sy + kBsReady1, want[k++] = 1u;
    if (seg == 2) addr[k] = sy + kBsTiles1, want[k++] = tiles_of(b);
    if (seg == 3) addr[k] = sy + kBsReady2, want[k++] = 1u;
    if (block) {
      for (uint32_t i = 0; i < k; ++i) wait_at_least(addr[i], want[i]);
    } else {
      uint32_t have[2] = {0xffffffffu, 0xffffffffu};  // both loads in flight together
      for (uint32_t i = 0; i < k; ++i) have[i] = ld_acquire_u32(addr[i]);
      for (uint32_t i = 0; i < k; ++i)
        if (have[i] < want[i]) return false;
    }
    return true;
  };
  auto flush = [&]() {  // the stores of the previous item happen before the loop-top barrier this thread has passed since
    if (pending) {
      __threadfence();
      atomicAdd(pending, 1u);
      pending = nullptr;
    }
  };
  // claiming an item: the ticket is taken early (one atomic round trip), decoded and checked for what it waits for later
  auto decode = [&](uint32_t t, uint32_t* it) {
    if (t >= p.n_items) {
      it[0] = kNone;
      return;
    }
    while (t >= s_round_first[round + 1]) ++round;
    uint32_t o = t - s_round_first[round], seg = 0, b = 0;
    for (; seg < 4; ++seg) {
      if (round < seg || round - seg >= p.nb) continue;
      b = round - seg;
      const uint32_t tiles = tiles_of(b);
      const uint32_t cnt = (seg & 1) ? tiles : (tiles + kSegChunkTiles - 1) / kSegChunkTiles;
      if (o < cnt) break;
      o -= cnt;
    }
    it[0] = seg;
    it[1] = b;
    it[2] = o;
    it[3] = deps(seg, b, false) ? 1u : 0u;
  };

  unsigned long long pf[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  const long long t_start = clock64();
  if (threadIdx.x == 0) decode(atomicAdd(p.ticket, 1u), items[0]);
  for (uint32_t iter = 0;; ++iter) {
    __syncthreads();  // the previous item is done with the shared memory; this item's description is there
    const uint32_t* it = items[iter & 1];
    uint32_t* next = items[(iter + 1) & 1];
    const uint32_t seg = it[0];
    if (seg == kNone) break;
    const uint32_t b = it[1], idx = it[2], slot = b % kBsSlots;
    uint32_t* sy = p.sync + (uint64_t)b * kBsSyncWords;
    if (threadIdx.x == 0) {
      if (!it[3]) {  // something it needs is not there yet: never wait while holding back a signal of one's own
        const long long t0 = clock64();
        flush();
        deps(seg, b, true);
        pf[0] += clock64() - t0;
        pf[5] += 1;
      }
      if (seg & 1) {
        const uint32_t ps = seg >> 1, start = __ldg(p.bstart + b);
        sp.delay_bits = p.delay_bits;
        sp.n = s_bsize[b];
        sp.recs_in = ps == 0 ? p.recs + start : p.slot[slot];
        sp.recs_out = p.slot[slot];
        sp.dig_out = p.slot_dig[slot];
        sp.out_src = p.out_src + start;
        sp.out_tgt = p.out_tgt + start;
        sp.out_w = p.out_w + start;
        sp.out_d = p.out_d + start;
        sp.out_perm = p.out_perm + start;
        sp.shift = p.shift[ps];
        sp.bits = p.bits[ps];
        sp.next_shift = p.shift[1];
        sp.next_bits = p.bits[1];
        sp.key_base = __ldg(p.bkey + b);
        sp.counts = p.counts[ps][slot];
        sp.chunk_base = p.chunk_base[ps][slot];
      }
    }
    __syncthreads();
    // the next item's ticket: asked for now, looked at in the hook
    uint32_t next_ticket = 0;
    if (threadIdx.x == 0) next_ticket = atomicAdd(p.ticket, 1u);
    // between the ranking and the stores of this item (this thread's loads are back, so the fence costs nothing): signal the
    // previous item, whose stores were issued a whole tile ago, and work out the next one
    auto hook = [&]() {
      if (threadIdx.x == 0) {
        flush();
        decode(next_ticket, next);
      }
    };
    const long long t_item = clock64();
    if (seg == 1) {
      scatter_tile<false, false, kBsWarps, kBsItems, kMatchBallot, 2, true, decltype(hook), ATOMIC_RANK>(sp, idx, sm, hook);
      pf[1] += clock64() - t_item;
    } else if (seg == 3) {
      scatter_tile<false, true, kBsWarps, kBsItems, kMatchBallot, 3, true, decltype(hook), ATOMIC_RANK>(sp, idx, sm, hook);
      pf[2] += clock64() - t_item;
    } else {
      hook();
      const uint32_t ps = seg >> 1, n = s_bsize[b];
      const uint32_t tiles = (n + kTile - 1) / kTile, chunks = (tiles + kSegChunkTiles - 1) / kSegChunkTiles;
      const uint8_t* dig = ps == 0 ? p.dig + __ldg(p.bstart + b) : p.slot_dig[slot];
      bucket_count_chunk(dig, n, idx, chunks, p.counts[ps][slot], p.chunk_base[ps][slot], sy + (ps == 0 ? kBsCount1 : kBsCount2),
                         sy + (ps == 0 ? kBsReady1 : kBsReady2), reinterpret_cast<uint32_t*>(sm.recs), scratch);
      pf[3] += clock64() - t_item;
      pf[6] += 1;
      continue;
    }
    pf[4] += 1;
    if (threadIdx.x == 0) pending = sy + (seg == 1 ? kBsTiles1 : kBsTiles2);
  }
  if (threadIdx.x == 0) {
    flush();
    if (p.prof) {
      pf[7] = clock64() - t_start;
      for (int k = 0; k < 8; ++k) p.prof[(uint64_t)blockIdx.x * 8 + k] = pf[k];
    }
  }
}

}  // namespace nc
