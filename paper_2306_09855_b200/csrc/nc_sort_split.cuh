// nc_sort_split.cuh -- stable LSD radix sort that carries the whole connection, digit passes WITHOUT any
// communication between the CTAs of a pass (steps a9-a11 of DESIGN.md; the default organisation path for keys
// of <= 32 bits).
//
// connections are sorted "using two sorting keys: the index of the source node as the first key
// and the delay as the second"; reading D10: ties keep creation order, so every step here is stable.
//
// Per digit pass (reduce - scan - scatter):
//   tile_count_*   : digit histogram of every tile of kTile consecutive records       -> counts[tile][256] (u16)
//                    first pass : digits come from (source, delay) in the storage blocks (6 B / connection)
//                    later      : digits come from the 1-byte-per-record side array the previous scatter wrote
//   chunk_total / chunk_scan / tile_offsets : exclusive scan of the counts in (digit, tile) order
//                                                                                     -> offs[tile][256]  (u32)
//   scatter_pass   : a tile is ranked in shared memory (per-warp digit counters + warp match), its records are
//                    staged in shared memory in tile-sorted order and written out as per-digit runs of
//                    consecutive 16-byte records, starting at offs[tile][digit]; it also writes the next
//                    pass's digit of every record to the side array.
// Record = (key, creation position, target, weight) = one uint4, key = (source << delay_bits) | delay.  The
// first pass builds records from the SoA storage blocks, the last pass writes the final SoA arrays (source and
// delay unpacked from the key, target, weight, permutation): there is no gather by the permutation, every byte
// the organisation step moves is streamed.
//
// Why not the single-pass ("onesweep") chaining of nc_sort.cuh: measured on B200 (profiles/README.md), the
// scatter kernel alone moves a 2.99e8-record pass in 2.0 ms; every variant that chains tile prefixes inside the
// pass (decoupled look-back by 256 threads, by a dedicated warp, or by scanner CTAs) cost 2.6 - 2.9 ms because
// ~450 tiles are in flight and each needs the counts of all tiles before it within a few L2 round trips.  The
// count + scan kernels cost 0.1 ms per pass and read 1 extra byte per record.
#pragma once

#include "nc_common.cuh"
#include "nc_sort.cuh"

namespace nc {

// ---------------------------------------------------------------------------------------------
// Per-tile digit counts.
// ---------------------------------------------------------------------------------------------
constexpr int kCountThreads = 256;

// First pass: digits of key = (source << delay_bits) | delay straight from the storage blocks.
template <bool VEC>
__global__ void __launch_bounds__(kCountThreads) tile_count_first_kernel(const __grid_constant__ BlockMap map, uint32_t n,
                                                                        uint32_t tile_size, uint32_t delay_bits,
                                                                        uint32_t shift, uint32_t bits,
                                                                        uint16_t* __restrict__ counts) {
  __shared__ uint32_t hist[kRadix];
  hist[threadIdx.x] = 0;
  __syncthreads();
  const uint32_t mask = (1u << bits) - 1u;
  const uint64_t tile0 = (uint64_t)blockIdx.x * tile_size;
  const uint32_t valid = (uint32_t)min((uint64_t)tile_size, (uint64_t)n - tile0);
  if (VEC) {
    // B % 4 == 0 and tile_size % 4 == 0: a 4-aligned group of positions sits in one block, 16-byte aligned
    for (uint32_t e = threadIdx.x * 4; e < valid; e += kCountThreads * 4) {
      const uint64_t pos = tile0 + e;
      if (e + 3 < valid) {
        const BlockAddr a = locate(map, pos);
        const uint4 s4 = *reinterpret_cast<const uint4*>(src_ptr(map, a));
        const uint2 d2 = *reinterpret_cast<const uint2*>(d_ptr(map, a));
        atomicAdd(&hist[(((s4.x << delay_bits) | (d2.x & 0xffffu)) >> shift) & mask], 1u);
        atomicAdd(&hist[(((s4.y << delay_bits) | (d2.x >> 16)) >> shift) & mask], 1u);
        atomicAdd(&hist[(((s4.z << delay_bits) | (d2.y & 0xffffu)) >> shift) & mask], 1u);
        atomicAdd(&hist[(((s4.w << delay_bits) | (d2.y >> 16)) >> shift) & mask], 1u);
      } else {
        for (uint32_t q = e; q < valid; ++q)
          atomicAdd(&hist[(load_key_from_storage<uint32_t>(map, tile0 + q, delay_bits) >> shift) & mask], 1u);
      }
    }
  } else {
    for (uint32_t e = threadIdx.x; e < valid; e += kCountThreads)
      atomicAdd(&hist[(load_key_from_storage<uint32_t>(map, tile0 + e, delay_bits) >> shift) & mask], 1u);
  }
  __syncthreads();
  counts[(uint64_t)blockIdx.x * kRadix + threadIdx.x] = (uint16_t)hist[threadIdx.x];
}

// Later passes: digits come from the side array (one byte per record) written by the previous scatter.
// One CTA counts kCountTilesPerCta consecutive tiles (tile_size % 16 == 0; the arrays are 256-byte aligned).
constexpr int kCountTilesPerCta = 8;

__global__ void __launch_bounds__(kCountThreads) tile_count_bytes_kernel(const uint8_t* __restrict__ dig, uint32_t n,
                                                                        uint32_t tile_size, uint32_t n_tiles,
                                                                        uint16_t* __restrict__ counts,
                                                                        uint32_t tiles_per_cta = kCountTilesPerCta) {
  __shared__ uint32_t hist[kRadix];
  hist[threadIdx.x] = 0;
  __syncthreads();
  for (uint32_t k = 0; k < tiles_per_cta; ++k) {
    const uint32_t tile = blockIdx.x * tiles_per_cta + k;
    if (tile >= n_tiles) break;
    const uint64_t tile0 = (uint64_t)tile * tile_size;
    const uint32_t valid = (uint32_t)min((uint64_t)tile_size, (uint64_t)n - tile0);
    for (uint32_t e = threadIdx.x * 16; e < valid; e += kCountThreads * 16) {
      if (e + 15 < valid) {
        const uint4 v = *reinterpret_cast<const uint4*>(dig + tile0 + e);
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          atomicAdd(&hist[w[j] & 0xffu], 1u);
          atomicAdd(&hist[(w[j] >> 8) & 0xffu], 1u);
          atomicAdd(&hist[(w[j] >> 16) & 0xffu], 1u);
          atomicAdd(&hist[w[j] >> 24], 1u);
        }
      } else {
        for (uint32_t q = e; q < valid; ++q) atomicAdd(&hist[dig[tile0 + q]], 1u);
      }
    }
    __syncthreads();
    counts[(uint64_t)tile * kRadix + threadIdx.x] = (uint16_t)hist[threadIdx.x];
    hist[threadIdx.x] = 0;
    __syncthreads();
  }
}

// ---------------------------------------------------------------------------------------------
// Exclusive scan of counts[tile][digit] in (digit, tile) order -> offs[tile][digit] = first output position
// of the tile's run of that digit.  Tiles are grouped into chunks of kScanChunkTiles; thread = digit.
// ---------------------------------------------------------------------------------------------
constexpr uint32_t kScanChunkTiles = 128;  // default; a block-sized sort (nc_copass.cuh) uses shorter chunks

__global__ void __launch_bounds__(kRadix) chunk_total_kernel(const uint16_t* __restrict__ counts, uint32_t n_tiles,
                                                            uint32_t* __restrict__ chunk_tot,
                                                            uint32_t chunk_tiles = kScanChunkTiles) {
  const uint32_t t0 = blockIdx.x * chunk_tiles;
  const uint32_t t1 = min(t0 + chunk_tiles, n_tiles);
  uint32_t s = 0;
#pragma unroll 8
  for (uint32_t t = t0; t < t1; ++t) s += counts[(uint64_t)t * kRadix + threadIdx.x];
  chunk_tot[(uint64_t)blockIdx.x * kRadix + threadIdx.x] = s;
}

// one CTA of kChunkScanSegs x 256 threads: thread (seg, digit) owns a contiguous segment of the chunks.  Digit
// totals -> exclusive scan over the digits (first output position of each digit), then the running start of
// every chunk, in place (chunk_tot becomes chunk_base).
constexpr int kChunkScanSegs = 4;

__global__ void __launch_bounds__(kRadix * kChunkScanSegs) chunk_scan_kernel(uint32_t* __restrict__ chunk_tot,
                                                                             uint32_t n_chunks) {
  __shared__ uint32_t seg_tot[kChunkScanSegs][kRadix];
  __shared__ uint32_t warp_tot[kRadix / 32];
  const uint32_t d = threadIdx.x & (kRadix - 1), seg = threadIdx.x / kRadix;
  const uint32_t per_seg = (n_chunks + kChunkScanSegs - 1) / kChunkScanSegs;
  const uint32_t c0 = min(seg * per_seg, n_chunks), c1 = min(c0 + per_seg, n_chunks);
  uint32_t total = 0;
#pragma unroll 8
  for (uint32_t c = c0; c < c1; ++c) total += chunk_tot[(uint64_t)c * kRadix + d];
  seg_tot[seg][d] = total;
  __syncthreads();
  uint32_t digit_total = 0, before = 0;  // over all segments / over the segments below mine
#pragma unroll
  for (int g = 0; g < kChunkScanSegs; ++g) {
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
  for (uint32_t c = c0; c < c1; ++c) {
    const uint32_t v = chunk_tot[(uint64_t)c * kRadix + d];
    chunk_tot[(uint64_t)c * kRadix + d] = run;
    run += v;
  }
}

__global__ void __launch_bounds__(kRadix) tile_offsets_kernel(const uint16_t* __restrict__ counts, uint32_t n_tiles,
                                                             const uint32_t* __restrict__ chunk_base,
                                                             uint32_t* __restrict__ offs,
                                                             uint32_t chunk_tiles = kScanChunkTiles) {
  const uint32_t t0 = blockIdx.x * chunk_tiles;
  const uint32_t t1 = min(t0 + chunk_tiles, n_tiles);
  uint32_t run = chunk_base[(uint64_t)blockIdx.x * kRadix + threadIdx.x];
#pragma unroll 8
  for (uint32_t t = t0; t < t1; ++t) {
    const uint32_t c = counts[(uint64_t)t * kRadix + threadIdx.x];
    offs[(uint64_t)t * kRadix + threadIdx.x] = run;
    run += c;
  }
}

// ---------------------------------------------------------------------------------------------
// Scatter pass.
// ---------------------------------------------------------------------------------------------
struct ScatterParams {
  BlockMap map;  // FIRST: records are built from the storage blocks
  uint32_t delay_bits;
  uint32_t n;
  uint32_t pos_base;  // FIRST: creation position of the first record (0 unless one storage block is sorted on its own)
  const uint4* recs_in;
  uint4* recs_out;
  uint8_t* dig_out;  // !LAST: digit of the NEXT pass for every record written
  uint32_t* out_src;  // LAST: final arrays
  uint32_t* out_tgt;
  float* out_w;
  uint16_t* out_d;
  uint32_t* out_perm;
  uint32_t shift, bits;            // this pass's digit
  uint32_t next_shift, next_bits;  // the next pass's digit
  const uint32_t* offs;            // [n_tiles][256]
  // bucket-first organisation (nc_sort_msd.cuh; MODE != 0 of scatter_pass_kernel)
  uint32_t msd_mul;                // MODE 1: bucket of a key = min(umulhi(source, msd_mul), 255)
  const uint32_t* key_base_tab;    // MODE 1: [256] smallest key of every bucket (the next pass's digits are relative to it)
  uint32_t key_base;               // MODE 2, 3: smallest key of the bucket this launch sorts; digits are those of key - key_base
  const uint16_t* counts;          // MODE 2, 3: [n_tiles][256] digit counts of the tiles and
  const uint32_t* chunk_base;      //            [n_chunks][256] first output position of every chunk of kSegChunkTiles tiles
};

// MODE of scatter_pass_kernel: 0 = a digit pass over the whole array (offsets from the scan kernels);
// 1 = the bucket pass of nc_sort_msd.cuh (digit = bucket of the source); 2 / 3 = a digit pass inside ONE bucket whose records
// come from HBM / from an L2-resident slot (offsets from chunk bases + the counts of the tiles before it in its chunk; L2
// eviction-priority hints on the loads and stores).
constexpr uint32_t kSegChunkTiles = 8;

template <int MODE>
__device__ __forceinline__ uint32_t pass_digit(uint32_t key, const ScatterParams& p, uint32_t mask) {
  if (MODE == 1) return min(__umulhi(key >> p.delay_bits, p.msd_mul), (uint32_t)kRadix - 1u);
  if (MODE >= 2) return ((key - p.key_base) >> p.shift) & mask;
  return (key >> p.shift) & mask;
}

// L2 eviction-priority hints (H: 0 none, 1 evict_first, 2 evict_last)
template <int H>
__device__ __forceinline__ uint64_t l2_policy() {
  uint64_t pol = 0;
  if (H == 1) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  if (H == 2) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
template <int H, bool PAST_L1 = false>
__device__ __forceinline__ uint4 ld_hint(const uint4* q, uint64_t pol) {
  if (H == 0) return PAST_L1 ? __ldcg(q) : *q;
  uint4 r;
  if (PAST_L1)
    asm volatile("ld.global.cg.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(q), "l"(pol));
  else
    asm volatile("ld.global.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(q), "l"(pol));
  return r;
}
template <int H>
__device__ __forceinline__ void st_hint(uint4* q, const uint4& v, uint64_t pol) {
  if (H == 0) *q = v;
  else asm volatile("st.global.L2::cache_hint.v4.b32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(q), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "l"(pol) : "memory");
}
template <int H>
__device__ __forceinline__ void st_hint(uint32_t* q, uint32_t v, uint64_t pol) {
  if (H == 0) *q = v;
  else asm volatile("st.global.L2::cache_hint.b32 [%0], %1, %2;" ::"l"(q), "r"(v), "l"(pol) : "memory");
}
template <int H>
__device__ __forceinline__ void st_hint(uint16_t* q, uint16_t v, uint64_t pol) {
  if (H == 0) *q = v;
  else asm volatile("st.global.L2::cache_hint.b16 [%0], %1, %2;" ::"l"(q), "h"(v), "l"(pol) : "memory");
}
template <int H>
__device__ __forceinline__ void st_hint(uint8_t* q, uint8_t v, uint64_t pol) {
  if (H == 0) *q = v;
  else asm volatile("st.global.L2::cache_hint.b8 [%0], %1, %2;" ::"l"(q), "r"((uint32_t)v), "l"(pol) : "memory");
}

template <int WARPS, int ITEMS, bool SMEM_MATCH>
struct ScatterSmem {
  static constexpr int kTile = WARPS * 32 * ITEMS;
  uint4 recs[kTile];
  uint32_t warp_hist[WARPS][kRadix];  // per-warp digit counts, then the warp's running tile position per digit
  uint32_t warp_masks[SMEM_MATCH ? WARPS : 1][kRadix];  // kMatchSmem: peer-mask words (zero between uses)
  uint32_t global_off[kRadix];  // (first output position of the tile's run of the digit) - (its start in the tile)
  uint32_t scan_tmp[kRadix / 32];
};

// One tile of a pass.  COHERENT (in-bucket passes run by the persistent kernel of nc_sort_msd.cuh): what other CTAs of the SAME
// launch wrote -- the offsets and, in MODE 3, the records -- is read past the L1.
struct NoHook {
  __device__ __forceinline__ void operator()() const {}
};

// ATOMIC_RANK: a record's place among the equal digits of its warp comes from ONE returning shared atomicAdd per record instead
// of eight ballots + a leader's atomic + a shuffle; rests on the lanes of one atomic instruction being served in ascending lane
// order (nc_sort_bulk.cuh, atomic_lane_order_kernel), so only where the context has checked that.
template <bool FIRST, bool LAST, int WARPS, int ITEMS, int MATCH, int MODE, bool COHERENT, typename Hook = NoHook,
          bool ATOMIC_RANK = false>
__device__ __forceinline__ void scatter_tile(const ScatterParams& p, const uint32_t tile,
                                             ScatterSmem<WARPS, ITEMS, MATCH == kMatchSmem>& sm, Hook late_hook = Hook()) {
  using Smem = ScatterSmem<WARPS, ITEMS, MATCH == kMatchSmem>;
  static_assert(MODE == 0 || (MODE == 1 && FIRST && !LAST) || (MODE >= 2 && !FIRST), "bucket pass: from the blocks; in-bucket: records");
  // in-bucket passes: what comes from HBM is read once (evict_first), what goes to the slot the next pass reads stays
  // (evict_last), the final arrays are not read again by this step (evict_first)
  constexpr int kLoadHint = MODE == 2 ? 1 : MODE == 3 ? 2 : 0;
  constexpr int kStoreHint = MODE >= 2 ? (LAST ? 1 : 2) : 0;
  const uint64_t lpol = l2_policy<kLoadHint>(), spol = l2_policy<kStoreHint>();
  const uint32_t pad_key = MODE >= 2 ? p.key_base - 1u : 0xffffffffu;  // its digits are the largest of every pass
  constexpr int kThreads = WARPS * 32;
  constexpr int kTile = Smem::kTile;
  static_assert(kThreads >= kRadix, "one thread per digit is needed for the in-tile scan");

  const uint32_t warp = threadIdx.x >> 5, lane = lane_id();
  {
    constexpr int kZero = (MATCH == kMatchSmem ? 2 : 1) * WARPS * kRadix / 4;  // warp_hist (+ warp_masks)
    uint4* z = reinterpret_cast<uint4*>(&sm.warp_hist[0][0]);
    for (int i = threadIdx.x; i < kZero; i += kThreads) z[i] = make_uint4(0u, 0u, 0u, 0u);
  }
  const uint64_t tile0 = (uint64_t)tile * kTile;
  const uint32_t valid = (uint32_t)min((uint64_t)kTile, (uint64_t)p.n - tile0);
  const uint32_t mask = (1u << p.bits) - 1u;
  // first output position of this tile's run of digit threadIdx.x: fetched now, needed after the histogram
  uint32_t out0 = 0u;
  if (threadIdx.x < kRadix) {
    if (MODE >= 2) {
      const uint32_t chunk = tile / kSegChunkTiles, k = tile % kSegChunkTiles;
      const uint32_t* bp = p.chunk_base + (uint64_t)chunk * kRadix + threadIdx.x;
      out0 = COHERENT ? __ldcg(bp) : __ldg(bp);
      const uint16_t* cp = p.counts + (uint64_t)chunk * kSegChunkTiles * kRadix + threadIdx.x;
#pragma unroll
      for (uint32_t kk = 0; kk + 1 < kSegChunkTiles; ++kk)
        if (kk < k) out0 += COHERENT ? __ldcg(cp + kk * kRadix) : __ldg(cp + kk * kRadix);
    } else {
      out0 = __ldg(p.offs + (uint64_t)tile * kRadix + threadIdx.x);
    }
  }

  // ---- load records, warp-striped: element (warp, i, lane) is tile position warp*ITEMS*32 + i*32 + lane ----
  uint4 rec[ITEMS];
  const uint32_t wbase = warp * (ITEMS * 32) + lane;
  uint32_t* my_hist = sm.warp_hist[warp];
  if (FIRST) {
    // records are built from the SoA storage blocks; when the whole tile sits in one block (the common case)
    // the block is located once per tile instead of once per record
    const BlockAddr a0 = locate(p.map, tile0);
    const bool one_block = a0.slot + kTile <= p.map.B;
    if (one_block && valid == kTile) {
      const uint32_t* sp = reinterpret_cast<const uint32_t*>(a0.base) + a0.slot + wbase;
      const uint32_t* tp = reinterpret_cast<const uint32_t*>(a0.base + p.map.off_tgt) + a0.slot + wbase;
      const uint32_t* wp = reinterpret_cast<const uint32_t*>(a0.base + p.map.off_w) + a0.slot + wbase;
      const uint16_t* dp = reinterpret_cast<const uint16_t*>(a0.base + p.map.off_d) + a0.slot + wbase;
      uint32_t s[ITEMS], d[ITEMS];
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) {
        s[i] = sp[i * 32];
        d[i] = dp[i * 32];
        rec[i].z = tp[i * 32];
        rec[i].w = wp[i * 32];
      }
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) {
        rec[i].x = (s[i] << p.delay_bits) | d[i];
        rec[i].y = p.pos_base + (uint32_t)(tile0 + wbase + i * 32);
      }
    } else {
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) {
        const uint32_t e = wbase + i * 32;
        if (e < valid) {
          const BlockAddr a = locate(p.map, tile0 + e);
          const uint32_t s = *src_ptr(p.map, a);
          const uint32_t d = *d_ptr(p.map, a);
          rec[i] = make_uint4((s << p.delay_bits) | d, p.pos_base + (uint32_t)(tile0 + e), *tgt_ptr(p.map, a),
                              __float_as_uint(*w_ptr(p.map, a)));
        } else {
          rec[i] = make_uint4(0xffffffffu, 0u, 0u, 0u);
        }
      }
    }
  } else {
    const uint4* in = p.recs_in + tile0 + wbase;
    if (valid == kTile) {
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) rec[i] = ld_hint<kLoadHint, COHERENT && MODE == 3>(in + i * 32, lpol);
    } else {
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) {
        // padding sorts behind every real record of the tile and is never written out
        rec[i] = wbase + i * 32 < valid ? ld_hint<kLoadHint, COHERENT && MODE == 3>(in + i * 32, lpol) : make_uint4(pad_key, 0u, 0u, 0u);
      }
    }
  }
  __syncthreads();  // the counters are zero
  // ---- per-warp digit histogram with fire-and-forget shared-memory atomics ----
#pragma unroll
  for (int i = 0; i < ITEMS; ++i) atomicAdd(&my_hist[pass_digit<MODE>(rec[i].x, p, mask)], 1u);
  __syncthreads();

  // ---- per digit: exclusive scan over the warps; exclusive scan over the digits -> where each digit's run
  //      starts inside the tile; where it starts in the output comes from the scan kernels ----
  if (threadIdx.x < kRadix) {
    const uint32_t d = threadIdx.x;
    uint32_t cnt[WARPS];
#pragma unroll
    for (int w = 0; w < WARPS; ++w) cnt[w] = sm.warp_hist[w][d];
    uint32_t run = 0;
#pragma unroll
    for (int w = 0; w < WARPS; ++w) {
      const uint32_t c = cnt[w];
      cnt[w] = run;
      run += c;
    }
    uint32_t inc = run;
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, s);
      if (lane >= (uint32_t)s) inc += t;
    }
    if (lane == 31) sm.scan_tmp[warp] = inc;
    asm volatile("bar.sync 1, %0;" ::"n"(kRadix));
    uint32_t base = 0;
#pragma unroll
    for (uint32_t w = 0; w < kRadix / 32; ++w) base += w < warp ? sm.scan_tmp[w] : 0u;
    const uint32_t my_excl = base + inc - run;
    sm.global_off[d] = out0 - my_excl;
#pragma unroll
    for (int w = 0; w < WARPS; ++w) sm.warp_hist[w][d] = my_excl + cnt[w];  // tile position of the warp's first
  }
  __syncthreads();

  // ---- stable rank + scatter into shared memory in one go: the lowest lane of each group of equal digits
  //      bumps the warp's running offset for that digit (atomics of one warp to one address retire in
  //      program order, so items keep their position order) and the group shares the old value ----
  if (ATOMIC_RANK) {
    uint32_t at[ITEMS];
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) at[i] = atomicAdd(&my_hist[pass_digit<MODE>(rec[i].x, p, mask)], 1u);
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) sm.recs[at[i]] = rec[i];
  } else {
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
      const uint32_t d = pass_digit<MODE>(rec[i].x, p, mask);
      const uint32_t peers = peers_of<MATCH>(d, sm.warp_masks[MATCH == kMatchSmem ? warp : 0]);
      const uint32_t below = __popc(peers & lanemask_lt());
      uint32_t old = 0;
      if (below == 0) old = atomicAdd(&my_hist[d], (uint32_t)__popc(peers));
      old = __shfl_sync(0xffffffffu, old, __ffs(peers) - 1);
      sm.recs[old + below] = rec[i];
    }
  }

  if (LAST) {
    __syncthreads();
    late_hook();  // (persistent kernel: bookkeeping of one thread; its loads have returned, the stores are not issued yet)
    // ---- final arrays: consecutive threads write consecutive records of a digit run ----
    const uint32_t dmask = (1u << p.delay_bits) - 1u;
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
      const uint32_t j = i * kThreads + threadIdx.x;
      if (j < valid) {
        const uint4 r = sm.recs[j];
        const uint32_t g = sm.global_off[pass_digit<MODE>(r.x, p, mask)] + j;
        st_hint<kStoreHint>(p.out_src + g, r.x >> p.delay_bits, spol);
        st_hint<kStoreHint>(p.out_d + g, (uint16_t)(r.x & dmask), spol);
        st_hint<kStoreHint>(p.out_tgt + g, r.z, spol);
        st_hint<kStoreHint>(reinterpret_cast<uint32_t*>(p.out_w) + g, r.w, spol);
        st_hint<kStoreHint>(p.out_perm + g, r.y, spol);
      }
    }
  } else {
    __syncthreads();
    late_hook();
    // ---- records and the next pass's digit of each: consecutive threads write consecutive records of a run.
    //      (One TMA bulk copy per run was measured slower: the 32 copies a warp issues are serialised.) ----
    const uint32_t next_mask = (1u << p.next_bits) - 1u;
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
      const uint32_t j = i * kThreads + threadIdx.x;
      if (j < valid) {
        const uint4 r = sm.recs[j];
        const uint32_t d = pass_digit<MODE>(r.x, p, mask);
        const uint32_t g = sm.global_off[d] + j;
        st_hint<kStoreHint>(p.recs_out + g, r, spol);
        // the next pass's digit: of the key itself, or (bucket-first organisation) of the key relative to its bucket's first
        const uint32_t rel = MODE == 1 ? r.x - __ldg(p.key_base_tab + d) : MODE >= 2 ? r.x - p.key_base : r.x;
        st_hint<kStoreHint>(p.dig_out + g, (uint8_t)((rel >> p.next_shift) & next_mask), spol);
      }
    }
  }
}

template <bool FIRST, bool LAST, int WARPS, int ITEMS, int MIN_CTAS, int MATCH, int MODE = 0>
__global__ void __launch_bounds__(WARPS * 32, MIN_CTAS) scatter_pass_kernel(const __grid_constant__ ScatterParams p) {
  using Smem = ScatterSmem<WARPS, ITEMS, MATCH == kMatchSmem>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  scatter_tile<FIRST, LAST, WARPS, ITEMS, MATCH, MODE, false>(p, blockIdx.x, *reinterpret_cast<Smem*>(smem_raw));
}

}  // namespace nc
