// nc_sort.cuh -- stable LSD radix sort of all connections by the packed (source, delay) key
// (steps a9-a11 of DESIGN.md; "hierarchically using two sorting keys: the index of the
// source node as the first key and the delay as the second"; reading D10: ties keep creation order).
//
//   key  = (source << delay_bits) | delay          payload = creation position (u32)
//   histogram_kernel : one read of (source, delay) from the storage blocks -> P digit histograms
//   onesweep_kernel  : one pass per digit: a tile is ranked in shared memory (warp match), its digit
//                      counts are chained to the previous tiles by decoupled look-back (Merrill & Garland
//                      style single-pass scan, one 64-bit status word per (tile, digit)), and keys +
//                      payload are written out as per-digit runs staged through shared memory
//   permute_kernel   : sorted target/weight gathered by the permutation; source/delay unpacked from the key
#pragma once

#include "nc_common.cuh"

namespace nc {

constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;
constexpr int kMaxPasses = 6;  // 48-bit keys: 32-bit source + 16-bit delay

struct PassPlan {
  uint32_t n_passes;
  uint32_t shift[kMaxPasses];
  uint32_t bits[kMaxPasses];
};

template <typename KeyT>
__device__ __forceinline__ uint32_t digit_of(KeyT key, uint32_t shift, uint32_t mask) {
  return (uint32_t)(key >> shift) & mask;
}

template <typename KeyT>
__device__ __forceinline__ KeyT load_key_from_storage(const BlockMap& map, uint64_t pos, uint32_t delay_bits) {
  const BlockAddr a = locate(map, pos);
  const uint32_t s = *src_ptr(map, a);
  const uint32_t d = *d_ptr(map, a);
  return ((KeyT)s << delay_bits) | (KeyT)d;
}

// ---------------------------------------------------------------------------------------------
// Digit histograms of all passes in one read of the keys.
// ---------------------------------------------------------------------------------------------
constexpr int kHistThreads = 512;
constexpr int kHistItems = 16;

template <typename KeyT, bool VEC>
__global__ void __launch_bounds__(kHistThreads) histogram_kernel(const __grid_constant__ BlockMap map, uint32_t n,
                                                                uint32_t delay_bits,
                                                                const __grid_constant__ PassPlan plan,
                                                                uint32_t* __restrict__ ghist /* [P][256] */) {
  __shared__ uint32_t hist[kMaxPasses][kRadix];
  for (int i = threadIdx.x; i < kMaxPasses * kRadix; i += kHistThreads) (&hist[0][0])[i] = 0;
  __syncthreads();
  uint32_t shift[kMaxPasses], dmask[kMaxPasses];
#pragma unroll
  for (int ps = 0; ps < kMaxPasses; ++ps) {
    shift[ps] = plan.shift[ps];
    dmask[ps] = (1u << plan.bits[ps]) - 1u;
  }
  const uint32_t n_passes = plan.n_passes;
  auto count = [&](KeyT key) {
#pragma unroll
    for (int ps = 0; ps < kMaxPasses; ++ps) {
      if ((uint32_t)ps < n_passes) atomicAdd(&hist[ps][digit_of(key, shift[ps], dmask[ps])], 1u);
    }
  };
  const uint64_t tile0 = (uint64_t)blockIdx.x * (kHistThreads * kHistItems);
  if (VEC) {
    // B % 4 == 0: a 4-aligned group of positions sits in one block, 16-byte aligned -> 128/64-bit loads
#pragma unroll
    for (int g = 0; g < kHistItems / 4; ++g) {
      const uint64_t pos = tile0 + ((uint64_t)g * kHistThreads + threadIdx.x) * 4;
      if (pos + 3 < n) {
        const BlockAddr a = locate(map, pos);
        const uint4 s4 = *reinterpret_cast<const uint4*>(src_ptr(map, a));
        const uint2 d2 = *reinterpret_cast<const uint2*>(d_ptr(map, a));
        count(((KeyT)s4.x << delay_bits) | (KeyT)(d2.x & 0xffffu));
        count(((KeyT)s4.y << delay_bits) | (KeyT)(d2.x >> 16));
        count(((KeyT)s4.z << delay_bits) | (KeyT)(d2.y & 0xffffu));
        count(((KeyT)s4.w << delay_bits) | (KeyT)(d2.y >> 16));
      } else {
        for (uint64_t q = pos; q < n; ++q) count(load_key_from_storage<KeyT>(map, q, delay_bits));
      }
    }
  } else {
#pragma unroll 4
    for (int i = 0; i < kHistItems; ++i) {
      const uint64_t pos = tile0 + (uint64_t)i * kHistThreads + threadIdx.x;
      if (pos < n) count(load_key_from_storage<KeyT>(map, pos, delay_bits));
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < (int)n_passes * kRadix; i += kHistThreads) {
    const uint32_t v = (&hist[0][0])[i];
    if (v) atomicAdd(ghist + i, v);
  }
}

// exclusive scan of each pass's 256 bins -> first output position of every digit
__global__ void __launch_bounds__(kRadix) bin_scan_kernel(const uint32_t* __restrict__ ghist,
                                                         uint32_t* __restrict__ bin_start) {
  __shared__ uint32_t warp_tot[kRadix / 32];
  const uint32_t ps = blockIdx.x;
  const uint32_t v = ghist[ps * kRadix + threadIdx.x];
  uint32_t inc = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
    if (lane_id() >= (uint32_t)d) inc += t;
  }
  if (lane_id() == 31) warp_tot[threadIdx.x >> 5] = inc;
  __syncthreads();
  uint32_t base = 0;
  for (uint32_t w = 0; w < (threadIdx.x >> 5); ++w) base += warp_tot[w];
  bin_start[ps * kRadix + threadIdx.x] = base + inc - v;
}

// ---------------------------------------------------------------------------------------------
// Onesweep digit pass.
// Look-back status word (one per tile and digit, never re-zeroed: the epoch tag tells passes apart):
//   bits  0..39 count | bits 40..41 flag (1 = tile aggregate, 2 = inclusive prefix) | bits 42..63 epoch
// ---------------------------------------------------------------------------------------------
constexpr uint64_t kFlagAggregate = 1ull << 40;
constexpr uint64_t kFlagInclusive = 2ull << 40;
constexpr uint64_t kCountMask = (1ull << 40) - 1;

// Lanes of the warp whose digit equals mine, three ways (measured on B200, cycles per warp-wide call per SM at
// full occupancy: match.any 61.5, eight ballots 25.3, shared-memory atomicOr 7.3 -- profiles/README.md):
//   kMatchAny   : one MATCH.ANY
//   kMatchBallot: one VOTE per digit bit
//   kMatchSmem  : every lane ORs its lane bit into a per-(warp, digit) mask word in shared memory, the warp
//                 reads the word back, the lowest peer clears it for the next item
enum MatchMode : int { kMatchAny = 0, kMatchBallot = 1, kMatchSmem = 2 };

template <int MODE>
__device__ __forceinline__ uint32_t peers_of(uint32_t d, uint32_t* warp_masks /* [256], all zero between calls */) {
  if (MODE == kMatchAny) return __match_any_sync(0xffffffffu, d);
  if (MODE == kMatchBallot) {
    uint32_t peers = 0xffffffffu;
#pragma unroll
    for (int b = 0; b < kRadixBits; ++b) {
      const bool bit = (d >> b) & 1u;
      const uint32_t vote = __ballot_sync(0xffffffffu, bit);
      peers &= bit ? vote : ~vote;
    }
    return peers;
  }
  uint32_t* m = warp_masks + d;
  atomicOr(m, 1u << lane_id());
  __syncwarp();
  const uint32_t peers = *m;
  __syncwarp();
  if ((peers & lanemask_lt()) == 0) *m = 0u;
  __syncwarp();
  return peers;
}

// Decoupled look-back for one digit of one tile: sum the counts of the preceding tiles, walking backwards
// until a tile that already knows its inclusive prefix.  The status words of kLookBatch predecessors are
// fetched with independent loads (they are L2 hits a few hundred cycles away; issuing them one at a time
// made the walk, not the data movement, the critical path of a pass), then consumed in order.
constexpr int kLookBatch = 8;

__device__ __forceinline__ bool status_ready(uint64_t w, uint64_t epoch) {
  return (w & ~(kCountMask | kFlagAggregate | kFlagInclusive)) == epoch && (w & (kFlagAggregate | kFlagInclusive)) != 0;
}

__device__ __forceinline__ uint64_t look_back(const uint64_t* status, uint32_t tile, uint32_t d, uint64_t epoch,
                                              uint32_t* error_flag) {
  uint64_t excl = 0;
  int64_t t = (int64_t)tile - 1;
  uint32_t spins = 0;
  while (t >= 0) {
    uint64_t w[kLookBatch];
#pragma unroll
    for (int k = 0; k < kLookBatch; ++k) {
      const int64_t tk = t - k;
      w[k] = tk >= 0 ? ld_relaxed_u64(status + (uint64_t)tk * kRadix + d) : (epoch | kFlagInclusive);
    }
    bool done = false;
    int used = 0;
#pragma unroll
    for (int k = 0; k < kLookBatch; ++k) {
      if (!done && used == k) {
        if (status_ready(w[k], epoch)) {
          excl += w[k] & kCountMask;
          used = k + 1;
          if (w[k] & kFlagInclusive) done = true;
        }
      }
    }
    if (done) break;
    t -= used;
    if (used == 0) {
      if (++spins > (1u << 22)) {  // seconds: a predecessor is lost -> report instead of hanging the GPU
        *error_flag = 1u;
        break;
      }
      __nanosleep(32);
    }
  }
  return excl;
}

template <typename KeyT>
struct SortPassParams {
  BlockMap map;  // FIRST pass: keys are built from the storage blocks and the payload is the position
  uint32_t delay_bits;
  uint32_t n;
  const KeyT* keys_in;
  const uint32_t* vals_in;
  KeyT* keys_out;
  uint32_t* vals_out;
  uint32_t shift, bits;
  const uint32_t* bin_start;  // [256]
  uint64_t* status;           // [n_tiles][256]
  uint32_t* ticket;
  uint32_t* error_flag;       // set to 1 if a look-back ever gives up (never expected; avoids a device hang)
  uint64_t epoch;             // already shifted to bits 42..63
};

template <typename KeyT, int THREADS, int ITEMS>
struct OnesweepSmem {
  static constexpr int kTile = THREADS * ITEMS;
  static constexpr int kWarps = THREADS / 32;
  KeyT keys[kTile];
  uint32_t vals[kTile];
  uint32_t warp_hist[kWarps][kRadix];
  uint32_t tile_excl[kRadix];   // exclusive scan of the tile's digit counts
  uint32_t global_off[kRadix];  // (global first position of the digit for this tile) - tile_excl[d]
  uint32_t scan_tmp[kRadix / 32];
  uint32_t tile_id;
};

template <typename KeyT, bool FIRST, int THREADS, int ITEMS>
__global__ void __launch_bounds__(THREADS) onesweep_kernel(const __grid_constant__ SortPassParams<KeyT> p) {
  using Smem = OnesweepSmem<KeyT, THREADS, ITEMS>;
  constexpr int kTile = Smem::kTile;
  constexpr int kWarps = Smem::kWarps;
  static_assert(THREADS >= kRadix, "one thread per digit is needed for the look-back");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);

  const uint32_t warp = threadIdx.x >> 5, lane = lane_id();
  // tiles are handed out in launch order so that a tile only ever waits on tiles that already run
  if (threadIdx.x == 0) sm.tile_id = atomicAdd(p.ticket, 1u);
  for (int i = threadIdx.x; i < kWarps * kRadix; i += THREADS) (&sm.warp_hist[0][0])[i] = 0;
  __syncthreads();
  const uint32_t tile = sm.tile_id;
  const uint64_t tile0 = (uint64_t)tile * kTile;
  const uint32_t valid = (uint32_t)min((uint64_t)kTile, (uint64_t)p.n - tile0);
  const uint32_t mask = (1u << p.bits) - 1u;

  // ---- load keys, warp-striped: element (warp, i, lane) is tile position warp*ITEMS*32 + i*32 + lane ----
  KeyT key[ITEMS];
  const uint32_t wbase = warp * (ITEMS * 32) + lane;
#pragma unroll
  for (int i = 0; i < ITEMS; ++i) {
    const uint32_t e = wbase + i * 32;
    if (e < valid) {
      if (FIRST) {
        key[i] = load_key_from_storage<KeyT>(p.map, tile0 + e, p.delay_bits);
      } else {
        key[i] = p.keys_in[tile0 + e];
      }
    } else {
      key[i] = ~(KeyT)0;  // sorts behind every real key of the tile and is never written out
    }
  }

  // ---- stable rank inside the warp: peers with the same digit, counted in position order ----
  uint32_t rank[ITEMS];
  uint32_t* my_hist = sm.warp_hist[warp];
#pragma unroll
  for (int i = 0; i < ITEMS; ++i) {
    const uint32_t d = digit_of(key[i], p.shift, mask);
    const uint32_t peers = __match_any_sync(0xffffffffu, d);
    const uint32_t below = __popc(peers & lanemask_lt());
    uint32_t pre = 0;
    if (below == 0) {  // lowest lane of the peer group owns the counter update
      pre = my_hist[d];
      my_hist[d] = pre + __popc(peers);
    }
    __syncwarp();
    pre = __shfl_sync(0xffffffffu, pre, __ffs(peers) - 1);
    rank[i] = pre + below;
  }
  __syncthreads();

  // ---- per digit: exclusive scan over the warps, tile count, look-back, global offset ----
  uint32_t tile_count = 0;
  if (threadIdx.x < kRadix) {
    const uint32_t d = threadIdx.x;
    uint32_t run = 0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) {
      const uint32_t c = sm.warp_hist[w][d];
      sm.warp_hist[w][d] = run;
      run += c;
    }
    tile_count = run;
    // padding keys of a ragged last tile all carry the largest digit; they are not part of the data
    const uint32_t real = (d == mask) ? run - (kTile - valid) : run;
    uint64_t* my_status = p.status + (uint64_t)tile * kRadix + d;
    uint64_t excl = 0;
    if (tile == 0) {
      st_relaxed_u64(my_status, p.epoch | kFlagInclusive | real);
    } else {
      st_relaxed_u64(my_status, p.epoch | kFlagAggregate | real);
      excl = look_back(p.status, tile, d, p.epoch, p.error_flag);
      st_relaxed_u64(my_status, p.epoch | kFlagInclusive | (excl + real));
    }
    // exclusive scan of tile_count across the 256 digits
    uint32_t inc = tile_count;
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, s);
      if (lane >= (uint32_t)s) inc += t;
    }
    if (lane == 31) sm.scan_tmp[warp] = inc;
    // (the sync below is only among the kRadix/32 warps that hold digits)
    asm volatile("bar.sync 1, %0;" ::"n"(kRadix));
    uint32_t base = 0;
    for (uint32_t w = 0; w < warp; ++w) base += sm.scan_tmp[w];
    const uint32_t te = base + inc - tile_count;
    sm.tile_excl[d] = te;
    sm.global_off[d] = p.bin_start[d] + (uint32_t)excl - te;
  }
  __syncthreads();

  // ---- scatter into shared memory in tile-sorted order ----
#pragma unroll
  for (int i = 0; i < ITEMS; ++i) {
    const uint32_t d = digit_of(key[i], p.shift, mask);
    const uint32_t pos = sm.tile_excl[d] + my_hist[d] + rank[i];
    rank[i] = pos;
    sm.keys[pos] = key[i];
  }
#pragma unroll
  for (int i = 0; i < ITEMS; ++i) {
    const uint32_t e = wbase + i * 32;
    uint32_t v = 0;
    if (e < valid) v = FIRST ? (uint32_t)(tile0 + e) : p.vals_in[tile0 + e];
    sm.vals[rank[i]] = v;
  }
  __syncthreads();

  // ---- write out: consecutive threads write consecutive elements of a digit run ----
#pragma unroll
  for (int i = 0; i < ITEMS; ++i) {
    const uint32_t j = i * THREADS + threadIdx.x;
    if (j < valid) {
      const KeyT k = sm.keys[j];
      const uint32_t g = sm.global_off[digit_of(k, p.shift, mask)] + j;
      p.keys_out[g] = k;
      p.vals_out[g] = sm.vals[j];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Onesweep digit pass that carries the whole connection (32-bit keys only).
//
// Record = (key, creation position, target, weight) = one uint4.  The first pass builds records from the
// storage blocks, middle passes move AoS records (128-bit loads and stores, digit runs of ~16 records =
// 256 contiguous bytes), and the last pass writes the final SoA arrays (source and delay unpacked from the
// key, target, weight, permutation) directly -- so there is no gather by the permutation at all: every byte
// the organisation step moves is streamed.  Same ranking, look-back and status words as onesweep_kernel.
// ---------------------------------------------------------------------------------------------
struct SortRecParams {
  BlockMap map;  // FIRST
  uint32_t delay_bits;
  uint32_t n;
  const uint4* recs_in;
  uint4* recs_out;
  // LAST: final arrays
  uint32_t* out_src;
  uint32_t* out_tgt;
  float* out_w;
  uint16_t* out_d;
  uint32_t* out_perm;
  uint32_t shift, bits;
  const uint32_t* bin_start;
  uint64_t* status;
  uint32_t* ticket;
  uint32_t* error_flag;
  uint64_t epoch;
};

template <int THREADS, int ITEMS>
struct OnesweepRecSmem {
  static constexpr int kTile = THREADS * ITEMS;
  static constexpr int kWarps = THREADS / 32;
  uint4 recs[kTile];
  uint32_t warp_hist[kWarps][kRadix];   // per-warp digit counts, then the warp's running offset per digit
  uint32_t warp_masks[kWarps][kRadix];  // kMatchSmem: peer-mask words (zero between uses)
  uint32_t tile_excl[kRadix];
  uint32_t global_off[kRadix];
  uint32_t scan_tmp[kRadix / 32];
  uint32_t tile_id;
};

template <bool FIRST, bool LAST, int THREADS, int ITEMS, int MIN_CTAS, int MATCH>
__global__ void __launch_bounds__(THREADS, MIN_CTAS) onesweep_rec_kernel(const __grid_constant__ SortRecParams p) {
  using Smem = OnesweepRecSmem<THREADS, ITEMS>;
  constexpr int kTile = Smem::kTile;
  constexpr int kWarps = Smem::kWarps;
  static_assert(THREADS >= kRadix, "one thread per digit is needed for the look-back");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);

  const uint32_t warp = threadIdx.x >> 5, lane = lane_id();
  // tiles are handed out in launch order so that a tile only ever waits on tiles that already run
  if (threadIdx.x == 0) sm.tile_id = atomicAdd(p.ticket, 1u);
  for (int i = threadIdx.x; i < 2 * kWarps * kRadix; i += THREADS) (&sm.warp_hist[0][0])[i] = 0;  // + warp_masks
  __syncthreads();
  const uint32_t tile = sm.tile_id;
  const uint64_t tile0 = (uint64_t)tile * kTile;
  const uint32_t valid = (uint32_t)min((uint64_t)kTile, (uint64_t)p.n - tile0);
  const uint32_t mask = (1u << p.bits) - 1u;

  // ---- load records, warp-striped: element (warp, i, lane) is tile position warp*ITEMS*32 + i*32 + lane ----
  uint4 rec[ITEMS];
  const uint32_t wbase = warp * (ITEMS * 32) + lane;
  if (FIRST) {
    // records are built from the SoA storage blocks; when the whole tile sits in one block (the common case)
    // the block is located once per tile instead of once per record
    const BlockAddr a0 = locate(p.map, tile0);
    const bool one_block = a0.slot + kTile <= p.map.B;
    const uint32_t* sp = reinterpret_cast<const uint32_t*>(a0.base) + a0.slot;
    const uint32_t* tp = reinterpret_cast<const uint32_t*>(a0.base + p.map.off_tgt) + a0.slot;
    const uint32_t* wp = reinterpret_cast<const uint32_t*>(a0.base + p.map.off_w) + a0.slot;
    const uint16_t* dp = reinterpret_cast<const uint16_t*>(a0.base + p.map.off_d) + a0.slot;
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
      const uint32_t e = wbase + i * 32;
      if (e < valid) {
        uint32_t s, d, t, w;
        if (one_block) {
          s = sp[e]; d = dp[e]; t = tp[e]; w = wp[e];
        } else {
          const BlockAddr a = locate(p.map, tile0 + e);
          s = *src_ptr(p.map, a);
          d = *d_ptr(p.map, a);
          t = *tgt_ptr(p.map, a);
          w = __float_as_uint(*w_ptr(p.map, a));
        }
        rec[i] = make_uint4((s << p.delay_bits) | d, (uint32_t)(tile0 + e), t, w);
      } else {
        rec[i] = make_uint4(0xffffffffu, 0u, 0u, 0u);
      }
    }
  } else {
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) {
      const uint32_t e = wbase + i * 32;
      // padding sorts behind every real record of the tile and is never written out
      rec[i] = e < valid ? p.recs_in[tile0 + e] : make_uint4(0xffffffffu, 0u, 0u, 0u);
    }
  }

  // ---- early counts: per-warp digit histogram with fire-and-forget shared-memory atomics ----
  uint32_t* my_hist = sm.warp_hist[warp];
#pragma unroll
  for (int i = 0; i < ITEMS; ++i) atomicAdd(&my_hist[(rec[i].x >> p.shift) & mask], 1u);
  __syncthreads();

  // ---- per digit: exclusive scan over the warps, tile count -> publish the tile aggregate right away;
  //      exclusive scan over the digits -> where each digit's run starts inside the tile ----
  uint32_t real = 0, my_excl = 0;
  if (threadIdx.x < kRadix) {
    const uint32_t d = threadIdx.x;
    uint32_t cnt[kWarps];
#pragma unroll
    for (int w = 0; w < kWarps; ++w) cnt[w] = sm.warp_hist[w][d];
    uint32_t run = 0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) {
      sm.warp_hist[w][d] = run;
      run += cnt[w];
    }
    const uint32_t tile_count = run;
    // padding records of a ragged last tile all carry the largest digit; they are not part of the data
    real = (d == mask) ? run - (kTile - valid) : run;
    st_relaxed_u64(p.status + (uint64_t)tile * kRadix + d, p.epoch | (tile == 0 ? kFlagInclusive : kFlagAggregate) | real);
    uint32_t inc = tile_count;
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, s);
      if (lane >= (uint32_t)s) inc += t;
    }
    if (lane == 31) sm.scan_tmp[warp] = inc;
    asm volatile("bar.sync 1, %0;" ::"n"(kRadix));
    uint32_t base = 0;
    for (uint32_t w = 0; w < warp; ++w) base += sm.scan_tmp[w];
    my_excl = base + inc - tile_count;
    sm.tile_excl[d] = my_excl;
  }
  __syncthreads();

  // ---- stable rank + scatter into shared memory in one go: the lowest lane of each group of equal digits
  //      bumps the warp's running offset for that digit (atomics of one warp to one address retire in
  //      program order, so items keep their position order) and the group shares the old value ----
#pragma unroll
  for (int i = 0; i < ITEMS; ++i) {
    const uint32_t d = (rec[i].x >> p.shift) & mask;
    const uint32_t peers = peers_of<MATCH>(d, sm.warp_masks[warp]);
    const uint32_t below = __popc(peers & lanemask_lt());
    uint32_t old = 0;
    if (below == 0) old = atomicAdd(&my_hist[d], (uint32_t)__popc(peers));
    old = __shfl_sync(0xffffffffu, old, __ffs(peers) - 1);
    sm.recs[sm.tile_excl[d] + old + below] = rec[i];
  }

  // ---- look-back: where this tile's run of each digit starts in the output ----
  if (threadIdx.x < kRadix) {
    const uint32_t d = threadIdx.x;
    uint64_t excl = 0;
    if (tile != 0) {
      excl = look_back(p.status, tile, d, p.epoch, p.error_flag);
      st_relaxed_u64(p.status + (uint64_t)tile * kRadix + d, p.epoch | kFlagInclusive | (excl + real));
    }
    sm.global_off[d] = p.bin_start[d] + (uint32_t)excl - my_excl;
  }
  __syncthreads();

  // ---- write out: consecutive threads write consecutive records of a digit run ----
  const uint32_t dmask = (1u << p.delay_bits) - 1u;
#pragma unroll
  for (int i = 0; i < ITEMS; ++i) {
    const uint32_t j = i * THREADS + threadIdx.x;
    if (j < valid) {
      const uint4 r = sm.recs[j];
      const uint32_t g = sm.global_off[(r.x >> p.shift) & mask] + j;
      if (LAST) {
        p.out_src[g] = r.x >> p.delay_bits;
        p.out_d[g] = (uint16_t)(r.x & dmask);
        p.out_tgt[g] = r.z;
        p.out_w[g] = __uint_as_float(r.w);
        p.out_perm[g] = r.y;
      } else {
        p.recs_out[g] = r;
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Permutation apply (step a11): sorted_target[j] = target[perm[j]], sorted_weight[j] = weight[perm[j]];
// source and delay are unpacked from the sorted key.
// ---------------------------------------------------------------------------------------------
constexpr int kPermThreads = 256;

template <typename KeyT>
__global__ void __launch_bounds__(kPermThreads) permute_kernel(const __grid_constant__ BlockMap map, uint32_t n,
                                                              uint32_t delay_bits, const KeyT* __restrict__ keys,
                                                              const uint32_t* __restrict__ perm,
                                                              uint32_t* __restrict__ out_src,
                                                              uint32_t* __restrict__ out_tgt,
                                                              float* __restrict__ out_w,
                                                              uint16_t* __restrict__ out_d) {
  const uint64_t j = (uint64_t)blockIdx.x * kPermThreads + threadIdx.x;
  if (j >= n) return;
  const KeyT k = keys[j];
  const uint32_t pos = perm[j];
  const BlockAddr a = locate(map, pos);
  out_src[j] = (uint32_t)(k >> delay_bits);
  out_d[j] = (uint16_t)((uint32_t)k & ((1u << delay_bits) - 1u));
  out_tgt[j] = *tgt_ptr(map, a);
  out_w[j] = *w_ptr(map, a);
}

}  // namespace nc
