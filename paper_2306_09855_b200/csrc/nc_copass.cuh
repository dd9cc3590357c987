// nc_copass.cuh -- COPASS block-sort of the connections inside their storage blocks (
// PAPER.md:426-642, Appendix A; readings C1-C6 of DESIGN.md section 8d).
//
// What the paper's algorithm is for: organise n connections held in k blocks of B with auxiliary memory of the
// order of ONE block instead of a second copy of everything.  Steps, Fig. 6:
//   (B) every block is sorted by the underlying sort           -> the record-carrying radix passes of nc_sort_split.cuh
//   (C) COPASS partition: a common threshold t and left partition sizes m_i with sum m_i = N_b (Sec. A2-A4)
//                                                              -> copass_partition_kernel (one CTA, one warp per
//                                                                 subarray, 32-ary searches)
//   (D) left partitions -> auxiliary array                     -> copass_segcopy_kernel (copass_gather_kernel)
//   (E) right partitions shifted right, block b freed          -> replaced by default: the k-1 partitions are taken at once
//                                                                 on the sorted blocks, the subarrays are kept as
//                                                                 extent lists, and after gathering an output block
//                                                                 ONE block is emptied into the holes the left
//                                                                 partitions left (copass_segcopy_kernel; host plan
//                                                                 in nc_api.cu, copass_extract_fill).  The shift to
//                                                                 the letter (NC_FLAG_COPASS_SHIFT):
//                                                                 copass_gather_kernel per destination block into a
//                                                                 spare block, then the two block pointers are
//                                                                 swapped (no overlapping move, each byte moved once)
//   (F) auxiliary array sorted into block b                    -> radix passes again; the last pass writes the block's
//                                                                 final arrays
// While this runs a block holds 16-byte records (key, creation position, target, weight), key = (source <<
// delay_bits) | delay: every move is a 128-bit copy whatever the shift.  Logical positions 0 .. n-1 map to
// (block, slot) through the same BlockMap as the creation-order storage (pos / B, pos % B).
//
// Ties: the radix passes are stable, candidates of Sec. A3 are ordered as pairs (value, i) and the d_i of Sec. A4
// are handed out lowest i first, so the block-sort as a whole is the stable sort reading D10 asks for.
#pragma once

#include "nc_common.cuh"

namespace nc {

constexpr uint32_t kCopassMaxBlocks = 4096;  // k: the partition keeps 7 words per subarray in shared memory
constexpr int kCopassThreads = 1024;

struct CopassInfo {  // what one partition did (device memory)
  uint32_t t;          // common threshold (A6, A7)
  uint32_t iterations; // iteration indices that computed mu / mu-bar
  int32_t last_step;   // 1 = Sec. A3, 2 = Sec. A4
  uint32_t pad;
};
struct CopassTotals {  // summed over the partitions of one organisation step (device memory)
  uint32_t partitions, iterations, last_step_1, last_step_2;
};

// ---- where the sorted keys of the subarrays are read from ----
struct FlatKeys {  // one array of 32-bit keys (nc_copass_partition, the stand-alone entry point)
  const uint32_t* k;
  __device__ __forceinline__ uint32_t operator()(uint32_t pos) const { return k[pos]; }
};
struct RecKeys {  // first word of the 16-byte record at logical position pos
  BlockMap map;
  __device__ __forceinline__ uint32_t operator()(uint32_t pos) const {
    const BlockAddr a = locate(map, pos);
    return reinterpret_cast<const uint4*>(a.base)[a.slot].x;
  }
};
__device__ __forceinline__ const uint4* rec_ptr(const BlockMap& m, uint32_t pos) {
  const BlockAddr a = locate(m, pos);
  return reinterpret_cast<const uint4*>(a.base) + a.slot;
}

// ---------------------------------------------------------------------------------------------
// Warp-wide 32-ary searches in the ascending subarray keys(base + j), j in [lo, hi):
//   LE = false: card{j : S_j <  t}   (Eqs. A13, A26)
//   LE = true : card{j : S_j <= t}   (Eqs. A12, A25)
// Every step probes 32 evenly spaced pivots at once (PAPER.md:494 uses one binary search per subarray; a warp
// turns log2 into log32 dependent loads).
// ---------------------------------------------------------------------------------------------
template <bool LE, typename Keys>
__device__ __forceinline__ uint32_t warp_card(const Keys& keys, uint32_t base, uint32_t lo, uint32_t hi, uint32_t t) {
  const uint32_t lane = lane_id();
  while (hi > lo) {
    const uint32_t width = hi - lo;
    if (width <= 32) {
      bool pred = false;
      if (lane < width) {
        const uint32_t v = keys(base + lo + lane);
        pred = LE ? v <= t : v < t;
      }
      return lo + __popc(__ballot_sync(0xffffffffu, pred));
    }
    const uint32_t step = (width + 31) / 32;
    const uint64_t want = (uint64_t)lo + (uint64_t)(lane + 1) * step - 1;
    const uint32_t idx = (uint32_t)min(want, (uint64_t)hi - 1);
    const uint32_t v = keys(base + idx);
    const uint32_t c = __popc(__ballot_sync(0xffffffffu, LE ? v <= t : v < t));  // pivots 0 .. c-1 hold
    const uint32_t pivot_c = __shfl_sync(0xffffffffu, idx, c & 31);
    const uint32_t pivot_b = __shfl_sync(0xffffffffu, idx, (c + 31) & 31);  // pivot c-1
    if (c == 32) return hi;  // the last pivot is hi - 1
    if (c > 0) lo = pivot_b + 1;
    hi = pivot_c;
  }
  return lo;
}

// ---- block-wide helpers for kCopassThreads threads ----
__device__ __forceinline__ uint64_t block_max_u64(uint64_t v, uint64_t* tmp /*[32]*/) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, d));
  __syncthreads();
  if (lane_id() == 0) tmp[threadIdx.x >> 5] = v;
  __syncthreads();
  uint64_t r = tmp[lane_id()];
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) r = max(r, __shfl_xor_sync(0xffffffffu, r, d));
  return r;
}
__device__ __forceinline__ uint64_t block_sum_u64(uint64_t v, uint64_t* tmp /*[32]*/) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
  __syncthreads();
  if (lane_id() == 0) tmp[threadIdx.x >> 5] = v;
  __syncthreads();
  uint64_t r = tmp[lane_id()];
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) r += __shfl_xor_sync(0xffffffffu, r, d);
  return r;
}
// exclusive scan of in[0..k) into out[0..k] (out[k] = total) plus an offset; all threads of the CTA call it
__device__ __forceinline__ void block_exscan(const uint32_t* in, uint32_t* out, uint32_t k, uint32_t offset,
                                             uint32_t* tmp /*[32]*/) {
  uint32_t carry = offset;
  for (uint32_t base = 0; base < k; base += kCopassThreads) {
    const uint32_t i = base + threadIdx.x;
    const uint32_t v = i < k ? in[i] : 0u;
    uint32_t inc = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t u = __shfl_up_sync(0xffffffffu, inc, d);
      if (lane_id() >= (uint32_t)d) inc += u;
    }
    __syncthreads();
    if (lane_id() == 31) tmp[threadIdx.x >> 5] = inc;
    __syncthreads();
    uint32_t before = 0, total = 0;
#pragma unroll
    for (uint32_t w = 0; w < kCopassThreads / 32; ++w) {
      const uint32_t u = tmp[w];
      if (w < (threadIdx.x >> 5)) before += u;
      total += u;
    }
    if (i < k) out[i] = carry + before + inc - v;
    carry += total;
  }
  __syncthreads();
  if (threadIdx.x == 0) out[k] = carry;
  __syncthreads();
}

// ---------------------------------------------------------------------------------------------
// COPASS partition.  One CTA.  Subarray i is keys(start[i] + j), j < len[i], ascending;
// 0 < m < sum len (the host guarantees it).  Outputs, all of k (+1) words in device memory:
//   m_out[i]        left partition sizes m_i (A8: sum = m)
//   left_prefix[i]  exclusive scan of m_i, left_prefix[k] = m          (where subarray i's left part goes in the aux)
//   right_src[i]    start[i] + m_i                                     (first element of the right partition)
//   new_start[i]    new_base + exclusive scan of (len - m_i), [k] = end (the subarrays after the shift of Fig. 6E)
//   new_len[i]      len[i] - m_i
// Shared memory: 7 arrays of k + 1 words.  Notation as in the appendix: m_lo = m-underbar, m_hi = m-bar,
// mu_lo = mu, mu_hi = mu-bar.  The thresholds t-underbar / t-bar themselves are never needed: only the counts
// they define enter Eqs. A19-A35.
// ---------------------------------------------------------------------------------------------
template <typename Keys>
__global__ void __launch_bounds__(kCopassThreads) copass_partition_kernel(
    const Keys keys, uint32_t k, uint32_t m, const uint32_t* __restrict__ start_g, const uint32_t* __restrict__ len_g,
    uint32_t new_base, uint32_t* __restrict__ m_out, uint32_t* __restrict__ left_prefix,
    uint32_t* __restrict__ right_src, uint32_t* __restrict__ new_start, uint32_t* __restrict__ new_len,
    CopassInfo* __restrict__ info, CopassTotals* __restrict__ totals, uint32_t m_step = 0, uint32_t out_stride = 0) {
  // several independent partitions of the same subarrays in one launch: CTA c takes m + c m_step and writes its
  // outputs out_stride words further on
  m += blockIdx.x * m_step;
  m_out += (size_t)blockIdx.x * out_stride;
  const bool for_moves = left_prefix != nullptr;  // the shift of Fig. 6E needs the prefixes; hole filling only m_i
  if (info) info += blockIdx.x;
  extern __shared__ uint32_t sh[];
  const size_t k1 = (size_t)k + 1;  // every array has a spare word for the total of a scan
  uint32_t* start = sh;
  uint32_t* len = sh + k1;
  uint32_t* m_lo = sh + 2 * k1;
  uint32_t* m_hi = sh + 3 * k1;
  uint32_t* mu_lo = sh + 4 * k1;
  uint32_t* mu_hi = sh + 5 * k1;
  uint32_t* res = sh + 6 * k1;  // m_i
  __shared__ uint64_t tmp64[32];
  __shared__ uint32_t tmp32[32];
  __shared__ uint32_t t_tilde_s, t_out_s;
  const uint32_t tid = threadIdx.x, warp = tid >> 5, lane = lane_id();
  constexpr uint32_t kWarps = kCopassThreads / 32;

  for (uint32_t i = tid; i < k; i += kCopassThreads) {
    start[i] = start_g[i];
    len[i] = len_g[i];
    m_lo[i] = 0;           // Eq. A16
    m_hi[i] = len_g[i];    // Eq. A17
  }
  __syncthreads();

  uint32_t iterations = 0;
  int last_step = 0;
  for (;;) {
    // Eqs. A20-A21: widest open interval, lowest i among equals (reading C2)
    uint64_t best = 0;
    for (uint32_t i = tid; i < k; i += kCopassThreads)
      best = max(best, ((uint64_t)(m_hi[i] - m_lo[i]) << 32) | (uint64_t)(0xffffffffu - i));
    best = block_max_u64(best, tmp64);
    const uint32_t widest = (uint32_t)(best >> 32), l = 0xffffffffu - (uint32_t)best;
    if (widest <= 1) {
      last_step = 1;
      break;
    }
    ++iterations;
    if (tid == 0) {
      const uint32_t m_tilde = m_lo[l] + (m_hi[l] - m_lo[l]) / 2;  // Eq. A22
      t_tilde_s = keys(start[l] + m_tilde);                       // Eq. A23
    }
    __syncthreads();
    const uint32_t t_tilde = t_tilde_s;
    for (uint32_t i = warp; i < k; i += kWarps) {  // Eqs. A25-A27: both counts lie inside [m_lo, m_hi]
      const uint32_t a = warp_card<false>(keys, start[i], m_lo[i], m_hi[i], t_tilde);
      const uint32_t b = warp_card<true>(keys, start[i], a, m_hi[i], t_tilde);
      if (lane == 0) {
        mu_lo[i] = a;
        mu_hi[i] = b;
      }
    }
    __syncthreads();
    uint64_t s_lo = 0, s_hi = 0;
    for (uint32_t i = tid; i < k; i += kCopassThreads) {
      s_lo += mu_lo[i];
      s_hi += mu_hi[i];
    }
    s_lo = block_sum_u64(s_lo, tmp64);
    s_hi = block_sum_u64(s_hi, tmp64);
    if (s_lo <= m && m <= s_hi) {  // Eq. A29 -> Sec. A4
      last_step = 2;
      if (tid == 0) t_out_s = t_tilde;
      break;
    }
    if (m < s_lo) {  // case 2, Eqs. A30-A32
      for (uint32_t i = tid; i < k; i += kCopassThreads) m_hi[i] = mu_lo[i];
    } else {         // case 3, Eqs. A33-A35
      for (uint32_t i = tid; i < k; i += kCopassThreads) m_lo[i] = mu_hi[i];
    }
    __syncthreads();
  }

  if (last_step == 2) {
    // Sec. A4: d = m - sum mu (A45); d_i = min(mu-bar_i - mu_i, what is left of d), lowest i first (reading C4)
    uint64_t s = 0;
    for (uint32_t i = tid; i < k; i += kCopassThreads) s += mu_lo[i];
    const uint32_t d = m - (uint32_t)block_sum_u64(s, tmp64);
    for (uint32_t i = tid; i < k; i += kCopassThreads) m_lo[i] = mu_hi[i] - mu_lo[i];  // the ranges
    __syncthreads();
    block_exscan(m_lo, m_hi, k, 0, tmp32);  // m_hi[i] = ranges of the subarrays before i
    for (uint32_t i = tid; i < k; i += kCopassThreads) {
      const uint32_t before = m_hi[i];
      const uint32_t d_i = min(m_lo[i], d > before ? d - before : 0u);
      res[i] = mu_lo[i] + d_i;  // Eq. A48
    }
  } else {
    // Sec. A3: candidates (S_{i, m_lo_i}, i) where m_hi = m_lo + 1 (A37, reading C3); the first d in the order of
    // the pairs go left (A38-A42)
    uint64_t s = 0;
    for (uint32_t i = tid; i < k; i += kCopassThreads) {
      s += m_lo[i];
      const bool cand = m_hi[i] == m_lo[i] + 1;
      mu_hi[i] = cand ? 1u : 0u;
      mu_lo[i] = cand ? keys(start[i] + m_lo[i]) : 0u;
    }
    const uint32_t d = m - (uint32_t)block_sum_u64(s, tmp64);  // Eq. A39 (the barrier inside publishes mu_lo / mu_hi)
    for (uint32_t i = tid; i < k; i += kCopassThreads) {
      uint32_t add = 0;
      if (mu_hi[i]) {
        const uint32_t v = mu_lo[i];
        uint32_t rank = 0;
        for (uint32_t j = 0; j < k; ++j)
          rank += (mu_hi[j] && (mu_lo[j] < v || (mu_lo[j] == v && j < i))) ? 1u : 0u;
        add = rank < d ? 1u : 0u;
        if (rank + 1 == d) t_out_s = v;  // the largest value put left
      }
      res[i] = m_lo[i] + add;
    }
  }
  __syncthreads();

  // what the moves of Fig. 6 D-E need
  for (uint32_t i = tid; i < k; i += kCopassThreads) {
    const uint32_t mi = res[i];
    m_out[i] = mi;
    m_hi[i] = len[i] - mi;
    if (for_moves) {
      right_src[i] = start[i] + mi;
      new_len[i] = len[i] - mi;
    }
  }
  __syncthreads();
  if (for_moves) {
    block_exscan(res, mu_lo, k, 0, tmp32);
    for (uint32_t i = tid; i < k; i += kCopassThreads) left_prefix[i] = mu_lo[i];
    if (tid == 0) left_prefix[k] = mu_lo[k];
    __syncthreads();
    block_exscan(m_hi, mu_lo, k, new_base, tmp32);
    for (uint32_t i = tid; i < k; i += kCopassThreads) new_start[i] = mu_lo[i];
  }
  if (tid == 0) {
    if (for_moves) new_start[k] = mu_lo[k];
    if (info) *info = CopassInfo{t_out_s, iterations, last_step, 0u};
    if (totals) {
      atomicAdd(&totals->partitions, 1u);
      atomicAdd(&totals->iterations, iterations);
      atomicAdd(last_step == 1 ? &totals->last_step_1 : &totals->last_step_2, 1u);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Moves of Fig. 6 D and E, one kernel: destination element j (j < count) is logical position p = p0 + j of a
// packing described by bound[0..k] (ascending; piece i covers [bound[i], bound[i+1])) and comes from logical
// position src_base[i] + (p - bound[i]).
//   D: bound = left_prefix, src_base = the subarray starts, p0 = 0, count = N_b      -> out = auxiliary array
//   E: bound = new_start,   src_base = right_src, p0 = first position of a block     -> out = the spare block
// 16 bytes per element in, 16 out (+ 1 for the digit side array in D).
// ---------------------------------------------------------------------------------------------
constexpr int kGatherThreads = 256;
constexpr int kGatherItems = 4;

__global__ void __launch_bounds__(kGatherThreads) copass_gather_kernel(const __grid_constant__ BlockMap map, uint32_t k,
                                                                      const uint32_t* __restrict__ bound,
                                                                      const uint32_t* __restrict__ src_base,
                                                                      uint32_t p0, uint32_t count,
                                                                      uint4* __restrict__ out,
                                                                      uint8_t* __restrict__ dig_out, uint32_t dig_shift,
                                                                      uint32_t dig_mask) {
  extern __shared__ uint32_t sh[];
  uint32_t* b = sh;            // k + 1
  uint32_t* s = sh + k + 1;    // k
  for (uint32_t i = threadIdx.x; i <= k; i += kGatherThreads) b[i] = bound[i];
  for (uint32_t i = threadIdx.x; i < k; i += kGatherThreads) s[i] = src_base[i];
  __syncthreads();
  const uint32_t j0 = blockIdx.x * (kGatherThreads * kGatherItems) + threadIdx.x;
  uint4 v[kGatherItems];
  bool ok[kGatherItems];
#pragma unroll
  for (int q = 0; q < kGatherItems; ++q) {
    const uint32_t j = j0 + q * kGatherThreads;
    ok[q] = j < count;
    if (ok[q]) {
      const uint32_t p = p0 + j;
      uint32_t lo = 0, hi = k;  // last piece i with b[i] <= p (empty pieces share their bound with the next one)
      while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (b[mid] <= p) lo = mid; else hi = mid;
      }
      v[q] = *rec_ptr(map, s[lo] + (p - b[lo]));
    }
  }
#pragma unroll
  for (int q = 0; q < kGatherItems; ++q)
    if (ok[q]) {
      out[j0 + q * kGatherThreads] = v[q];
      // D: the digit of the first radix pass over the auxiliary array, so that its tile counts read 1 B per record
      if (dig_out) dig_out[j0 + q * kGatherThreads] = (uint8_t)((v[q].x >> dig_shift) & dig_mask);
    }
}

// ---------------------------------------------------------------------------------------------
// Segmented copy for the hole-filling organisation (organise_copass_fill in nc_api.cu): element e (e < total) of
// the launch belongs to command c with prefix[c] <= e < prefix[c+1] and goes from position src[c] + (e - prefix[c])
// to position dst[c] + (e - prefix[c]); positions index the PHYSICAL blocks (block id * B + slot, the map's table
// lists the block pointers by id).  The commands are planned on the host from the partition results.
// ---------------------------------------------------------------------------------------------
constexpr uint32_t kSegSmemCmds = 2048;

__global__ void __launch_bounds__(kGatherThreads) copass_segcopy_kernel(const __grid_constant__ BlockMap map,
                                                                       const uint32_t* __restrict__ src,
                                                                       const uint32_t* __restrict__ dst,
                                                                       const uint32_t* __restrict__ prefix,
                                                                       uint32_t n_cmds, uint32_t total,
                                                                       uint8_t* __restrict__ dig_out, uint32_t dig_shift,
                                                                       uint32_t dig_mask) {
  __shared__ uint32_t s_src[kSegSmemCmds], s_dst[kSegSmemCmds], s_pre[kSegSmemCmds];
  const uint32_t *ps = src, *pd = dst, *pp = prefix;
  if (n_cmds <= kSegSmemCmds) {
    for (uint32_t i = threadIdx.x; i < n_cmds; i += kGatherThreads) {
      s_src[i] = src[i];
      s_dst[i] = dst[i];
      s_pre[i] = prefix[i];
    }
    __syncthreads();
    ps = s_src;
    pd = s_dst;
    pp = s_pre;
  }
  const uint32_t e0 = blockIdx.x * (kGatherThreads * kGatherItems) + threadIdx.x;
  uint4 v[kGatherItems];
  uint32_t to[kGatherItems];
  bool ok[kGatherItems];
#pragma unroll
  for (int q = 0; q < kGatherItems; ++q) {
    const uint32_t e = e0 + q * kGatherThreads;
    ok[q] = e < total;
    if (ok[q]) {
      uint32_t lo = 0, hi = n_cmds;  // last command with prefix <= e (commands are never empty)
      while (hi - lo > 1) {
        const uint32_t mid = (lo + hi) >> 1;
        if (pp[mid] <= e) lo = mid; else hi = mid;
      }
      const uint32_t off = e - pp[lo];
      v[q] = *rec_ptr(map, ps[lo] + off);
      to[q] = pd[lo] + off;
    }
  }
#pragma unroll
  for (int q = 0; q < kGatherItems; ++q)
    if (ok[q]) {
      *const_cast<uint4*>(rec_ptr(map, to[q])) = v[q];
      if (dig_out) dig_out[e0 + q * kGatherThreads] = (uint8_t)((v[q].x >> dig_shift) & dig_mask);
    }
}

// Digit counts of the first radix pass when the input is an array of records (the auxiliary array).
__global__ void __launch_bounds__(kCountThreads) tile_count_recs_kernel(const uint4* __restrict__ recs, uint32_t n,
                                                                       uint32_t tile_size, uint32_t shift, uint32_t bits,
                                                                       uint16_t* __restrict__ counts) {
  __shared__ uint32_t hist[kRadix];
  hist[threadIdx.x] = 0;
  __syncthreads();
  const uint32_t mask = (1u << bits) - 1u;
  const uint64_t tile0 = (uint64_t)blockIdx.x * tile_size;
  const uint32_t valid = (uint32_t)min((uint64_t)tile_size, (uint64_t)n - tile0);
  for (uint32_t e = threadIdx.x; e < valid; e += kCountThreads)
    atomicAdd(&hist[(recs[tile0 + e].x >> shift) & mask], 1u);
  __syncthreads();
  counts[(uint64_t)blockIdx.x * kRadix + threadIdx.x] = (uint16_t)hist[threadIdx.x];
}

// Records of one block -> the final block layout: source, target, weight, delay, creation position as five arrays.
__global__ void __launch_bounds__(256) copass_unpack_kernel(const uint4* __restrict__ recs, uint32_t n,
                                                           uint32_t delay_bits, uint32_t* __restrict__ src,
                                                           uint32_t* __restrict__ tgt, float* __restrict__ w,
                                                           uint16_t* __restrict__ d, uint32_t* __restrict__ perm) {
  const uint32_t dmask = (1u << delay_bits) - 1u;
  for (uint32_t j = blockIdx.x * 256u + threadIdx.x; j < n; j += gridDim.x * 256u) {
    const uint4 r = recs[j];
    src[j] = r.x >> delay_bits;
    d[j] = (uint16_t)(r.x & dmask);
    perm[j] = r.y;
    tgt[j] = r.z;
    w[j] = __uint_as_float(r.w);
  }
}

__global__ void copass_poke_kernel(uint64_t* table, uint32_t i, uint64_t a, uint32_t j, uint64_t b) {
  table[i] = a;
  if (j != 0xffffffffu) table[j] = b;
}

__global__ void copass_init_subarrays_kernel(uint32_t* start, uint32_t* len, uint32_t k, uint32_t B, uint32_t n) {
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < k; i += gridDim.x * blockDim.x) {
    const uint64_t s = (uint64_t)i * B;
    start[i] = (uint32_t)s;
    len[i] = (uint32_t)min((uint64_t)B, (uint64_t)n - s);
  }
}

}  // namespace nc
