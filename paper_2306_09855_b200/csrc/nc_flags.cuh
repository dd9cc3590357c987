// nc_flags.cuh -- connect calls with autapses and / or multapses prohibited ("Autapses and multapses are
// currently always allowed in NEST GPU; therefore another useful addition would be the possibility to prohibit them (for
// example, using a flag as in the CPU version of NEST)").  Readings A1-A6 (include/nc.h):
//   A2  one_to_one / all_to_all / pairwise_bernoulli without autapses: the pair-mask machinery of pairwise_bernoulli
//       (mask of accepted pairs -> exact count -> Eq. 1 reservation -> ordered write) with the equal-id pairs cleared:
//       pair_mask_fill_kernel (every pair accepted) and pair_mask_clear_autapses_kernel.
//   A3-A5  fixed_indegree / fixed_outdegree / fixed_total_number: generate_flagged_kernel, one connection per thread --
//       bounded redraws on further Philox streams, or the k-th value of a keyed permutation of the allowed partners
//       (cycle walking over a balanced Feistel network) when partners must not repeat.
// These calls are off the bench path: clarity over speed (scalar stores, a division per connection).
#pragma once

#include "nc_common.cuh"
#include "nc_generate.cuh"

namespace nc {

constexpr uint32_t kNoAutapses = 1u, kNoMultapses = 2u;
constexpr uint32_t kNoIndex = 0xffffffffu;

// ---------------------------------------------------------------------------------------------
// A2: pair masks
// ---------------------------------------------------------------------------------------------
struct PairMaskParams {
  uint64_t n_pairs;
  uint32_t n_src, n_tgt, s0, t0;
  uint32_t one_to_one;        // pair q is (q, q) instead of (q div N_tgt, q mod N_tgt)
  const uint32_t* self_tgt;   // node arrays on either side: for source index sl the target index with the same id, or kNoIndex
  uint32_t* mask;             // [ceil(n_pairs / 32)]
  uint32_t* tile_count;       // [ceil(n_pairs / kBernTile)]
};

// every pair accepted: all_to_all and one_to_one through the pair-mask path
__global__ void __launch_bounds__(kBernThreads) pair_mask_fill_kernel(const __grid_constant__ PairMaskParams p) {
  const uint64_t gt = (uint64_t)blockIdx.x * kBernThreads + threadIdx.x;
  const uint64_t q0 = gt * kBernTrialsPerThread;
  uint32_t m = 0;
  if (q0 < p.n_pairs) {
    const uint64_t left = p.n_pairs - q0;
    m = left < 32 ? (1u << (uint32_t)left) - 1u : 0xffffffffu;
    p.mask[gt] = m;
  }
  __shared__ uint32_t warp_sum[kBernThreads / 32];
  uint32_t c = __reduce_add_sync(0xffffffffu, __popc(m));
  if (lane_id() == 0) warp_sum[threadIdx.x >> 5] = c;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t tot = 0;
#pragma unroll
    for (int w = 0; w < kBernThreads / 32; ++w) tot += warp_sum[w];
    p.tile_count[blockIdx.x] = tot;
  }
}

// one thread per source index: the (at most one) pair of that source whose target has the same id leaves the mask
__global__ void __launch_bounds__(256) pair_mask_clear_autapses_kernel(const __grid_constant__ PairMaskParams p) {
  const uint32_t sl = blockIdx.x * 256u + threadIdx.x;
  if (sl >= p.n_src) return;
  uint32_t tl = kNoIndex;
  if (p.self_tgt) {
    tl = p.self_tgt[sl];
  } else {
    const uint64_t id = (uint64_t)p.s0 + sl;
    if (id >= p.t0 && id < (uint64_t)p.t0 + p.n_tgt) tl = (uint32_t)(id - p.t0);
  }
  if (tl == kNoIndex) return;
  if (p.one_to_one && tl != sl) return;  // only the pair (sl, sl) exists
  const uint64_t q = p.one_to_one ? (uint64_t)sl : (uint64_t)sl * p.n_tgt + tl;
  const uint32_t bit = 1u << (uint32_t)(q & 31);
  const uint32_t old = atomicAnd(p.mask + (q >> 5), ~bit);
  if (old & bit) atomicSub(p.tile_count + q / kBernTile, 1u);
}

// ---------------------------------------------------------------------------------------------
// A5: permutation of [0, M) keyed by four words -- cycle walking over a balanced Feistel network on 2h bits,
// h = max(1, ceil(bits(M - 1) / 2)), 6 + ceil(24 / h) rounds (L, R) <- (R, L ^ (mix32(R ^ key_r) & (2^h - 1))),
// key_r = keys[r & 3] + r * 0x9E3779B9 (a two-round differential trail has probability 2^-h: narrow halves get more rounds).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t mix32(uint32_t v) {
  v ^= v >> 16;
  v *= 0x7feb352du;
  v ^= v >> 15;
  v *= 0x846ca68bu;
  v ^= v >> 16;
  return v;
}

__device__ __forceinline__ uint32_t keyed_permutation(uint32_t M, uint32_t k, const Philox4& keys) {
  if (M <= 1) return 0;
  const uint32_t bits = 32u - (uint32_t)__clz(M - 1);
  const uint32_t h = max(1u, (bits + 1) >> 1);
  const uint32_t mask = (1u << h) - 1u;
  const uint32_t rounds = 6u + (24u + h - 1u) / h;
  const uint32_t kw[4] = {keys.x, keys.y, keys.z, keys.w};
  uint32_t x = k;
  do {
    uint32_t L = x >> h, R = x & mask;
    for (uint32_t r = 0; r < rounds; ++r) {
      const uint32_t key_r = kw[r & 3] + r * 0x9E3779B9u;
      const uint32_t nR = L ^ (mix32(R ^ key_r) & mask);
      L = R;
      R = nR;
    }
    x = (L << h) | R;
  } while (x >= M);
  return x;
}

// ---------------------------------------------------------------------------------------------
// A3-A5: the random-partner rules under the flags
// ---------------------------------------------------------------------------------------------
struct FlagGenParams {
  GenParams g;       // as for generate_kernel (rng = stream 0 of the projection)
  uint32_t rule;     // kFixedIndegree, kFixedOutdegree or kFixedTotalNumber
  uint32_t flags;    // kNoAutapses | kNoMultapses
  uint32_t seed_lo, seed_hi, proj;
  const uint32_t* self_idx;  // A5 with kNoAutapses and node arrays: per fixed node its index among the partners, or kNoIndex
};

__global__ void __launch_bounds__(256) generate_flagged_kernel(const __grid_constant__ FlagGenParams p) {
  const GenParams& g = p.g;
  const bool no_aut = (p.flags & kNoAutapses) != 0, no_mult = (p.flags & kNoMultapses) != 0;
  const bool indeg = p.rule == (uint32_t)kFixedIndegree;
  auto sid = [&](uint32_t sl) { return g.src_nodes ? __ldg(g.src_nodes + sl) : g.s0 + sl; };
  auto tid = [&](uint32_t tl) { return g.tgt_nodes ? __ldg(g.tgt_nodes + tl) : g.t0 + tl; };
  const uint64_t stride = (uint64_t)gridDim.x * 256u;
  for (uint64_t i64 = (uint64_t)blockIdx.x * 256u + threadIdx.x; i64 < g.n; i64 += stride) {
    const uint32_t i = (uint32_t)i64;  // N_newconns <= 2^32 - 1
    const Philox4 rnd = philox_stream<true>(i, 0u, g.rng);
    float wgt;
    uint32_t dly;
    draw_weight_delay(rnd.z, rnd.w, g.syn, wgt, dly);  // weight and delay: words 2, 3 of the attempt-0 call, always
    uint32_t s_id, t_id;
    if (p.rule == (uint32_t)kFixedTotalNumber) {  // A4: both coordinates redrawn
      uint32_t sl = 0, tl = 0;
      for (uint32_t a = 0;; ++a) {
        const Philox4 w = a == 0 ? rnd : philox4x32_10(i, 0u, p.proj, 1u + a, p.seed_lo, p.seed_hi);
        sl = bounded(w.x, g.n_src);
        tl = bounded(w.y, g.n_tgt);
        if (sid(sl) != tid(tl)) break;
        if (a == 63) {  // never reached in practice
          tl = (tl + 1) % g.n_tgt;
          if (sid(sl) == tid(tl)) sl = (sl + 1) % g.n_src;
          break;
        }
      }
      s_id = sid(sl);
      t_id = tid(tl);
    } else {
      const uint32_t f = i / g.K, k = i - f * g.K;  // fixed node number, which of its K partners
      const uint32_t fid = indeg ? tid(f) : sid(f);
      const uint32_t n_part = indeg ? g.n_src : g.n_tgt;
      uint32_t x = 0;
      if (!no_mult) {  // A3: redraw the partner until its id differs
        for (uint32_t a = 0;; ++a) {
          const Philox4 w = a == 0 ? rnd : philox4x32_10(i, 0u, p.proj, 1u + a, p.seed_lo, p.seed_hi);
          x = bounded(indeg ? w.x : w.y, n_part);
          if ((indeg ? sid(x) : tid(x)) != fid) break;
          if (a == 63) {
            x = (x + 1) % n_part;
            break;
          }
        }
      } else {  // A5: k-th value of the keyed permutation of the allowed partner indexes
        uint32_t z = kNoIndex;
        if (no_aut) {
          if (p.self_idx) {
            z = p.self_idx[f];
          } else {
            const uint32_t first = indeg ? g.s0 : g.t0;
            if (fid >= first && (uint64_t)fid < (uint64_t)first + n_part) z = fid - first;
          }
        }
        const uint32_t M = n_part - (z != kNoIndex ? 1u : 0u);
        const Philox4 keys = philox4x32_10(f, 0u, p.proj, 2u, p.seed_lo, p.seed_hi);
        x = keyed_permutation(M, k, keys);
        if (z != kNoIndex && x >= z) x += 1;
      }
      s_id = indeg ? sid(x) : fid;
      t_id = indeg ? fid : tid(x);
    }
    const BlockAddr a = locate(g.map, g.pos0 + i64);
    *src_ptr(g.map, a) = s_id;
    *tgt_ptr(g.map, a) = t_id;
    *w_ptr(g.map, a) = wgt;
    *d_ptr(g.map, a) = (uint16_t)dly;
  }
}

}  // namespace nc
