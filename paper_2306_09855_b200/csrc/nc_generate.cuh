// nc_generate.cuh -- rule expansion + per-synapse draws + append (steps a3-a8 of DESIGN.md).
//
// One Philox4x32-10 call per synapse (reading D2): word 0 -> source draw, word 1 -> target draw,
// words 2,3 -> the Box-Muller pair whose cosine branch gives the weight and sine branch the delay
// (D5-D8).  Every synapse is a pure function of (seed, projection_id, i_newconns), so the mapping of
// synapses to threads is free: a thread owns GROUPS x 4 consecutive creation positions aligned to 4, and
// writes them with 128-bit stores into the SoA arrays of the storage block (Eqs. 1-3).
#pragma once

#include "nc_common.cuh"

namespace nc {

enum Rule : int {
  kOneToOne = 0,
  kAllToAll = 1,
  kFixedIndegree = 2,
  kFixedOutdegree = 3,
  kFixedTotalNumber = 4,
  kPairwiseBernoulli = 5
};

// Constants of one projection's weight and delay transforms (D7, D8).
struct SynConst {
  // fp32 fast path
  float w_mean, w_sd, w_lo, w_hi;
  float d_mean, d_sd, d_lo, d_hi, inv_dt;
  // guard band around a rounding boundary inside which the delay is redone in fp64:
  //   eps = eps_scale * (bound on |z1_32 - z1|) + eps_rel * |x| + eps_abs
  float eps_scale, eps_rel, eps_abs;
  int exact;               // NC_FLAG_EXACT_FP64: always take the fp64 path
  // fp64 path (same operations, in the order reading D8 writes them)
  double dd_mean, dd_sd, dd_lo, dd_hi, dinv_dt;
};

struct GenParams {
  BlockMap map;
  uint64_t pos0;  // N_conns before this call: first creation position written
  uint64_t n;     // N_newconns (Eq. 2)
  uint32_t s0, n_src, t0, n_tgt;
  uint32_t K;     // in/out-degree for the fixed-degree rules
  uint32_t seed_lo, seed_hi, projection_id;
  SynConst syn;
};

// Delay on the fp64 path: D5, D6 (sine branch) and D8 evaluated exactly in the order the readings state,
// with explicit round-to-nearest multiplies/adds so that nvcc cannot contract them into FMAs.
__device__ __noinline__ uint32_t delay_steps_fp64(uint32_t w2, uint32_t w3, const SynConst& c) {
  const double u1 = (double)((w2 >> 8) + 1u) * (1.0 / 16777216.0);
  const double u2 = (double)(w3 >> 8) * (1.0 / 16777216.0);
  const double r = sqrt(__dmul_rn(-2.0, log(u1)));
  const double theta = __dmul_rn(6.283185307179586, u2);
  const double z1 = __dmul_rn(r, sin(theta));
  double d = __dadd_rn(c.dd_mean, __dmul_rn(c.dd_sd, z1));
  d = d < c.dd_lo ? c.dd_lo : (d > c.dd_hi ? c.dd_hi : d);
  const double x = __dmul_rn(d, c.dinv_dt);
  double st = floor(__dadd_rn(x, 0.5));
  st = st < 1.0 ? 1.0 : (st > 65535.0 ? 65535.0 : st);
  return (uint32_t)st;
}

// ---------------------------------------------------------------------------------------------
// fp32 fast path of D5/D6 on the special-function unit.
//   r^2 = -2 ln u1 : lg2.approx away from u1 = 1; for t = 1 - u1 < 2^-5 (exact in fp32) the series
//         2t(1 + t/2 + t^2/3 + t^3/4 + t^4/5), because the absolute error of lg2.approx would otherwise
//         dominate a small r.  r = r^2 * rsqrt.approx(r^2).
//   (sin, cos)(2 pi u2) : sin.approx / cos.approx.
// Error model the guard band relies on (nc_selftest_fastpath checks it exhaustively, all 2^24 u1 and all
// 2^24 u2, against fp64 on the device, and the GPU tests require a 4x margin):
//   |r32 - r| <= kErrRa / r + kErrRb * r        |sin32 - sin|, |cos32 - cos| <= kErrTrig
// ---------------------------------------------------------------------------------------------
constexpr float kErrRa = 8.0e-7f;
constexpr float kErrRb = 1.0e-6f;
constexpr float kErrTrig = 4.0e-6f;

__device__ __forceinline__ float fast_radius(uint32_t w2, float& inv_r) {
  const float u1 = (float)((w2 >> 8) + 1u) * (1.0f / 16777216.0f);  // D5: exact in fp32
  const float t = 1.0f - u1;                                        // exact
  const float series = 2.0f * t * fmaf(t, fmaf(t, fmaf(t, fmaf(t, 0.2f, 0.25f), 0.33333334f), 0.5f), 1.0f);
  const float r2 = t < 0.03125f ? series : -1.3862943611198906f * __log2f(u1);
  inv_r = rsqrtf(r2);  // +inf when u1 == 1
  return r2 > 0.0f ? r2 * inv_r : 0.0f;
}
__device__ __forceinline__ void fast_sincos(uint32_t w3, float& sn, float& cs) {
  const float theta = (float)(w3 >> 8) * (6.283185307179586f / 16777216.0f);
  sn = __sinf(theta);
  cs = __cosf(theta);
}

// Weight (fp32) and delay (steps) of one synapse from Philox words 2 and 3.
__device__ __forceinline__ void draw_weight_delay(uint32_t w2, uint32_t w3, const SynConst& c, float& weight,
                                                  uint32_t& steps) {
  float inv_r;
  const float r = fast_radius(w2, inv_r);
  float sn, cs;
  fast_sincos(w3, sn, cs);
  const float z0 = r * cs, z1 = r * sn;
  // D7
  weight = fminf(fmaxf(fmaf(c.w_sd, z0, c.w_mean), c.w_lo), c.w_hi);
  // D8 on the fast path.  y = x + 0.5; m = nearest integer to y (magic-number rounding, exact for
  // |y| < 2^22); |y - m| is the distance of x to the nearest rounding boundary.  Outside the guard band
  // floor(y) is the same integer in fp32 and in the oracle's fp64; inside it the delay is redone in fp64.
  const float d = fminf(fmaxf(fmaf(c.d_sd, z1, c.d_mean), c.d_lo), c.d_hi);
  const float y = fmaf(d, c.inv_dt, 0.5f);
  const float m = (y + 12582912.0f) - 12582912.0f;
  const float err_z = fmaf(kErrRa, inv_r, (kErrRb + kErrTrig) * r);      // bound on |z1_32 - z1| (x 1/4 margin)
  const float eps = fmaf(c.eps_scale, err_z, fmaf(c.eps_rel, fabsf(y), c.eps_abs));
  const bool near = !(fabsf(y - m) >= eps);  // also true for NaN / inf
  if (near || c.exact || !(fabsf(y) < 4.0e6f)) {
    steps = delay_steps_fp64(w2, w3, c);
  } else {
    const float fl = m > y ? m - 1.0f : m;  // floor(y)
    steps = (uint32_t)(int)fminf(fmaxf(fl, 1.0f), 65535.0f);
  }
}

// ---------------------------------------------------------------------------------------------
// Generation kernel for every rule whose N_newconns is known up front (Eqs. 4-13).
//   VEC = true  : B % 4 == 0, so a 4-aligned group of positions never straddles a block and its four
//                 SoA slices are 16-byte aligned -> 128-bit stores (64-bit for the u16 delays).
//   VEC = false : any B (e.g. the paper's Fig. 1 example with B = 10): scalar stores.
// Thread t of a CTA owns groups (cta * GROUPS + k) * THREADS + t, k = 0..GROUPS-1, so that each warp-wide
// store instruction covers 512 contiguous bytes.
// ---------------------------------------------------------------------------------------------
constexpr int kGenThreads = 256;
constexpr int kGenGroups = 2;

template <int RULE, bool VEC>
__global__ void __launch_bounds__(kGenThreads) generate_kernel(const __grid_constant__ GenParams p) {
  const uint64_t first_group = p.pos0 >> 2;
  const uint64_t end = p.pos0 + p.n;
#pragma unroll
  for (int k = 0; k < kGenGroups; ++k) {
    const uint64_t g = first_group + ((uint64_t)blockIdx.x * kGenGroups + k) * kGenThreads + threadIdx.x;
    const uint64_t gpos = g << 2;
    if (gpos >= end) continue;

    uint32_t src[4], tgt[4], dly[4];
    float wgt[4];
    bool valid[4];
    // deterministic coordinate of the first in-range element of the group, then incremental
    // (N_newconns <= 2^32 - 1 for these rules, so i fits 32 bits and the division is a 32-bit one)
    const uint32_t i_first = gpos >= p.pos0 ? (uint32_t)(gpos - p.pos0) : 0u;
    uint32_t quo = 0, rem = 0;
    if (RULE == kAllToAll) {
      quo = i_first / p.n_tgt;
      rem = i_first - quo * p.n_tgt;
    } else if (RULE == kFixedIndegree || RULE == kFixedOutdegree) {
      quo = i_first / p.K;
      rem = i_first - quo * p.K;
    }
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const uint64_t pos = gpos + e;
      valid[e] = pos >= p.pos0 && pos < end;
      const uint64_t i = pos - p.pos0;  // i_newconns (Eq. 3); garbage when !valid, never stored
      const Philox4 rnd = philox4x32_10((uint32_t)i, (uint32_t)(i >> 32), p.projection_id, 0u, p.seed_lo, p.seed_hi);
      uint32_t s, t;
      if (RULE == kOneToOne) {  // Eqs. 4-5
        s = p.s0 + (uint32_t)i;
        t = p.t0 + (uint32_t)i;
      } else if (RULE == kAllToAll) {  // Eqs. 6-7
        s = p.s0 + quo;
        t = p.t0 + rem;
      } else if (RULE == kFixedOutdegree) {  // Eqs. 8-9
        s = p.s0 + quo;
        t = p.t0 + bounded(rnd.y, p.n_tgt);
      } else if (RULE == kFixedIndegree) {  // Eqs. 10-11
        s = p.s0 + bounded(rnd.x, p.n_src);
        t = p.t0 + quo;
      } else {  // fixed_total_number, Eqs. 12-13
        s = p.s0 + bounded(rnd.x, p.n_src);
        t = p.t0 + bounded(rnd.y, p.n_tgt);
      }
      if (RULE == kAllToAll || RULE == kFixedIndegree || RULE == kFixedOutdegree) {
        if (valid[e]) {
          const uint32_t lim = RULE == kAllToAll ? p.n_tgt : p.K;
          if (++rem == lim) {
            rem = 0;
            ++quo;
          }
        }
      }
      src[e] = s;
      tgt[e] = t;
      draw_weight_delay(rnd.z, rnd.w, p.syn, wgt[e], dly[e]);
    }

    if (VEC && valid[0] && valid[3]) {
      const BlockAddr a = locate(p.map, gpos);
      *reinterpret_cast<uint4*>(src_ptr(p.map, a)) = make_uint4(src[0], src[1], src[2], src[3]);
      *reinterpret_cast<uint4*>(tgt_ptr(p.map, a)) = make_uint4(tgt[0], tgt[1], tgt[2], tgt[3]);
      *reinterpret_cast<float4*>(w_ptr(p.map, a)) = make_float4(wgt[0], wgt[1], wgt[2], wgt[3]);
      *reinterpret_cast<uint2*>(d_ptr(p.map, a)) = make_uint2(dly[0] | (dly[1] << 16), dly[2] | (dly[3] << 16));
    } else {
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        if (!valid[e]) continue;
        const BlockAddr a = locate(p.map, gpos + e);
        *src_ptr(p.map, a) = src[e];
        *tgt_ptr(p.map, a) = tgt[e];
        *w_ptr(p.map, a) = wgt[e];
        *d_ptr(p.map, a) = (uint16_t)dly[e];
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// pairwise_bernoulli (readings D4, Q13, Q14), two kernels around an exact count:
//   trials : thread gt tries the 32 pairs q = 32 gt .. 32 gt + 31 with 8 Philox calls on the trial
//            stream (stream 1: ctr idx = q >> 2, word = q & 3), accept iff word < T; the 32 decisions
//            are one mask word, stored; a CTA (8192 trials) also stores its accepted count.
//   [device-wide exclusive scan of the CTA counts; the host reads the total and reserves blocks (Eq. 1)]
//   write  : one CTA per 8192 trials turns its 256 mask words into an ordered list of accepted pairs
//            in shared memory (warp-scan compaction), then generates the synapses densely, one thread
//            per accepted pair, at position pos0 + tile_offset + rank: ascending q, no atomics needed.
// ---------------------------------------------------------------------------------------------
constexpr int kBernThreads = 256;
constexpr int kBernTrialsPerThread = 32;
constexpr int kBernTile = kBernThreads * kBernTrialsPerThread;  // 8192 trials per CTA

struct BernParams {
  uint64_t n_pairs;       // N_src * N_tgt
  uint64_t threshold;     // T = floor(p 2^32), up to 2^32
  uint32_t seed_lo, seed_hi, projection_id;
  uint32_t* mask;         // [ceil(n_pairs / 32)]
  uint32_t* tile_count;   // [n_tiles]
};

__global__ void __launch_bounds__(kBernThreads) bernoulli_trials_kernel(const __grid_constant__ BernParams p) {
  const uint64_t gt = (uint64_t)blockIdx.x * kBernThreads + threadIdx.x;
  const uint64_t q0 = gt * kBernTrialsPerThread;
  uint32_t m = 0;
  if (q0 < p.n_pairs) {
    const uint64_t c0 = q0 >> 2;
#pragma unroll
    for (int j = 0; j < kBernTrialsPerThread / 4; ++j) {
      const uint64_t c = c0 + j;
      const Philox4 r = philox4x32_10((uint32_t)c, (uint32_t)(c >> 32), p.projection_id, 1u, p.seed_lo, p.seed_hi);
      m |= ((uint64_t)r.x < p.threshold ? 1u : 0u) << (4 * j + 0);
      m |= ((uint64_t)r.y < p.threshold ? 1u : 0u) << (4 * j + 1);
      m |= ((uint64_t)r.z < p.threshold ? 1u : 0u) << (4 * j + 2);
      m |= ((uint64_t)r.w < p.threshold ? 1u : 0u) << (4 * j + 3);
    }
    const uint64_t left = p.n_pairs - q0;
    if (left < 32) m &= (1u << (uint32_t)left) - 1u;
    p.mask[gt] = m;
  }
  // CTA count
  __shared__ uint32_t warp_sum[kBernThreads / 32];
  uint32_t c = __popc(m);
  c = __reduce_add_sync(0xffffffffu, c);
  if (lane_id() == 0) warp_sum[threadIdx.x >> 5] = c;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t tot = 0;
#pragma unroll
    for (int w = 0; w < kBernThreads / 32; ++w) tot += warp_sum[w];
    p.tile_count[blockIdx.x] = tot;
  }
}

struct BernWriteParams {
  GenParams g;                 // pos0 = N_conns before the call, n = accepted total
  uint64_t n_pairs;
  const uint32_t* mask;
  const uint32_t* tile_offset; // exclusive scan of tile_count
};

__global__ void __launch_bounds__(kBernThreads) bernoulli_write_kernel(const __grid_constant__ BernWriteParams p) {
  __shared__ uint16_t list[kBernTile];
  __shared__ uint32_t warp_off[kBernThreads / 32];
  __shared__ uint32_t tile_total;
  const uint64_t gt = (uint64_t)blockIdx.x * kBernThreads + threadIdx.x;
  const uint64_t tile_q0 = (uint64_t)blockIdx.x * kBernTile;
  const uint64_t n_words = (p.n_pairs + 31) >> 5;
  const uint32_t m = gt < n_words ? p.mask[gt] : 0u;
  // ordered compaction: warp inclusive scan of popcounts, then scan of the warp totals
  const uint32_t c = __popc(m);
  uint32_t inc = c;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t v = __shfl_up_sync(0xffffffffu, inc, d);
    if (lane_id() >= (uint32_t)d) inc += v;
  }
  if (lane_id() == 31) warp_off[threadIdx.x >> 5] = inc;
  __syncthreads();
  if (threadIdx.x == 0) {
    uint32_t run = 0;
#pragma unroll
    for (int w = 0; w < kBernThreads / 32; ++w) {
      const uint32_t v = warp_off[w];
      warp_off[w] = run;
      run += v;
    }
    tile_total = run;
  }
  __syncthreads();
  uint32_t o = warp_off[threadIdx.x >> 5] + inc - c;
  uint32_t mm = m;
  while (mm) {
    const int b = __ffs(mm) - 1;
    mm &= mm - 1;
    list[o++] = (uint16_t)(threadIdx.x * kBernTrialsPerThread + b);
  }
  __syncthreads();

  const uint32_t total = tile_total;
  const uint64_t out0 = p.g.pos0 + p.tile_offset[blockIdx.x];
  // source-major pair enumeration (same as Eqs. 6-7): q = (s - s0) N_tgt + (t - t0)
  const uint64_t row0 = tile_q0 / p.g.n_tgt;
  const uint64_t col0 = tile_q0 - row0 * p.g.n_tgt;
  for (uint32_t k = threadIdx.x; k < total; k += kBernThreads) {
    const uint32_t off = list[k];
    const uint64_t q = tile_q0 + off;
    const uint64_t v = col0 + off;  // < N_tgt + 8192
    uint32_t dq, col;
    if (p.g.n_tgt >= (uint32_t)kBernTile) {
      dq = v >= p.g.n_tgt ? 1u : 0u;
      col = (uint32_t)(v - (dq ? p.g.n_tgt : 0u));
    } else {
      dq = (uint32_t)v / p.g.n_tgt;
      col = (uint32_t)v - dq * p.g.n_tgt;
    }
    // the synapse stream is indexed by the pair index q, not by the rank (D2)
    const Philox4 rnd = philox4x32_10((uint32_t)q, (uint32_t)(q >> 32), p.g.projection_id, 0u, p.g.seed_lo, p.g.seed_hi);
    float wgt;
    uint32_t dly;
    draw_weight_delay(rnd.z, rnd.w, p.g.syn, wgt, dly);
    const BlockAddr a = locate(p.g.map, out0 + k);
    *src_ptr(p.g.map, a) = p.g.s0 + (uint32_t)row0 + dq;
    *tgt_ptr(p.g.map, a) = p.g.t0 + col;
    *w_ptr(p.g.map, a) = wgt;
    *d_ptr(p.g.map, a) = (uint16_t)dly;
  }
}

}  // namespace nc
