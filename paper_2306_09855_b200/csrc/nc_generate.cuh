// nc_generate.cuh -- rule expansion + per-synapse draws + append (steps a3-a8 of DESIGN.md).
//
// One Philox4x32-10 call per synapse (reading D2): word 0 -> source draw, word 1 -> target draw,
// words 2,3 -> the Box-Muller pair whose cosine branch gives the weight and sine branch the delay
// (D5-D8).  Every synapse is a pure function of (seed, projection_id, i_newconns), so the mapping of
// synapses to threads is free: a thread owns groups of 4 consecutive creation positions aligned to 4, and
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
  kPairwiseBernoulli = 5,
  kAllToAllSub = 6  // all_to_all restricted to a strip of target columns (a shard's owned targets, nc_set_shard): internal
};

// Constants of one projection's weight and delay transforms (D7, D8).
struct SynConst {
  // fp32 fast path
  float w_mean, w_sd, w_lo, w_hi;
  float d_mean, d_sd, d_lo, d_hi, inv_dt;
  // guard band around a rounding boundary inside which the synapse is redone in fp64:
  //   eps = eps_a / r + eps_b * r + eps_rel * |y| + eps_abs,   eps_a = (sd/dt) kErrRa, eps_b = (sd/dt) (kErrRb + kErrTrig)
  // NC_FLAG_EXACT_FP64 sets eps_abs = +inf: every synapse takes the fp64 path.
  float eps_a, eps_b, eps_rel, eps_abs;
  // fp64 path (same operations, in the order readings D7 / D8 write them)
  double dd_mean, dd_sd, dd_lo, dd_hi, dinv_dt;
  double dw_mean, dw_sd, dw_lo, dw_hi;
};

struct GenParams {
  BlockMap map;
  uint64_t pos0;  // N_conns before this call: first creation position written
  uint64_t n;     // N_newconns (Eq. 2)
  uint32_t s0, n_src, t0, n_tgt;
  // explicit node arrays ("the above formulas are used to derive the indexes of the array elements
  // from which to extract the node indexes"): when set, s0 / t0 are 0 and the formula's result indexes the array
  const uint32_t* src_nodes;
  const uint32_t* tgt_nodes;
  uint32_t K;          // in/out-degree for the fixed-degree rules
  uint32_t div;        // divisor of the deterministic coordinate (N_tgt for all_to_all, K for fixed degree)
  uint64_t div_magic;  // floor(2^64 / div) + 1
  PhiloxStream rng;    // synapse stream (stream 0) of this projection
  SynConst syn;
  uint32_t i_first;    // i_newconns of the first connection this launch creates (a shard generates a sub-range of a call's
                       // indexes, nc_set_shard); 0 for a whole call
  // kAllToAllSub: the launch creates, source by source, only target columns sub_off .. sub_off + sub_w - 1 of the call's
  // N_src x N_tgt grid (div = sub_w).  Local index j -> row j / sub_w, column sub_off + j % sub_w; the connection keeps the
  // index of the FULL call, i = row * n_tgt + column, for its random numbers (reading S1).
  uint32_t sub_w, sub_off;
};

// Weight and delay on the fp64 path: D5, D6, D7, D8 evaluated in the order the readings state, with explicit
// round-to-nearest multiplies/adds so that nvcc cannot contract them into FMAs.
__device__ __noinline__ void draw_fp64(uint32_t w2, uint32_t w3, const SynConst& c, float* weight, uint32_t* steps) {
  const double u1 = (double)((w2 >> 8) + 1u) * (1.0 / 16777216.0);
  const double u2 = (double)(w3 >> 8) * (1.0 / 16777216.0);
  const double r = sqrt(__dmul_rn(-2.0, log(u1)));
  const double theta = __dmul_rn(6.283185307179586, u2);
  double sn, cs;
  sincos(theta, &sn, &cs);
  const double z0 = __dmul_rn(r, cs), z1 = __dmul_rn(r, sn);
  double w = __dadd_rn(c.dw_mean, __dmul_rn(c.dw_sd, z0));
  w = w < c.dw_lo ? c.dw_lo : (w > c.dw_hi ? c.dw_hi : w);
  *weight = (float)w;
  double d = __dadd_rn(c.dd_mean, __dmul_rn(c.dd_sd, z1));
  d = d < c.dd_lo ? c.dd_lo : (d > c.dd_hi ? c.dd_hi : d);
  const double x = __dmul_rn(d, c.dinv_dt);
  double st = floor(__dadd_rn(x, 0.5));
  st = st < 1.0 ? 1.0 : (st > 65535.0 ? 65535.0 : st);
  *steps = (uint32_t)st;
}

// ---------------------------------------------------------------------------------------------
// fp32 fast path of D5/D6 on the special-function unit.
//   r^2 = -2 ln u1 : lg2.approx (absolute error ~2^-22 on [0.5, 2], so the error of r grows like 1/r);
//         for t = 1 - u1 < 2^-10 (exact in fp32) the series 2t(1 + t/2 + t^2/3) instead -- rare, so the generator
//         takes it behind a warp-uniform branch.
//         r = r^2 * rsqrt.approx(r^2); u1 = 1 gives r^2 = 0, which is lifted to 1e-30: 1/r = 1e15 makes the
//         guard band infinite and the synapse takes the fp64 path.
//   (sin, cos)(2 pi u2) : the argument is shifted by -pi into the interval where sin.approx / cos.approx are
//         most accurate; the shift flips both signs, which the NEGATED radius rn = -r undoes.
// Error model the guard band relies on (nc_selftest_fastpath checks it exhaustively, all 2^24 u1 and all
// 2^24 u2, against fp64 on the device, and the GPU tests require a 4x margin):
//   |r32 - r| <= kErrRa / r + kErrRb * r        |sin32 - sin|, |cos32 - cos| <= kErrTrig
// ---------------------------------------------------------------------------------------------
constexpr float kErrRa = 8.0e-7f;
constexpr float kErrRb = 1.0e-6f;
constexpr float kErrTrig = 4.0e-6f;
constexpr uint32_t kSeriesWord = 0xffc00000u;  // w2 >= this  <=>  t = 1 - u1 < 2^-10

__device__ __forceinline__ float lg2_approx(float x) {
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float sin_approx(float x) {
  float y;
  asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float cos_approx(float x) {
  float y;
  asm("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// r^2 from Philox word 2 by lg2.approx (accurate enough away from u1 = 1), and by the series.
__device__ __forceinline__ float fast_r2_log(uint32_t w2) {
  const float u1 = (float)((w2 >> 8) + 1u) * (1.0f / 16777216.0f);  // D5: exact in fp32
  return -1.3862943611198906f * lg2_approx(u1);
}
__device__ __forceinline__ float fast_r2_series(uint32_t w2) {
  const float t = (float)((~w2) >> 8) * (1.0f / 16777216.0f);  // 1 - u1, exact
  return (t + t) * fmaf(t, fmaf(t, 0.33333334f, 0.5f), 1.0f);
}
__device__ __forceinline__ float fast_r2(uint32_t w2) { return w2 >= kSeriesWord ? fast_r2_series(w2) : fast_r2_log(w2); }

// sin and cos of (2 pi u2 - pi) from Philox word 3.
__device__ __forceinline__ void fast_sincos_shifted(uint32_t w3, float& sn, float& cs) {
  const float theta = fmaf((float)(w3 >> 8), 6.283185307179586f / 16777216.0f, -3.14159265358979f);
  sn = sin_approx(theta);
  cs = cos_approx(theta);
}

// Weight (fp32) and delay (steps) of one synapse on the fast path, from r^2 (fast_r2) and Philox word 3.
// Returns true when the result is not proven equal to the oracle's and the synapse has to be redone by draw_fp64.
__device__ __forceinline__ bool draw_fast(float r2, uint32_t w3, const SynConst& c, float& weight, uint32_t& steps) {
  r2 = fmaxf(r2, 1e-30f);
  const float inv_r = rsqrt_approx(r2);
  const float rn = -r2 * inv_r;  // negated radius: undoes the sign flip of the shifted angle
  float sn, cs;
  fast_sincos_shifted(w3, sn, cs);
  const float z0 = rn * cs, z1 = rn * sn;
  // D7
  weight = fminf(fmaxf(fmaf(c.w_sd, z0, c.w_mean), c.w_lo), c.w_hi);
  // D8.  y = x + 0.5; m = nearest integer to y (magic-number rounding, exact for |y| < 2^22; the planner's
  // capacity check bounds y by 65536); |y - m| is the distance of x to the nearest rounding boundary.  Outside
  // the guard band floor(y) is the same integer in fp32 and in the oracle's fp64.
  const float d = fminf(fmaxf(fmaf(c.d_sd, z1, c.d_mean), c.d_lo), c.d_hi);
  const float y = fmaf(d, c.inv_dt, 0.5f);
  const float m = (y + 12582912.0f) - 12582912.0f;
  const float eps = fmaf(c.eps_a, inv_r, fmaf(-c.eps_b, rn, fmaf(c.eps_rel, fabsf(y), c.eps_abs)));
  steps = (uint32_t)max(__float2int_rd(y), 1);
  return !(fabsf(y - m) >= eps);  // also true for NaN / inf
}

// One synapse, any path (edge CTAs, pairwise_bernoulli).
__device__ __forceinline__ void draw_weight_delay(uint32_t w2, uint32_t w3, const SynConst& c, float& weight,
                                                  uint32_t& steps) {
  if (draw_fast(fast_r2(w2), w3, c, weight, steps)) draw_fp64(w2, w3, c, &weight, &steps);
}

// ---------------------------------------------------------------------------------------------
// Generation kernel for every rule whose N_newconns is known up front (Eqs. 4-13).
// A CTA owns one tile of kGenTile = 4096 consecutive creation positions aligned to the tile size (the same
// tiles the organisation step sorts), thread t the 4-aligned groups k * 256 + t, k = 0..3, of the tile, so
// that each warp-wide store instruction covers 512 contiguous bytes.
//   interior tiles (inside the projection and inside one storage block, B % 4 == 0): straight-line code, the
//       four SoA slices of a group are 128-bit stores (64-bit for the u16 delays); synapses the fast path
//       cannot prove (about 2e-4 of them) are redone in fp64 afterwards and overwrite their slots.
//   edge tiles (first / last tile of a projection, a tile straddling two blocks, any B): one synapse at a
//       time with scalar stores.
// ---------------------------------------------------------------------------------------------
constexpr int kGenThreads = 256;
constexpr int kGenGroups = 4;
constexpr int kGenTile = kGenThreads * kGenGroups * 4;

template <int RULE>
__device__ __forceinline__ void rule_coords(const GenParams& p, uint32_t i, uint32_t quo, uint32_t rem, uint32_t wx,
                                            uint32_t wy, uint32_t& s, uint32_t& t) {
  if (RULE == kOneToOne) {  // Eqs. 4-5
    s = p.s0 + i;
    t = p.t0 + i;
  } else if (RULE == kAllToAll) {  // Eqs. 6-7
    s = p.s0 + quo;
    t = p.t0 + rem;
  } else if (RULE == kAllToAllSub) {  // Eqs. 6-7 over the owned strip of columns
    s = p.s0 + quo;
    t = p.t0 + p.sub_off + rem;
  } else if (RULE == kFixedOutdegree) {  // Eqs. 8-9
    s = p.s0 + quo;
    t = p.t0 + bounded(wy, p.n_tgt);
  } else if (RULE == kFixedIndegree) {  // Eqs. 10-11
    s = p.s0 + bounded(wx, p.n_src);
    t = p.t0 + quo;
  } else {  // fixed_total_number, Eqs. 12-13
    s = p.s0 + bounded(wx, p.n_src);
    t = p.t0 + bounded(wy, p.n_tgt);
  }
}

template <int RULE>
__device__ __forceinline__ void split_index(const GenParams& p, uint32_t i, uint32_t& quo, uint32_t& rem) {
  quo = rem = 0;
  if (RULE == kAllToAll || RULE == kAllToAllSub || RULE == kFixedIndegree || RULE == kFixedOutdegree) {
    quo = p.div == 1 ? i : div_magic(i, p.div_magic);
    rem = i - quo * p.div;
  }
}

// Index of the connection in its (full) connect call, which keys its random numbers: the launch's own index except for a
// strip of all_to_all columns.
template <int RULE>
__device__ __forceinline__ uint32_t philox_index(const GenParams& p, uint32_t i, uint32_t quo, uint32_t rem) {
  return RULE == kAllToAllSub ? quo * p.n_tgt + p.sub_off + rem : i;
}

// Redo synapse i of the projection in fp64 and overwrite its weight and delay at creation position pos.
__device__ __noinline__ void redo_fp64(const GenParams& p, uint32_t i, uint64_t pos) {
  const Philox4 rnd = philox_stream<true>(i, 0u, p.rng);
  float w;
  uint32_t st;
  draw_fp64(rnd.z, rnd.w, p.syn, &w, &st);
  const BlockAddr a = locate(p.map, pos);
  *w_ptr(p.map, a) = w;
  *d_ptr(p.map, a) = (uint16_t)st;
}

__device__ __forceinline__ void map_nodes(const GenParams& p, uint32_t& s, uint32_t& t) {
  if (p.src_nodes) s = __ldg(p.src_nodes + s);
  if (p.tgt_nodes) t = __ldg(p.tgt_nodes + t);
}

// ARR: the projection names its sources and/or targets by explicit node arrays (kept out of the range kernels)
template <int RULE, bool ARR>
__global__ void __launch_bounds__(kGenThreads) generate_kernel(const __grid_constant__ GenParams p) {
  pdl_launch_dependents();
  const uint64_t end = p.pos0 + p.n;
  const uint64_t tile0 = (p.pos0 / kGenTile + blockIdx.x) * kGenTile;
  const BlockAddr a0 = locate(p.map, tile0);
  const bool interior = (p.map.B & 3) == 0 && tile0 >= p.pos0 && tile0 + kGenTile <= end && a0.slot + kGenTile <= p.map.B;
  if (interior) {
    // N_newconns <= 2^32 - 1 for these rules, so i fits 32 bits
    const uint32_t i_thread = p.i_first + (uint32_t)(tile0 - p.pos0) + threadIdx.x * 4;
    const uint64_t slot = a0.slot + threadIdx.x * 4;
    uint4* const sp = reinterpret_cast<uint4*>(reinterpret_cast<uint32_t*>(a0.base) + slot);
    uint4* const tp = reinterpret_cast<uint4*>(reinterpret_cast<uint32_t*>(a0.base + p.map.off_tgt) + slot);
    float4* const wp = reinterpret_cast<float4*>(reinterpret_cast<float*>(a0.base + p.map.off_w) + slot);
    uint2* const dp = reinterpret_cast<uint2*>(reinterpret_cast<uint16_t*>(a0.base + p.map.off_d) + slot);
    uint32_t redo = 0;
#pragma unroll
    for (int k = 0; k < kGenGroups; ++k) {
      const uint32_t i0 = i_thread + k * (kGenThreads * 4);
      uint32_t quo, rem;
      split_index<RULE>(p, i0, quo, rem);
      uint32_t src[4], tgt[4], dly[4], w2[4], w3[4];
      float wgt[4], r2[4];
      bool series = false;
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const Philox4 rnd = philox_stream<true>(philox_index<RULE>(p, i0 + e, quo, rem), 0u, p.rng);
        rule_coords<RULE>(p, i0 + e, quo, rem, rnd.x, rnd.y, src[e], tgt[e]);
        if (ARR) map_nodes(p, src[e], tgt[e]);
        if (RULE == kAllToAll || RULE == kAllToAllSub || RULE == kFixedIndegree || RULE == kFixedOutdegree) {
          if (++rem == p.div) {
            rem = 0;
            ++quo;
          }
        }
        w2[e] = rnd.z;
        w3[e] = rnd.w;
        r2[e] = fast_r2_log(w2[e]);
        series = series || w2[e] >= kSeriesWord;
      }
      if (__any_sync(0xffffffffu, series)) {  // about one group in eight
#pragma unroll
        for (int e = 0; e < 4; ++e)
          if (w2[e] >= kSeriesWord) r2[e] = fast_r2_series(w2[e]);
      }
#pragma unroll
      for (int e = 0; e < 4; ++e)
        if (draw_fast(r2[e], w3[e], p.syn, wgt[e], dly[e])) redo |= 1u << (k * 4 + e);
      sp[k * kGenThreads] = make_uint4(src[0], src[1], src[2], src[3]);
      tp[k * kGenThreads] = make_uint4(tgt[0], tgt[1], tgt[2], tgt[3]);
      wp[k * kGenThreads] = make_float4(wgt[0], wgt[1], wgt[2], wgt[3]);
      dp[k * kGenThreads] = make_uint2(dly[0] | (dly[1] << 16), dly[2] | (dly[3] << 16));
    }
    while (redo) {  // rare: the same thread wrote these slots above, so program order makes the overwrite final
      const int b = __ffs(redo) - 1;
      redo &= redo - 1;
      const uint32_t off = (uint32_t)(b >> 2) * (kGenThreads * 4) + (b & 3);
      uint32_t ri = i_thread + off;
      if (RULE == kAllToAllSub) {
        uint32_t q, r;
        split_index<RULE>(p, ri, q, r);
        ri = philox_index<RULE>(p, ri, q, r);
      }
      redo_fp64(p, ri, tile0 + threadIdx.x * 4 + off);
    }
  } else {
    for (int k = 0; k < kGenGroups * 4; ++k) {
      const uint64_t pos = tile0 + (uint64_t)(k >> 2) * (kGenThreads * 4) + threadIdx.x * 4 + (k & 3);
      if (pos < p.pos0 || pos >= end) continue;
      const uint32_t i = p.i_first + (uint32_t)(pos - p.pos0);  // i_newconns (Eq. 3)
      uint32_t quo, rem, s, t, dly;
      float wgt;
      split_index<RULE>(p, i, quo, rem);
      const Philox4 rnd = philox_stream<true>(philox_index<RULE>(p, i, quo, rem), 0u, p.rng);
      rule_coords<RULE>(p, i, quo, rem, rnd.x, rnd.y, s, t);
      if (ARR) map_nodes(p, s, t);
      draw_weight_delay(rnd.z, rnd.w, p.syn, wgt, dly);
      const BlockAddr a = locate(p.map, pos);
      *src_ptr(p.map, a) = s;
      *tgt_ptr(p.map, a) = t;
      *w_ptr(p.map, a) = wgt;
      *d_ptr(p.map, a) = (uint16_t)dly;
    }
  }
  pdl_wait_prior();
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
  PhiloxStream rng;       // trial stream (stream 1) of this projection
  uint32_t* mask;         // [ceil(n_pairs / 32)]
  uint32_t* tile_count;   // [n_tiles]
};

// T32: the threshold fits 32 bits (p < 1), so a trial is one 32-bit compare; T = 2^32 (p = 1, every word is below it) keeps
// the 64-bit compare.
template <bool T32>
__global__ void __launch_bounds__(kBernThreads) bernoulli_trials_kernel(const __grid_constant__ BernParams p) {
  const uint64_t gt = (uint64_t)blockIdx.x * kBernThreads + threadIdx.x;
  const uint64_t q0 = gt * kBernTrialsPerThread;
  uint32_t m = 0;
  if (q0 < p.n_pairs) {
    const uint64_t c0 = q0 >> 2;
    if (T32) {
      // The COMPLEMENT of the mask is built from the carry-out of the addition word + (2^32 - T), which is 1 iff word >= T
      // (1 <= T < 2^32 here): m' = 2 m' + (word >= T), two instructions per trial, one complement at the end; trials are
      // taken from the last to the first so that trial k ends up in bit k.  add.cc / addc rather than sub.cc / addc: PTX
      // defines the carry-out of add.cc and that addc adds it; it does not say what addc sees after a sub.cc.
      const uint32_t neg_t = 0u - (uint32_t)p.threshold;
#pragma unroll
      for (int j = kBernTrialsPerThread / 4 - 1; j >= 0; --j) {
        const uint64_t c = c0 + j;
        const Philox4 r = philox_stream<false>((uint32_t)c, (uint32_t)(c >> 32), p.rng);
        asm("{\n .reg .u32 d;\n"
            " add.cc.u32 d, %1, %5;\n addc.u32 %0, %0, %0;\n"
            " add.cc.u32 d, %2, %5;\n addc.u32 %0, %0, %0;\n"
            " add.cc.u32 d, %3, %5;\n addc.u32 %0, %0, %0;\n"
            " add.cc.u32 d, %4, %5;\n addc.u32 %0, %0, %0;\n}"
            : "+r"(m)
            : "r"(r.w), "r"(r.z), "r"(r.y), "r"(r.x), "r"(neg_t));
      }
      m = ~m;
    } else {
#pragma unroll
      for (int j = 0; j < kBernTrialsPerThread / 4; ++j) {
        const uint64_t c = c0 + j;
        const Philox4 r = philox_stream<false>((uint32_t)c, (uint32_t)(c >> 32), p.rng);
        m |= ((uint64_t)r.x < p.threshold ? 1u : 0u) << (4 * j + 0);
        m |= ((uint64_t)r.y < p.threshold ? 1u : 0u) << (4 * j + 1);
        m |= ((uint64_t)r.z < p.threshold ? 1u : 0u) << (4 * j + 2);
        m |= ((uint64_t)r.w < p.threshold ? 1u : 0u) << (4 * j + 3);
      }
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
  uint32_t one_to_one;         // pair q is (q, q) (one_to_one through the pair-mask path, nc_flags.cuh) instead of source-major
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
    const Philox4 rnd = philox_stream<false>((uint32_t)q, (uint32_t)(q >> 32), p.g.rng);
    float wgt;
    uint32_t dly;
    draw_weight_delay(rnd.z, rnd.w, p.g.syn, wgt, dly);
    const BlockAddr a = locate(p.g.map, out0 + k);
    uint32_t s = p.g.s0 + (uint32_t)row0 + dq, t = p.g.t0 + col;
    if (p.one_to_one) {
      s = p.g.s0 + (uint32_t)q;
      t = p.g.t0 + (uint32_t)q;
    }
    map_nodes(p.g, s, t);
    *src_ptr(p.g.map, a) = s;
    *tgt_ptr(p.g.map, a) = t;
    *w_ptr(p.g.map, a) = wgt;
    *d_ptr(p.g.map, a) = (uint16_t)dly;
  }
}

// ---------------------------------------------------------------------------------------------
// Per-connection value arrays (weights and delays "specified for each connection by an array having a
// size equal to the number of connections"): connection i of the projection, at creation position pos0 + i, takes
// w[i] as it is and / or d_ms[i] through reading D8 in fp64 (one multiply by 1/dt, round half up, at least one
// step).  Runs after the projection's generate kernel; the arrays come from the host, so PCIe bounds this path.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) set_values_kernel(const __grid_constant__ BlockMap map, uint64_t pos0, uint64_t n,
                                                        const float* __restrict__ w, const double* __restrict__ d_ms,
                                                        double inv_dt) {
  const uint64_t stride = (uint64_t)gridDim.x * 256u;
  for (uint64_t i = (uint64_t)blockIdx.x * 256u + threadIdx.x; i < n; i += stride) {
    const BlockAddr a = locate(map, pos0 + i);
    if (w) *w_ptr(map, a) = w[i];
    if (d_ms) {
      const double x = __dmul_rn(d_ms[i], inv_dt);
      double steps = floor(__dadd_rn(x, 0.5));
      steps = steps < 1.0 ? 1.0 : (steps > 65535.0 ? 65535.0 : steps);
      *d_ptr(map, a) = (uint16_t)(int)steps;
    }
  }
}

}  // namespace nc
