// nc_common.cuh -- shared device helpers of libnc (sm_100a): storage-block addressing, Philox4x32-10,
// relaxed/acquire global accesses, small warp utilities.  Product code: shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace nc {

constexpr int kWarp = 32;

// ---------------------------------------------------------------------------------------------
// Block-allocated SoA storage (reading D9).  Creation position pos lives in entry
// pos % B of block pos / B.  One block = one allocation holding four arrays of B entries:
//   u32 source[B] | u32 target[B] | f32 weight[B] | u16 delay[B]     (each start 256-byte aligned)
// The device-side table holds one base address per block.
// ---------------------------------------------------------------------------------------------
struct BlockMap {
  const uint64_t* table;  // device array of block base addresses
  uint64_t B;             // connections per block
  uint64_t magic;         // floor(2^64 / B) + 1 when B is not a power of two (exact for pos < 2^32)
  uint64_t off_tgt, off_w, off_d;  // byte offsets of the target / weight / delay arrays in a block
  uint32_t shift;         // log2(B) when B is a power of two, else 0xffffffff
  uint32_t pad_;
};

struct BlockAddr {
  uint64_t base;  // block base address
  uint64_t slot;  // entry inside the block
};

__device__ __forceinline__ BlockAddr locate(const BlockMap& m, uint64_t pos) {
  uint64_t blk;
  if (m.shift != 0xffffffffu) {
    blk = pos >> m.shift;
  } else {
    blk = __umul64hi(pos, m.magic);
  }
  BlockAddr a;
  a.slot = pos - blk * m.B;
  a.base = __ldg(m.table + blk);
  return a;
}

__device__ __forceinline__ uint32_t* src_ptr(const BlockMap&, const BlockAddr& a) {
  return reinterpret_cast<uint32_t*>(a.base) + a.slot;
}
__device__ __forceinline__ uint32_t* tgt_ptr(const BlockMap& m, const BlockAddr& a) {
  return reinterpret_cast<uint32_t*>(a.base + m.off_tgt) + a.slot;
}
__device__ __forceinline__ float* w_ptr(const BlockMap& m, const BlockAddr& a) {
  return reinterpret_cast<float*>(a.base + m.off_w) + a.slot;
}
__device__ __forceinline__ uint16_t* d_ptr(const BlockMap& m, const BlockAddr& a) {
  return reinterpret_cast<uint16_t*>(a.base + m.off_d) + a.slot;
}

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11; reading D2).  Ten rounds of
//   (c0,c1,c2,c3) <- (hi(M1 c2) ^ c1 ^ k0, lo(M1 c2), hi(M0 c0) ^ c3 ^ k1, lo(M0 c0))
// with the Weyl key bump (k0 += 0x9E3779B9, k1 += 0xBB67AE85) between rounds.  The key schedule is
// uniform across the grid, so after unrolling it lives on the uniform datapath; the per-thread cost is
// 20 IMAD.WIDE + 20 LOP3.
// ---------------------------------------------------------------------------------------------
struct Philox4 {
  uint32_t x, y, z, w;
};

__device__ __forceinline__ Philox4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                 uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
    c0 = n0;
    c2 = n2;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  return Philox4{c0, c1, c2, c3};
}

// ---------------------------------------------------------------------------------------------
// Philox4x32-10 specialised for one stream of counters (x, y, projection_id, stream) under one key
// (reading D2).  Everything that does not depend on (x, y) is evaluated once on the host
// (make_philox_stream) and reaches the kernel as launch constants: the ten round keys, the product
// M1 * projection_id of the first round and, when y == 0 (every rule with N_newconns < 2^32), the
// uniform halves of rounds two and three.  Per call: 18 IMAD.WIDE + 19 LOP3 (Y0) or 19 + 20 (general),
// no key-schedule additions.
// ---------------------------------------------------------------------------------------------
constexpr uint32_t kPhiloxM0 = 0xD2511F53u, kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u, kPhiloxW1 = 0xBB67AE85u;

struct PhiloxStream {
  uint32_t k0[10], k1[10];  // round keys: k0[r] = seed_lo + r W0, k1[r] = seed_hi + r W1
  uint32_t u0;              // hi(M1 projection) ^ k0[0]      after round 1: c0 = u0 ^ y
  uint32_t l1;              // lo(M1 projection)                             c1 = l1
  uint32_t a;               // stream ^ k1[0]                                c2 = hi(M0 x) ^ a,  c3 = lo(M0 x)
  uint32_t b;               // y == 0: l1 ^ k0[1]             after round 2: c0 = hi(M1 c2) ^ b, c1 = lo(M1 c2)
  uint32_t c;               // y == 0: hi(M0 u0) ^ k1[1]                     c2 = lo(M0 x) ^ c,  c3 = lo(M0 u0)
  uint32_t d;               // y == 0: lo(M0 u0) ^ k1[2]      after round 3: c2 = hi(M0 c0) ^ d
};

inline PhiloxStream make_philox_stream(uint32_t seed_lo, uint32_t seed_hi, uint32_t projection_id, uint32_t stream) {
  PhiloxStream s{};
  for (int r = 0; r < 10; ++r) {
    s.k0[r] = seed_lo + (uint32_t)r * kPhiloxW0;
    s.k1[r] = seed_hi + (uint32_t)r * kPhiloxW1;
  }
  const uint64_t p1 = (uint64_t)kPhiloxM1 * projection_id;
  s.u0 = (uint32_t)(p1 >> 32) ^ s.k0[0];
  s.l1 = (uint32_t)p1;
  s.a = stream ^ s.k1[0];
  const uint64_t q0 = (uint64_t)kPhiloxM0 * s.u0;
  s.b = s.l1 ^ s.k0[1];
  s.c = (uint32_t)(q0 >> 32) ^ s.k1[1];
  s.d = (uint32_t)q0 ^ s.k1[2];
  return s;
}

template <bool Y0>
__device__ __forceinline__ Philox4 philox_stream(uint32_t x, uint32_t y, const PhiloxStream& s) {
  uint32_t c0, c1, c2, c3;
  const uint64_t px = (uint64_t)kPhiloxM0 * (uint64_t)x;
  int first;
  if (Y0) {
    const uint32_t e2 = (uint32_t)(px >> 32) ^ s.a;             // round 1, lane-dependent half
    const uint64_t p1 = (uint64_t)kPhiloxM1 * (uint64_t)e2;     // round 2
    const uint32_t f0 = (uint32_t)(p1 >> 32) ^ s.b;
    const uint32_t f2 = (uint32_t)px ^ s.c;
    const uint64_t q0 = (uint64_t)kPhiloxM0 * (uint64_t)f0;     // round 3
    const uint64_t q1 = (uint64_t)kPhiloxM1 * (uint64_t)f2;
    c0 = (uint32_t)(q1 >> 32) ^ (uint32_t)p1 ^ s.k0[2];
    c1 = (uint32_t)q1;
    c2 = (uint32_t)(q0 >> 32) ^ s.d;
    c3 = (uint32_t)q0;
    first = 3;
  } else {
    c0 = s.u0 ^ y;
    c1 = s.l1;
    c2 = (uint32_t)(px >> 32) ^ s.a;
    c3 = (uint32_t)px;
    first = 1;
  }
#pragma unroll
  for (int r = 1; r < 10; ++r) {
    if (r < first) continue;
    const uint64_t p0 = (uint64_t)kPhiloxM0 * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)kPhiloxM1 * (uint64_t)c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ s.k0[r];
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ s.k1[r];
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
    c0 = n0;
    c2 = n2;
  }
  return Philox4{c0, c1, c2, c3};
}

// rand(N) of PAPER.md:95 as a multiply-high (reading D3): floor(word * N / 2^32), no rejection.
__device__ __forceinline__ uint32_t bounded(uint32_t word, uint32_t n) { return __umulhi(word, n); }

// i / d and i % d for 32-bit i with a host-computed reciprocal m = floor(2^64 / d) + 1 (exact for i < 2^32).
__device__ __forceinline__ uint32_t div_magic(uint32_t i, uint64_t m) { return (uint32_t)__umul64hi((uint64_t)i, m); }
inline uint64_t make_div_magic(uint32_t d) {
  return d <= 1 ? 0ull : (uint64_t)(((unsigned __int128)1 << 64) / d) + 1ull;  // d == 1 is handled by the caller
}

// Programmatic dependent launch (sm_90+): lets the next kernel of the stream start while this one drains,
// and (at the end of a kernel) waits for the previous one, so completion stays in stream order.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait_prior() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// ---------------------------------------------------------------------------------------------
// Global-memory accesses with explicit ordering (decoupled look-back status words).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void st_relaxed_u64(uint64_t* p, uint64_t v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ uint64_t ld_relaxed_u64(const uint64_t* p) {
  uint64_t v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}

__device__ __forceinline__ uint32_t lane_id() { return threadIdx.x & 31u; }
__device__ __forceinline__ uint32_t lanemask_lt() {
  uint32_t m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

}  // namespace nc
