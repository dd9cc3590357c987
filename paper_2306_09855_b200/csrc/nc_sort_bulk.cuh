// nc_sort_bulk.cuh -- the digit pass of nc_sort_split.cuh as a PERSISTENT kernel fed by the bulk-async copy engine
// (NC_FLAG_SORT_BULK; steps a10-a11 of DESIGN.md; PAPER.md:121 for what is sorted).  Kept selectable beside the default
// scatter_pass_kernel: same inputs (per-tile offsets from the count / scan kernels), same outputs bit for bit.
//
// One CTA per SM loops over tiles blockIdx.x, blockIdx.x + gridDim.x, ... (adjacent tiles are then written by different
// SMs at about the same time, which is what completes a shared 32-byte sector soonest -- tests/cuda/membench.cu,
// "pattern", R > 1).  A ring of kBulkBuffers tile buffers in shared memory:
//   load   : thread 0 issues cp.async.bulk (global -> shared, completion on an mbarrier) for the tile one iteration
//            ahead: 64 KB of records, or the four SoA slices of a storage block in the first pass, plus the tile's
//            256 output offsets;
//   rank   : as in scatter_pass_kernel (per-warp digit counters, ballots to find equal-digit peers), records read
//            from shared memory; the permutation is done IN PLACE through registers (every record of the tile is in
//            a register before the first is written back);
//   store  : middle passes: thread d issues ONE bulk store (shared -> global) for the tile's run of digit d -- the
//            records never pass through the load/store unit on their way out; the next pass's digit bytes are byte
//            stores (a run of bytes has no 16-byte alignment, so it cannot be a bulk copy).  Last pass: the final SoA
//            arrays by ordinary stores (4-byte runs cannot be bulk copies either).
// A buffer is refilled once the bulk stores that read it have completed their shared-memory reads
// (cp.async.bulk.wait_group.read).
//
// Measured on B200 (profiles/r02_scatter.md): 7.23 ms of digit passes per configs[2] step against 5.95 ms for the default
// kernels (the middle pass alone was on par in the working harness, 1.86 - 1.90 against 1.91 ms; the first pass with its four
// SoA slices and the last pass with ordinary stores from one CTA per SM are slower).  Not faster, because the pass is bound by
// how the memory system takes runs that start inside a sector, not by how the SM is fed; a bulk store costs its issuing warp
// ~70 cycles, and separating the ranking warps from store-issuing warps, ticketed tiles, and several consumer groups all
// measured slower.
//   rank   : (in place of the ballots above) one returning shared atomicAdd per record once atomic_lane_order_kernel has
//            confirmed on the device that same-address lanes are served in ascending lane order; the ballot form otherwise.
#pragma once

#include "nc_sort_split.cuh"

namespace nc {

constexpr int kBulkWarps = 8, kBulkItems = 16, kBulkBuffers = 3;
constexpr int kBulkTile = kBulkWarps * 32 * kBulkItems;  // 4096 records, 64 KB

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// Waits for the phase with the given parity; a wait that never ends (a lost copy) traps instead of hanging the device.
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t a = smem_u32(bar);
  uint32_t ok = 0, spins = 0;
  do {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok)
                 : "r"(a), "r"(parity)
                 : "memory");
    if (!ok && ++spins > (1u << 26)) __trap();
  } while (!ok);
}
__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
               "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void bulk_store(void* gdst, const void* smem_src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes)
               : "memory");
}

struct BulkSmem {
  uint4 buf[kBulkBuffers][kBulkTile];  // first pass: source | target | weight | delay slices, then the sorted records
  uint32_t offs_in[kBulkBuffers][kRadix];
  uint32_t warp_hist[kBulkWarps][kRadix];
  uint32_t global_off[kRadix];
  uint32_t scan_tmp[kRadix / 32];
  uint64_t full[kBulkBuffers];
};

// Do the lanes of ONE shared-memory atomicAdd instruction that hit the same address get their old values in ascending lane
// order?  (Not documented; measured true on B200, tests/cuda/membench.cu `atomorder`.)  The bulk kernel's ATOMIC_RANK form
// takes a record's rank among the equal digits of its warp from exactly that; nc_create checks it on the device it runs on
// and the ballot form is used wherever the check fails.
__global__ void __launch_bounds__(256) atomic_lane_order_kernel(uint32_t* violations, uint32_t iters) {
  __shared__ uint32_t hist[8][kRadix];
  const uint32_t warp = threadIdx.x >> 5, lane = lane_id();
  for (int i = lane; i < kRadix; i += 32) hist[warp][i] = 0;
  __syncwarp();
  uint32_t bad = 0;
  for (uint32_t it = 0; it < iters; ++it) {
    uint32_t x = (blockIdx.x * 256u + threadIdx.x) * 2654435761u + it * 40503u;
    x ^= x >> 15;
    x *= 0x846ca68bu;
    const uint32_t d = (x >> 16) % ((it & 3u) == 0 ? 2u : (it & 3u) == 1 ? 8u : kRadix);
    const uint32_t old = atomicAdd(&hist[warp][d], 1u);
    const uint32_t peers = __match_any_sync(0xffffffffu, d);
    // among equal digits the returned values must ascend with the lane: old = (value before the instruction) + (peers below)
    const uint32_t lowest = __shfl_sync(0xffffffffu, old, __ffs(peers) - 1);
    if (old != lowest + (uint32_t)__popc(peers & lanemask_lt())) ++bad;
  }
  if (bad) atomicAdd(violations, bad);
}

// FIRST requires every tile to lie inside one storage block with 16-byte aligned slices (B % kBulkTile == 0).
// ATOMIC_RANK: rank from one returning shared atomicAdd per record (see above) instead of a histogram round + eight ballots.
template <bool FIRST, bool LAST, bool ATOMIC_RANK>
__global__ void __launch_bounds__(kBulkWarps * 32, 1) scatter_bulk_kernel(const __grid_constant__ ScatterParams p,
                                                                         uint32_t n_tiles) {
  constexpr int kT = kBulkWarps * 32;
  constexpr int NB = kBulkBuffers;
  constexpr int ITEMS = kBulkItems;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  BulkSmem& sm = *reinterpret_cast<BulkSmem*>(smem_raw);
  const uint32_t warp = threadIdx.x >> 5, lane = lane_id(), tid = threadIdx.x;
  if (tid == 0) {
    for (int s = 0; s < NB; ++s) mbar_init(&sm.full[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const uint32_t my_tiles = blockIdx.x < n_tiles ? (n_tiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0u;
  const uint32_t mask = (1u << p.bits) - 1u;
  const uint32_t wbase = warp * (ITEMS * 32) + lane;
  uint32_t* my_hist = sm.warp_hist[warp];

  auto issue = [&](uint32_t it) {  // thread 0: bulk loads of the it-th tile of this CTA
    const uint32_t b = it % NB;
    const uint32_t tile = blockIdx.x + it * gridDim.x;
    const uint64_t tile0 = (uint64_t)tile * kBulkTile;
    const uint32_t valid = (uint32_t)min((uint64_t)kBulkTile, (uint64_t)p.n - tile0);
    unsigned char* dst = reinterpret_cast<unsigned char*>(sm.buf[b]);
    if (FIRST) {
      const BlockAddr a = locate(p.map, tile0);
      const uint32_t b4 = (valid * 4u + 15u) & ~15u, b2 = (valid * 2u + 15u) & ~15u;  // slices end 16-byte aligned inside a block
      mbar_expect_tx(&sm.full[b], 3u * b4 + b2 + kRadix * 4u);
      bulk_load(dst, reinterpret_cast<const unsigned char*>(a.base) + a.slot * 4, b4, &sm.full[b]);
      bulk_load(dst + kBulkTile * 4, reinterpret_cast<const unsigned char*>(a.base + p.map.off_tgt) + a.slot * 4, b4, &sm.full[b]);
      bulk_load(dst + kBulkTile * 8, reinterpret_cast<const unsigned char*>(a.base + p.map.off_w) + a.slot * 4, b4, &sm.full[b]);
      bulk_load(dst + kBulkTile * 12, reinterpret_cast<const unsigned char*>(a.base + p.map.off_d) + a.slot * 2, b2, &sm.full[b]);
    } else {
      mbar_expect_tx(&sm.full[b], valid * 16u + kRadix * 4u);
      bulk_load(dst, p.recs_in + tile0, valid * 16u, &sm.full[b]);
    }
    bulk_load(sm.offs_in[b], p.offs + (uint64_t)tile * kRadix, kRadix * 4u, &sm.full[b]);
  };
  if (tid == 0 && my_tiles > 0) issue(0);

  for (uint32_t k = 0; k < my_tiles; ++k) {
    const uint32_t b = k % NB, ph = (k / NB) & 1u;
    const uint32_t tile = blockIdx.x + k * gridDim.x;
    const uint64_t tile0 = (uint64_t)tile * kBulkTile;
    const uint32_t valid = (uint32_t)min((uint64_t)kBulkTile, (uint64_t)p.n - tile0);
    reinterpret_cast<uint4*>(my_hist)[lane] = make_uint4(0u, 0u, 0u, 0u);
    reinterpret_cast<uint4*>(my_hist)[lane + 32] = make_uint4(0u, 0u, 0u, 0u);
    __syncwarp();
    mbar_wait(&sm.full[b], ph);
    uint4* buf = sm.buf[b];
    // ---- records into registers, warp-striped: element (warp, i, lane) is tile position warp*ITEMS*32 + i*32 + lane ----
    uint4 rec[ITEMS];
    if (FIRST) {
      const uint32_t* sp = reinterpret_cast<const uint32_t*>(buf);
      const uint32_t* tp = sp + kBulkTile;
      const uint32_t* wp = sp + 2 * kBulkTile;
      const uint16_t* dp = reinterpret_cast<const uint16_t*>(sp + 3 * kBulkTile);
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) {
        const uint32_t e = wbase + i * 32;
        rec[i] = e < valid ? make_uint4((sp[e] << p.delay_bits) | dp[e], p.pos_base + (uint32_t)(tile0 + e), tp[e], wp[e])
                           : make_uint4(0xffffffffu, 0u, 0u, 0u);
      }
    } else {
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) {
        const uint32_t e = wbase + i * 32;
        // padding sorts behind every real record of the tile and is never written out
        rec[i] = e < valid ? buf[e] : make_uint4(0xffffffffu, 0u, 0u, 0u);
      }
    }
    uint32_t rk[ITEMS];
#pragma unroll
    for (int i = 0; i < ITEMS; ++i) rk[i] = atomicAdd(&my_hist[(rec[i].x >> p.shift) & mask], 1u);  // ATOMIC_RANK uses the value
    // the bulk stores of the previous tile may still read their buffer; those of the tile before it must have, before
    // its buffer (the one the next tile lands in) is refilled
    if (!LAST) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
    __syncthreads();  // every record of the tile is in a register; nobody reads the buffer of tile k - 2 any more
    if (tid == 0 && k + 1 < my_tiles) issue(k + 1);

    // ---- per digit: exclusive scan over the warps and over the digits (as in scatter_pass_kernel) ----
    uint32_t my_excl = 0, run = 0, out0 = 0;
    {
      const uint32_t d = tid;  // kT == kRadix
      out0 = sm.offs_in[b][d];
      uint32_t cnt[kBulkWarps];
#pragma unroll
      for (int w = 0; w < kBulkWarps; ++w) cnt[w] = sm.warp_hist[w][d];
#pragma unroll
      for (int w = 0; w < kBulkWarps; ++w) {
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
      __syncthreads();
      uint32_t base = 0;
#pragma unroll
      for (uint32_t w = 0; w < kRadix / 32; ++w) base += w < warp ? sm.scan_tmp[w] : 0u;
      my_excl = base + inc - run;
      sm.global_off[d] = out0 - my_excl;
#pragma unroll
      for (int w = 0; w < kBulkWarps; ++w) sm.warp_hist[w][d] = my_excl + cnt[w];
      if (d == mask) run -= kBulkTile - valid;  // padding records are not data
    }
    __syncthreads();

    // ---- stable rank, records back into the SAME buffer in tile-sorted order ----
    if (ATOMIC_RANK) {
      // my_hist[d] now holds the tile position of the warp's first record of digit d; rk[i] the record's rank behind it
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) rk[i] += my_hist[(rec[i].x >> p.shift) & mask];
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) buf[rk[i]] = rec[i];
    } else {
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) {
        const uint32_t d = (rec[i].x >> p.shift) & mask;
        const uint32_t peers = peers_of<kMatchBallot>(d, nullptr);
        const uint32_t below = __popc(peers & lanemask_lt());
        uint32_t old = 0;
        if (below == 0) old = atomicAdd(&my_hist[d], (uint32_t)__popc(peers));
        old = __shfl_sync(0xffffffffu, old, __ffs(peers) - 1);
        buf[old + below] = rec[i];
      }
    }
    if (!LAST) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the copy engine reads what was just written
    __syncthreads();

    if (LAST) {
      const uint32_t dmask = (1u << p.delay_bits) - 1u;
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) {
        const uint32_t j = i * kT + tid;
        if (j < valid) {
          const uint4 r = buf[j];
          const uint32_t g = sm.global_off[(r.x >> p.shift) & mask] + j;
          p.out_src[g] = r.x >> p.delay_bits;
          p.out_d[g] = (uint16_t)(r.x & dmask);
          p.out_tgt[g] = r.z;
          p.out_w[g] = __uint_as_float(r.w);
          p.out_perm[g] = r.y;
        }
      }
    } else {
      // ---- one bulk store per digit run; the next pass's digit of every record by byte stores ----
      if (run != 0) bulk_store(p.recs_out + out0, buf + my_excl, run * 16u);
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
      const uint32_t next_mask = (1u << p.next_bits) - 1u;
#pragma unroll
      for (int i = 0; i < ITEMS; ++i) {
        const uint32_t j = i * kT + tid;
        if (j < valid) {
          const uint32_t kx = buf[j].x;
          p.dig_out[sm.global_off[(kx >> p.shift) & mask] + j] = (uint8_t)((kx >> p.next_shift) & next_mask);
        }
      }
    }
  }
  if (!LAST) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

}  // namespace nc
