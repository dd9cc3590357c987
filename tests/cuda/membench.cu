// membench.cu -- TEST-ONLY microbenchmarks behind the bounds DESIGN.md quotes (built by __graft_entry__.build() and by
// tests/test_gpu_membench.py into tests/cuda/membench, git-ignored; nothing under paper_2306_09855_b200/ includes,
// links or runs this file).  Each section prints one table; profiles/r02_membench.md holds a run on one B200.
//
//   pattern   : the memory-system ceiling of a digit pass's WRITE PATTERN without any ranking: a plain copy that reads
//               64 KB tiles contiguously and writes them as `chunk`-byte pieces round-robin into S sequential streams,
//               pieces aligned to 128 B, or shifted by 16 / 32 B so that every piece starts inside a 32-byte sector /
//               a 128-byte line (what a stable radix scatter of 16-byte records produces: a run of tile t ends where
//               the run of tile t + 1 begins).  R > 1: one CTA writes R consecutive tiles, so the two parts of a shared
//               line are written by the same SM one tile period apart.
//   ring      : whether two consecutive digit passes can keep their intermediate array in the 126 MB L2 when the data is
//               processed group by group (a group = one bucket of an MSD first pass): per group, copy HBM -> ring slot
//               (256-byte pieces, 256 streams inside the group) and ring slot -> HBM (512-byte pieces, 128 streams),
//               groups alternating over CUDA streams so that the two kernels of neighbouring groups overlap; against
//               the same launches with a full-size intermediate array, and against the two full-array passes.
//   bulk      : the same pattern moved by cp.async.bulk alone (bulk load of a tile into shared memory, one bulk store
//               per piece), persistent CTAs with static or ticketed tiles -- the ceiling of a TMA-fed pass.
//   atomorder : whether same-address shared-memory atomics of ONE warp instruction return their old values in ascending
//               lane order (the property a rank-by-atomic variant of the pass would rest on).
//   red       : the ceiling of spike delivery's inner loop: read a target and a weight (8 B), one fp32
//               red.global.add into one of 77,169 accumulators (the node count of configs[2]), nothing else.
//   pipes     : issue cost of IMAD.WIDE.U32, IMAD, LOP3, FFMA per warp instruction per SM sub-partition, the figures
//               behind the integer-pipe bound of the generators.
#include <cuda_runtime.h>
#include <stdint.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>

#define CK(x)                                                                                   \
  do {                                                                                          \
    cudaError_t e_ = (x);                                                                       \
    if (e_ != cudaSuccess) {                                                                    \
      printf("CUDA error %s at line %d\n", cudaGetErrorString(e_), __LINE__);                   \
      exit(1);                                                                                  \
    }                                                                                           \
  } while (0)

namespace {

constexpr uint32_t kTileRecs = 4096;  // 64 KB of 16-byte records

struct Timer {
  cudaEvent_t a, b;
  Timer() {
    cudaEventCreate(&a);
    cudaEventCreate(&b);
  }
  void start() { cudaEventRecord(a); }
  float stop() {
    cudaEventRecord(b);
    cudaEventSynchronize(b);
    float ms;
    cudaEventElapsedTime(&ms, a, b);
    return ms;
  }
};

// ---------------------------------------------------------------------------------------------------------------
// pattern: LSU copy
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) pattern_copy(const uint4* __restrict__ in, uint4* __restrict__ out, uint32_t n_tiles,
                                                    uint32_t S, uint32_t cr_shift, uint32_t region, uint32_t sh, uint32_t R) {
  const uint32_t cpt = kTileRecs >> cr_shift, per = cpt / S;  // pieces per tile, pieces per tile and stream
  for (uint32_t t = 0; t < R; ++t) {
    const uint32_t tile = blockIdx.x * R + t;
    if (tile >= n_tiles) return;
    uint4 r[16];
    const uint4* src = in + (uint64_t)tile * kTileRecs;
#pragma unroll
    for (int i = 0; i < 16; ++i) r[i] = src[i * 256 + threadIdx.x];
#pragma unroll
    for (int i = 0; i < 16; ++i) {
      const uint32_t j = i * 256 + threadIdx.x;
      const uint32_t c = j >> cr_shift, o = j & ((1u << cr_shift) - 1u);
      const uint32_t s = c % S, q = c / S;
      out[(uint64_t)s * region + (((uint64_t)tile * per + q) << cr_shift) + o + sh] = r[i];
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// ring: the copy of `pattern` with L2 eviction-priority hints on its loads (LH) and stores (SH): 0 none, 1 evict_first,
// 2 evict_last
// ---------------------------------------------------------------------------------------------------------------
template <int H>
__device__ __forceinline__ uint64_t l2_policy() {
  uint64_t pol = 0;
  if (H == 1) asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  if (H == 2) asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}

template <int LH, int SH>
__global__ void __launch_bounds__(256) pattern_copy_hint(const uint4* __restrict__ in, uint4* __restrict__ out, uint32_t n_tiles,
                                                         uint32_t S, uint32_t cr_shift, uint32_t region, uint32_t sh) {
  const uint32_t cpt = kTileRecs >> cr_shift, per = cpt / S;
  const uint32_t tile = blockIdx.x;
  if (tile >= n_tiles) return;
  const uint64_t lpol = l2_policy<LH>(), spol = l2_policy<SH>();
  uint4 r[16];
  const uint4* src = in + (uint64_t)tile * kTileRecs;
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const uint4* q = src + i * 256 + threadIdx.x;
    if (LH == 0)
      r[i] = *q;
    else
      asm volatile("ld.global.L2::cache_hint.v4.u32 {%0,%1,%2,%3}, [%4], %5;"
                   : "=r"(r[i].x), "=r"(r[i].y), "=r"(r[i].z), "=r"(r[i].w)
                   : "l"(q), "l"(lpol));
  }
#pragma unroll
  for (int i = 0; i < 16; ++i) {
    const uint32_t j = i * 256 + threadIdx.x;
    const uint32_t c = j >> cr_shift, o = j & ((1u << cr_shift) - 1u);
    const uint32_t s = c % S, q = c / S;
    uint4* dst = out + (uint64_t)s * region + (((uint64_t)tile * per + q) << cr_shift) + o + sh;
    if (SH == 0)
      *dst = r[i];
    else
      asm volatile("st.global.L2::cache_hint.v4.b32 [%0], {%1,%2,%3,%4}, %5;" ::"l"(dst), "r"(r[i].x), "r"(r[i].y), "r"(r[i].z),
                   "r"(r[i].w), "l"(spol)
                   : "memory");
  }
}

// ---------------------------------------------------------------------------------------------------------------
// bulk: cp.async.bulk in and out
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t a = smem_u32(bar);
  uint32_t ok = 0, spins = 0;
  do {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok)
                 : "r"(a), "r"(parity)
                 : "memory");
    if (!ok && ++spins > (1u << 24)) __trap();  // never hang the device
  } while (!ok);
}
__device__ __forceinline__ void bulk_load(void* s, const void* g, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(s)),
               "l"(g), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
__device__ __forceinline__ void bulk_store(void* g, const void* s, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(g), "r"(smem_u32(s)), "r"(bytes) : "memory");
}

constexpr int kBulkStages = 3;
struct BulkSmem {
  uint4 buf[kBulkStages][kTileRecs];
  uint64_t full[kBulkStages];
  uint32_t tile_of[kBulkStages];
};

__global__ void __launch_bounds__(256, 1) bulk_copy(const uint4* in, uint4* out, uint32_t n_tiles, uint32_t S, uint32_t cr_shift,
                                                    uint32_t region, uint32_t sh, int ticketed, uint32_t* ticket,
                                                    unsigned long long* per_cta) {
  extern __shared__ __align__(128) unsigned char raw[];
  BulkSmem& sm = *reinterpret_cast<BulkSmem*>(raw);
  if (threadIdx.x == 0) {
    for (int s = 0; s < kBulkStages; ++s) mbar_init(&sm.full[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  const long long t0 = clock64();
  const uint32_t cpt = kTileRecs >> cr_shift, per = cpt / S;
  auto issue = [&](uint32_t it) {
    const uint32_t tile = ticketed ? atomicAdd(ticket, 1u) : blockIdx.x + it * gridDim.x;
    sm.tile_of[it % kBulkStages] = tile;
    if (tile < n_tiles) {
      mbar_expect_tx(&sm.full[it % kBulkStages], kTileRecs * 16u);
      bulk_load(sm.buf[it % kBulkStages], in + (uint64_t)tile * kTileRecs, kTileRecs * 16u, &sm.full[it % kBulkStages]);
    }
  };
  if (threadIdx.x == 0)
    for (uint32_t it = 0; it < kBulkStages; ++it) issue(it);
  __syncthreads();
  uint32_t done = 0;
  for (uint32_t k = 0;; ++k) {
    const uint32_t b = k % kBulkStages, ph = (k / kBulkStages) & 1u;
    const uint32_t tile = sm.tile_of[b];
    if (tile >= n_tiles) break;
    mbar_wait(&sm.full[b], ph);
    for (uint32_t c = threadIdx.x; c < cpt; c += 256) {
      const uint32_t s = c % S, q = c / S;
      bulk_store(out + (uint64_t)s * region + (((uint64_t)tile * per + q) << cr_shift) + sh, &sm.buf[b][c << cr_shift],
                 16u << cr_shift);
    }
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    __syncthreads();
    if (threadIdx.x == 0) issue(k + kBulkStages);
    __syncthreads();
    ++done;
  }
  asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  if (threadIdx.x == 0) {
    per_cta[2 * blockIdx.x] = (unsigned long long)(clock64() - t0);
    per_cta[2 * blockIdx.x + 1] = done;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// atomorder
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t mix(uint32_t x) {
  x ^= x >> 16;
  x *= 0x7feb352du;
  x ^= x >> 15;
  x *= 0x846ca68bu;
  x ^= x >> 16;
  return x;
}

__global__ void atom_order(unsigned long long* out /* [0] violations, [1] same-address lane pairs */, int iters,
                           uint32_t n_bins, uint32_t seed) {
  __shared__ uint32_t hist[32][256];
  const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int i = lane; i < 256; i += 32) hist[warp][i] = 0;
  __syncwarp();
  unsigned long long v = 0, pr = 0;
  for (int it = 0; it < iters; ++it) {
    const uint32_t d = mix(seed + (blockIdx.x * 1024u + threadIdx.x) * 7919u + it * 104729u) % n_bins;
    const uint32_t old = atomicAdd(&hist[warp][d], 1u);
    for (int l = 0; l < 32; ++l) {
      const uint32_t dl = __shfl_sync(0xffffffffu, d, l);
      const uint32_t ol = __shfl_sync(0xffffffffu, old, l);
      if (dl == d && l < (int)lane) {
        pr++;
        if (!(ol < old)) v++;
      }
    }
  }
  atomicAdd(out, v);
  atomicAdd(out + 1, pr);
}

// ---------------------------------------------------------------------------------------------------------------
// red: scattered fp32 reductions into a small L2-resident array
// ---------------------------------------------------------------------------------------------------------------
__global__ void fill_targets(uint32_t* tgt, float* w, uint32_t n, uint32_t n_nodes) {
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
    tgt[i] = mix(i * 2654435761u + 99u) % n_nodes;
    w[i] = 1.0f;
  }
}
__global__ void __launch_bounds__(256) red_kernel(const uint32_t* __restrict__ tgt, const float* __restrict__ w, uint32_t n,
                                                  float* __restrict__ acc) {
  for (uint32_t i = blockIdx.x * 256u + threadIdx.x; i < n; i += gridDim.x * 256u) atomicAdd(acc + tgt[i], w[i]);
}

// ---------------------------------------------------------------------------------------------------------------
// pipes: N independent chains of one instruction per thread, timed with clock64 by every warp; the figure printed is
// cycles per warp instruction per SM sub-partition with `warps` resident warps per sub-partition.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kChains = 8, kPipeIters = 2048;

template <int OP>
__global__ void pipe_rate(uint32_t* sink, unsigned long long* cycles, uint32_t a0) {
  uint32_t x[kChains], y[kChains];
  float f[kChains];
#pragma unroll
  for (int c = 0; c < kChains; ++c) {
    x[c] = a0 + threadIdx.x * 31u + c;
    y[c] = a0 ^ (c * 977u);
    f[c] = (float)(threadIdx.x + c);
  }
  __syncthreads();
  const long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < kPipeIters; ++it) {
#pragma unroll
    for (int c = 0; c < kChains; ++c) {
      if (OP == 0) {  // IMAD.WIDE.U32 (the Philox multiply); the low half feeds the next one
        uint64_t p;
        asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(x[c]), "r"(0xD2511F53u));
        x[c] = (uint32_t)p;
        y[c] = (uint32_t)(p >> 32);
      } else if (OP == 1) {  // IMAD (32-bit multiply-add)
        asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(x[c]) : "r"(0x9E3779B1u), "r"(y[c]));
      } else if (OP == 2) {  // LOP3 (three-input xor)
        asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[c]) : "r"(y[c]), "r"(a0));
      } else if (OP == 3) {  // FFMA
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[c]) : "f"(1.0000001f), "f"(0.5f));
      } else {  // Philox round: 2 IMAD.WIDE + 2 LOP3
        uint64_t p0, p1;
        asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p0) : "r"(x[c]), "r"(0xD2511F53u));
        asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p1) : "r"(y[c]), "r"(0xCD9E8D57u));
        asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[c]) : "r"((uint32_t)(p1 >> 32)), "r"((uint32_t)p0), "r"(a0));
        asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(y[c]) : "r"((uint32_t)(p0 >> 32)), "r"((uint32_t)p1), "r"(a0));
      }
    }
  }
  const long long t1 = clock64();
  uint32_t acc = 0;
#pragma unroll
  for (int c = 0; c < kChains; ++c) acc += x[c] + y[c] + __float_as_uint(f[c]);
  if (acc == 0x12345678u) sink[0] = acc;
  if ((threadIdx.x & 31) == 0) atomicMax(cycles + blockIdx.x, (unsigned long long)(t1 - t0));
}

}  // namespace

int main(int argc, char** argv) {
  const char* what = argc > 1 ? argv[1] : "all";
  const bool all = !strcmp(what, "all");
  cudaDeviceProp prop;
  CK(cudaGetDeviceProperties(&prop, 0));
  printf("# membench on %s, %d SMs\n", prop.name, prop.multiProcessorCount);
  Timer t;

  if (all || !strcmp(what, "pattern") || !strcmp(what, "bulk")) {
    const uint32_t n_tiles = 72960;  // 298.8e6 records of 16 bytes: the size of one configs[2] digit pass
    const uint64_t n = (uint64_t)n_tiles * kTileRecs;
    uint4 *in, *out;
    CK(cudaMalloc(&in, n * 16));
    CK(cudaMalloc(&out, n * 16 + (1 << 20)));
    CK(cudaMemset(in, 1, n * 16));
    float ms = 0;
    for (int r = 0; r < 2; ++r) {
      t.start();
      CK(cudaMemcpyAsync(out, in, n * 16, cudaMemcpyDeviceToDevice));
      ms = t.stop();
    }
    printf("\n## copy of %.2f GB (read + write %.2f GB)\ncudaMemcpy device to device: %.3f ms  %.0f GB/s\n", n * 16e-9,
           n * 32e-9, ms, 32.0 * n / ms * 1e-6);
    if (all || !strcmp(what, "pattern")) {
      printf("\n## pattern: LSU copy, 16 records per thread, one 64 KB tile per CTA (R tiles when R > 1)\n");
      printf("| piece B | streams | start offset B | R | ms | GB/s |\n|---|---|---|---|---|---|\n");
      struct Case {
        uint32_t cr_shift, S, sh, R;
      };
      const Case cases[] = {{4, 256, 0, 1}, {4, 256, 2, 1}, {4, 256, 4, 1}, {4, 256, 1, 1}, {4, 256, 3, 1}, {4, 16, 1, 1},
                            {4, 64, 1, 1},  {4, 128, 1, 1}, {5, 128, 0, 1}, {5, 128, 1, 1}, {6, 64, 0, 1},  {6, 64, 1, 1},
                            {3, 256, 0, 1}, {3, 256, 1, 1}, {4, 256, 1, 2}, {4, 256, 1, 4}, {4, 256, 1, 16},
                            {4, 256, 2, 8}, {4, 256, 0, 8}, {0, 256, 0, 1}, {1, 256, 0, 1}, {2, 256, 1, 1}};
      for (const Case& c : cases) {
        float best = 1e9f;
        for (int r = 0; r < 4; ++r) {
          t.start();
          pattern_copy<<<(n_tiles + c.R - 1) / c.R, 256>>>(in, out, n_tiles, c.S, c.cr_shift, (uint32_t)(n / c.S), c.sh, c.R);
          best = fminf(best, t.stop());
        }
        CK(cudaGetLastError());
        printf("| %u | %u | %u | %u | %.3f | %.0f |\n", 16u << c.cr_shift, c.S, c.sh * 16, c.R, best, 32.0 * n / best * 1e-6);
      }
    }
    if (all || !strcmp(what, "bulk")) {
      printf("\n## bulk: cp.async.bulk load of a tile + one bulk store per piece, 148 persistent CTAs, 3 tile buffers\n");
      printf("| piece B | streams | start offset B | tiles | ms | GB/s | CTA kcycles min..max | tiles per CTA min..max |\n"
             "|---|---|---|---|---|---|---|---|\n");
      uint32_t* ticket;
      unsigned long long* per_cta;
      CK(cudaMalloc(&ticket, 4));
      CK(cudaMalloc(&per_cta, 148 * 16));
      CK(cudaFuncSetAttribute(bulk_copy, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(BulkSmem)));
      struct Case {
        uint32_t cr_shift, S, sh;
        int ticketed;
      };
      const Case cases[] = {{12, 1, 0, 0}, {12, 1, 0, 1}, {4, 256, 0, 0}, {4, 256, 0, 1}, {4, 256, 1, 0}, {4, 256, 1, 1}, {4, 16, 1, 1}};
      for (const Case& c : cases) {
        float best = 1e9f;
        for (int r = 0; r < 3; ++r) {
          CK(cudaMemset(ticket, 0, 4));
          t.start();
          bulk_copy<<<148, 256, sizeof(BulkSmem)>>>(in, out, n_tiles, c.S, c.cr_shift, (uint32_t)(n / c.S), c.sh, c.ticketed, ticket,
                                                    per_cta);
          best = fminf(best, t.stop());
        }
        CK(cudaGetLastError());
        unsigned long long h[296];
        CK(cudaMemcpy(h, per_cta, sizeof(h), cudaMemcpyDeviceToHost));
        unsigned long long mn = ~0ull, mx = 0, tmn = ~0ull, tmx = 0;
        for (int q = 0; q < 148; ++q) {
          mn = h[2 * q] < mn ? h[2 * q] : mn;
          mx = h[2 * q] > mx ? h[2 * q] : mx;
          tmn = h[2 * q + 1] < tmn ? h[2 * q + 1] : tmn;
          tmx = h[2 * q + 1] > tmx ? h[2 * q + 1] : tmx;
        }
        printf("| %u | %u | %u | %s | %.3f | %.0f | %llu..%llu | %llu..%llu |\n", 16u << c.cr_shift, c.S, c.sh * 16,
               c.ticketed ? "ticketed" : "static", best, 32.0 * n / best * 1e-6, mn / 1000, mx / 1000, tmn, tmx);
      }
      cudaFree(ticket);
      cudaFree(per_cta);
    }
    cudaFree(in);
    cudaFree(out);
  }

  if (all || !strcmp(what, "ring")) {
    const uint32_t n_tiles = 72960;
    const uint64_t n = (uint64_t)n_tiles * kTileRecs;
    uint4 *in, *tmp, *out;
    CK(cudaMalloc(&in, n * 16));
    CK(cudaMalloc(&tmp, n * 16 + (1 << 20)));
    CK(cudaMalloc(&out, n * 16 + (1 << 20)));
    CK(cudaMemset(in, 1, n * 16));
    printf("\n## ring: two passes over %.2f GB (pass 1: 256 B pieces into 256 streams, pass 2: 512 B pieces into 128 streams, every piece\n"
           "## starting 16 B into a sector), whole-array launches against per-group launches; 'ring' = the intermediate array is one\n"
           "## slot per CUDA stream, reused by every group, 'full' = every group has its own part of a full-size intermediate array\n",
           n * 16e-9);
    printf("| group MB | CUDA streams | intermediate | hints (load 1, store 1, load 2, store 2) | ms | GB/s of 64 B per record |\n|---|---|---|---|---|---|\n");
    {
      float best = 1e9f;
      for (int r = 0; r < 3; ++r) {
        t.start();
        pattern_copy_hint<0, 0><<<n_tiles, 256>>>(in, tmp, n_tiles, 256, 4, (uint32_t)(n / 256), 1);
        pattern_copy_hint<0, 0><<<n_tiles, 256>>>(tmp, out, n_tiles, 128, 5, (uint32_t)(n / 128), 1);
        best = fminf(best, t.stop());
      }
      CK(cudaGetLastError());
      printf("| whole array | 1 | full | none | %.3f | %.0f |\n", best, 64.0 * n / best * 1e-6);
    }
    cudaStream_t st[4];
    cudaEvent_t fork, join[4];
    CK(cudaEventCreateWithFlags(&fork, cudaEventDisableTiming));
    for (int q = 0; q < 4; ++q) {
      CK(cudaStreamCreateWithFlags(&st[q], cudaStreamNonBlocking));
      CK(cudaEventCreateWithFlags(&join[q], cudaEventDisableTiming));
    }
    struct Case {
      uint32_t gt;  // tiles per group
      int ns, ring, hints;
    };
    // hints: 0 = none; else decimal digits (load 1, store 1, load 2, store 2), 0 none / 1 evict_first / 2 evict_last
    const Case cases[] = {{512, 2, 0, 0},    {512, 2, 1, 0},    {512, 2, 1, 1211}, {512, 2, 1, 1221}, {512, 2, 1, 1201},
                          {512, 2, 1, 1210}, {512, 2, 1, 210},  {512, 2, 1, 1200}, {512, 2, 0, 1211}, {256, 2, 0, 0},
                          {256, 2, 1, 0},    {256, 2, 1, 1211}, {256, 3, 1, 1211}, {256, 3, 1, 1221}, {256, 3, 1, 1201},
                          {128, 4, 1, 1211}, {768, 2, 1, 1211}, {1024, 2, 1, 1211}, {256, 1, 1, 1211}};
    for (const Case& c : cases) {
      float best = 1e9f;
      for (int r = 0; r < 3; ++r) {
        t.start();
        CK(cudaEventRecord(fork, 0));
        for (int q = 0; q < c.ns; ++q) CK(cudaStreamWaitEvent(st[q], fork, 0));
        uint32_t g = 0;
        for (uint32_t t0 = 0; t0 < n_tiles; t0 += c.gt, ++g) {
          const uint32_t gt = n_tiles - t0 < c.gt ? n_tiles - t0 : c.gt;
          const int q = g % c.ns;
          const uint64_t recs = (uint64_t)gt * kTileRecs;
          const uint4* gin = in + (uint64_t)t0 * kTileRecs;
          uint4* gtmp = c.ring ? tmp + (uint64_t)q * ((uint64_t)c.gt * kTileRecs + 4096) : tmp + (uint64_t)t0 * kTileRecs;
          uint4* gout = out + (uint64_t)t0 * kTileRecs;
          const uint32_t r1 = (uint32_t)(recs / 256), r2 = (uint32_t)(recs / 128);
#define NC_P1(L, S) pattern_copy_hint<L, S><<<gt, 256, 0, st[q]>>>(gin, gtmp, gt, 256, 4, r1, 1)
#define NC_P2(L, S) pattern_copy_hint<L, S><<<gt, 256, 0, st[q]>>>(gtmp, gout, gt, 128, 5, r2, 1)
          switch (c.hints / 100) {
            case 12: NC_P1(1, 2); break;
            case 2: NC_P1(0, 2); break;
            default: NC_P1(0, 0); break;
          }
          switch (c.hints % 100) {
            case 11: NC_P2(1, 1); break;
            case 21: NC_P2(2, 1); break;
            case 1: NC_P2(0, 1); break;
            case 10: NC_P2(1, 0); break;
            default: NC_P2(0, 0); break;
          }
#undef NC_P1
#undef NC_P2
        }
        for (int q = 0; q < c.ns; ++q) {
          CK(cudaEventRecord(join[q], st[q]));
          CK(cudaStreamWaitEvent(0, join[q], 0));
        }
        best = fminf(best, t.stop());
      }
      CK(cudaGetLastError());
      const char* hn[] = {"none", "evict_first", "evict_last"};
      printf("| %u | %d | %s | %s, %s, %s, %s | %.3f | %.0f |\n", c.gt / 16, c.ns, c.ring ? "ring" : "full", hn[c.hints / 1000],
             hn[c.hints / 100 % 10], hn[c.hints / 10 % 10], hn[c.hints % 10], best, 64.0 * n / best * 1e-6);
    }
    for (int q = 0; q < 4; ++q) {
      cudaStreamDestroy(st[q]);
      cudaEventDestroy(join[q]);
    }
    cudaEventDestroy(fork);
    cudaFree(in);
    cudaFree(tmp);
    cudaFree(out);
  }

  if (all || !strcmp(what, "atomorder")) {
    printf("\n## atomorder: old values of same-address shared atomicAdd lanes of one warp instruction, 296 CTAs x 32 warps\n");
    printf("| bins | same-address lane pairs | pairs not in ascending lane order |\n|---|---|---|\n");
    unsigned long long *d, h[2], total = 0;
    CK(cudaMalloc(&d, 16));
    for (uint32_t nb : {1u, 2u, 8u, 32u, 256u}) {
      CK(cudaMemset(d, 0, 16));
      atom_order<<<296, 1024>>>(d, 1000, nb, nb * 17u + 1u);
      CK(cudaMemcpy(h, d, 16, cudaMemcpyDeviceToHost));
      CK(cudaGetLastError());
      printf("| %u | %llu | %llu |\n", nb, h[1], h[0]);
      total += h[0];
    }
    printf("atomorder violations total: %llu\n", total);
    cudaFree(d);
  }

  if (all || !strcmp(what, "red")) {
    printf("\n## red: n x (4 B target + 4 B weight read, one red.global.add.f32) into 77,169 accumulators\n");
    printf("| events | us | events/s | GB/s of the 8 B per event |\n|---|---|---|---|\n");
    const uint32_t n_nodes = 77169, n_max = 1u << 26;
    uint32_t* tgt;
    float *w, *acc;
    CK(cudaMalloc(&tgt, (size_t)n_max * 4));
    CK(cudaMalloc(&w, (size_t)n_max * 4));
    CK(cudaMalloc(&acc, n_nodes * 4));
    CK(cudaMemset(acc, 0, n_nodes * 4));
    fill_targets<<<1184, 256>>>(tgt, w, n_max, n_nodes);
    for (uint32_t n : {240000u, 3000000u, 15000000u, 1u << 26}) {
      float best = 1e9f;
      for (int r = 0; r < 5; ++r) {
        t.start();
        red_kernel<<<(n + 255) / 256 < 148 * 8 ? (n + 255) / 256 : 148 * 8, 256>>>(tgt, w, n, acc);
        best = fminf(best, t.stop());
      }
      CK(cudaGetLastError());
      printf("| %u | %.1f | %.3g | %.0f |\n", n, best * 1e3, n / (best * 1e-3), 8.0 * n / best * 1e-6);
    }
    cudaFree(tgt);
    cudaFree(w);
    cudaFree(acc);
  }

  if (all || !strcmp(what, "pipes")) {
    printf("\n## pipes: cycles per warp instruction per SM sub-partition (148 CTAs, %d independent chains per thread)\n", kChains);
    printf("| instruction | 2 warps / sub-partition | 4 warps | 8 warps |\n|---|---|---|---|\n");
    uint32_t* sink;
    unsigned long long* cyc;
    CK(cudaMalloc(&sink, 4));
    CK(cudaMalloc(&cyc, 148 * 8));
    const char* names[] = {"IMAD.WIDE.U32 (32x32->64, both halves used)", "IMAD (32-bit multiply-add)", "LOP3", "FFMA",
                           "Philox round (2 IMAD.WIDE + 2 LOP3)"};
    for (int op = 0; op < 5; ++op) {
      printf("| %s |", names[op]);
      for (int wps : {2, 4, 8}) {
        const int threads = wps * 4 * 32;
        const int ctas_per_sm = 1;
        unsigned long long* cyc2;
        CK(cudaMalloc(&cyc2, 148 * ctas_per_sm * 8));
        CK(cudaMemset(cyc2, 0, 148 * ctas_per_sm * 8));
        for (int r = 0; r < 2; ++r) {
          switch (op) {
            case 0: pipe_rate<0><<<148 * ctas_per_sm, threads>>>(sink, cyc2, 12345u); break;
            case 1: pipe_rate<1><<<148 * ctas_per_sm, threads>>>(sink, cyc2, 12345u); break;
            case 2: pipe_rate<2><<<148 * ctas_per_sm, threads>>>(sink, cyc2, 12345u); break;
            case 3: pipe_rate<3><<<148 * ctas_per_sm, threads>>>(sink, cyc2, 12345u); break;
            default: pipe_rate<4><<<148 * ctas_per_sm, threads>>>(sink, cyc2, 12345u); break;
          }
          CK(cudaDeviceSynchronize());
        }
        unsigned long long h[148 * 2];
        CK(cudaMemcpy(h, cyc2, 148 * ctas_per_sm * 8, cudaMemcpyDeviceToHost));
        double sum = 0;
        for (int q = 0; q < 148 * ctas_per_sm; ++q) sum += (double)h[q];
        const double mean_cycles = sum / (148 * ctas_per_sm);
        // warp instructions one sub-partition issued: wps warps x kPipeIters x kChains (x instructions per chain step)
        const double per_step = op == 4 ? 4.0 : 1.0;
        printf(" %.2f |", mean_cycles / (wps * (double)kPipeIters * kChains * per_step));
        cudaFree(cyc2);
      }
      printf("\n");
    }
    cudaFree(sink);
    cudaFree(cyc);
  }
  return 0;
}
