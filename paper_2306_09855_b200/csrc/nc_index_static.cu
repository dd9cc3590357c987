// nc_index_static.cu -- nc_index_static (include/nc_static.h): the group index of PAPER.md:121-132 over organised connections
// for callers that cannot allocate device memory where they need it (a loop with a latency budget, where cudaMalloc /
// cudaFree would stall every stream of the process; a process whose own pool already owns the whole card, where a
// library's cudaMalloc just fails; code that may only touch the buffers and the stream it was handed).
//
// The kernel is the single-read index of nc_index.cuh (index_fused_kernel: a tile counts its group heads, chains the count
// to the tiles before it by decoupled look-back, and writes the index from the keys it still holds in registers), restated
// here with a capacity check on the group arrays.  Its scratch -- one status word per tile and a tile ticket -- does not come
// from an allocator: it is the file-scope device array below, which is part of the library image.  Consequences:
//   * every GPU that loads libnc.so holds kScratchWords * 8 bytes for this from module load to process exit;
//   * n is limited to kMaxTiles tiles (NC_INDEX_STATIC_MAX_CONNECTIONS);
//   * all calls on a device share the one array: each call clears what it uses on its own stream first, and calls that
//     overlap on the GPU race (the caller orders them);
//   * in HOST code the name g_index_scratch is only a handle for the runtime, not a device address.  The address the kernel
//     gets is looked up once per device with cudaGetSymbolAddress while that device is current (scratch_of_current_device).
// Nothing in this file calls cudaMalloc, cudaFree, or a library routine that allocates; nothing here is used by nc_finalize.
#include "../../include/nc_static.h"

#include <cuda_runtime.h>

#include <cstdio>
#include <cstring>
#include <mutex>

#include "nc_common.cuh"

using namespace nc;

namespace {

constexpr int kThreads = 1024;  // one CTA per SM is resident: a look-back seldom walks further than the tiles in flight
constexpr int kChunks = 2;      // chunks of 8 consecutive positions per thread
constexpr uint32_t kTile = kThreads * 8 * kChunks;  // 16,384 positions
constexpr uint64_t kMaxTiles = NC_INDEX_STATIC_MAX_CONNECTIONS / kTile;
constexpr uint64_t kScratchWords = kMaxTiles + 32;  // [kMaxTiles] status words | ticket (first word of the tail)
static_assert(kScratchWords * 8 == NC_INDEX_STATIC_SCRATCH_BYTES, "nc_static.h states the size of the scratch array");
static_assert(NC_INDEX_STATIC_MAX_CONNECTIONS % kTile == 0, "whole tiles");

// The scratch memory itself.  Device code may name it directly; host code must not pass this name to a kernel.
static __device__ __align__(256) unsigned long long g_index_scratch[kScratchWords];

// status word of a tile: bits 0..31 group heads | bit 32 = this tile's own count is there | bit 33 = count of all tiles up
// to and including this one is there
constexpr uint64_t kOwn = 1ull << 32, kInclusive = 2ull << 32;

struct Out {
  uint32_t* src_offsets;  // [n_nodes + 1]
  uint32_t* group_ptr;    // [n_nodes + 1]
  uint32_t* group_start;  // [group_capacity]
  uint16_t* group_delay;  // [group_capacity]
  uint32_t* total_groups;
  uint32_t* error;
  uint32_t group_capacity;
  uint32_t n_nodes;
};

__device__ __forceinline__ uint32_t cta_exclusive_scan(uint32_t v, uint32_t* warp_tmp /*[kThreads / 32]*/, uint32_t& total) {
  uint32_t inc = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, inc, d);
    if (lane_id() >= (uint32_t)d) inc += t;
  }
  __syncthreads();  // warp_tmp may still be read by the previous scan
  if (lane_id() == 31) warp_tmp[threadIdx.x >> 5] = inc;
  __syncthreads();
  uint32_t base = 0, tot = 0;
#pragma unroll
  for (uint32_t w = 0; w < kThreads / 32; ++w) {
    const uint32_t t = warp_tmp[w];
    if (w < (threadIdx.x >> 5)) base += t;
    tot += t;
  }
  total = tot;
  return base + inc - v;
}

// A head is a connection whose source or delay differs from the one before it; head number g starts group
// g.  The first head of source s also closes the entries of the nodes between the previous source and s (they have no
// outgoing connection): src_offsets = position, group_ptr = g, which is Eq. 14 written as a scatter.
__global__ void __launch_bounds__(kThreads) index_static_kernel(const uint32_t* __restrict__ src,
                                                               const uint16_t* __restrict__ dly, uint32_t n,
                                                               uint64_t* __restrict__ status, uint32_t* __restrict__ ticket,
                                                               const __grid_constant__ Out out) {
  __shared__ uint32_t warp_tmp[kThreads / 32];
  __shared__ uint32_t sh_tile, sh_prefix;
  // tiles are handed out in the order CTAs start, so a tile only ever waits for tiles that are already running
  if (threadIdx.x == 0) sh_tile = atomicAdd(ticket, 1u);
  __syncthreads();
  const uint32_t tile = sh_tile;
  uint32_t s[kChunks][9], d[kChunks][9], cnt[kChunks], heads[kChunks], first_src[kChunks];
#pragma unroll
  for (int c = 0; c < kChunks; ++c) {
    // chunk c: thread t owns positions tile * kTile + c * 8 * kThreads + t * 8 .. + 7; [0] is the position before them
    const uint64_t base64 = (uint64_t)tile * kTile + (uint64_t)c * (kThreads * 8) + threadIdx.x * 8u;
    const uint32_t base = (uint32_t)base64;
    const bool in_range = base64 < n;
#pragma unroll
    for (int i = 0; i < 9; ++i) s[c][i] = d[c][i] = 0;
    cnt[c] = 0;
    if (in_range) {
      if (n - base >= 8u) {
        const uint4 s0 = *reinterpret_cast<const uint4*>(src + base);
        const uint4 s1 = *reinterpret_cast<const uint4*>(src + base + 4);
        const uint4 dd = *reinterpret_cast<const uint4*>(dly + base);
        s[c][1] = s0.x; s[c][2] = s0.y; s[c][3] = s0.z; s[c][4] = s0.w;
        s[c][5] = s1.x; s[c][6] = s1.y; s[c][7] = s1.z; s[c][8] = s1.w;
        d[c][1] = dd.x & 0xffffu; d[c][2] = dd.x >> 16; d[c][3] = dd.y & 0xffffu; d[c][4] = dd.y >> 16;
        d[c][5] = dd.z & 0xffffu; d[c][6] = dd.z >> 16; d[c][7] = dd.w & 0xffffu; d[c][8] = dd.w >> 16;
        cnt[c] = 8;
      } else {
        cnt[c] = n - base;
#pragma unroll
        for (int i = 0; i < 8; ++i)
          if ((uint32_t)i < cnt[c]) {
            s[c][i + 1] = src[base + i];
            d[c][i + 1] = dly[base + i];
          }
      }
    }
    const uint32_t up_s = __shfl_up_sync(0xffffffffu, s[c][8], 1), up_d = __shfl_up_sync(0xffffffffu, d[c][8], 1);
    s[c][0] = up_s;
    d[c][0] = up_d;
    if (lane_id() == 0 && in_range && base > 0) {
      s[c][0] = src[base - 1];
      d[c][0] = dly[base - 1];
    }
    uint32_t h = 0, f = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const bool new_s = s[c][i + 1] != s[c][i];
      if (new_s | (d[c][i + 1] != d[c][i])) h |= 1u << i;
      if (new_s) f |= 1u << i;
    }
    if (in_range && base == 0) {  // position 0 starts a group and a source whatever its key
      h |= 1u;
      f |= 1u;
    }
    const uint32_t live = cnt[c] >= 8 ? 0xffu : ((1u << cnt[c]) - 1u);
    heads[c] = h & live;
    first_src[c] = f & live;
  }
  // exclusive scan in POSITION order: chunk 0 of every thread lies before chunk 1 of any thread
  static_assert(kChunks == 2, "the scan below is written for two chunks");
  uint32_t tot0, tot1;
  const uint32_t ex0 = cta_exclusive_scan(__popc(heads[0]), warp_tmp, tot0);
  const uint32_t ex1 = cta_exclusive_scan(__popc(heads[1]), warp_tmp, tot1) + tot0;
  const uint32_t tile_total = tot0 + tot1;

  // ---- heads in the tiles before this one: warp 0 polls 32 predecessors per load ----
  if (threadIdx.x < 32) {
    uint64_t* mine_w = status + tile;
    uint32_t excl = 0;
    if (tile == 0) {
      if (threadIdx.x == 0) st_relaxed_u64(mine_w, kInclusive | tile_total);
    } else {
      if (threadIdx.x == 0) st_relaxed_u64(mine_w, kOwn | tile_total);
      int64_t t = (int64_t)tile - 1;
      uint32_t spins = 0;
      while (true) {
        const int64_t look = t - (int64_t)lane_id();
        const uint64_t w = look >= 0 ? ld_relaxed_u64(status + look) : kInclusive;  // before tile 0: nothing
        const uint32_t ready = __ballot_sync(0xffffffffu, (w >> 32) != 0);
        const uint32_t incl = __ballot_sync(0xffffffffu, (w >> 33) != 0);
        // usable: the unbroken run of published predecessors from lane 0 on, cut after the first inclusive one
        uint32_t usable = ready == 0xffffffffu ? 32u : (uint32_t)__ffs(~ready) - 1u;
        const uint32_t first_incl = incl ? (uint32_t)__ffs(incl) - 1u : 32u;
        const bool done = first_incl < usable;
        if (done) usable = first_incl + 1;
        uint32_t v = lane_id() < usable ? (uint32_t)w : 0u;
        v = __reduce_add_sync(0xffffffffu, v);
        excl += v;
        if (done) break;
        t -= usable;
        if (usable == 0) {
          if (++spins > (1u << 22)) {  // report a lost predecessor instead of hanging the device
            if (lane_id() == 0) atomicOr(out.error, (uint32_t)NC_INDEX_STATIC_LOOKBACK);
            break;
          }
          __nanosleep(20);
        }
      }
      if (threadIdx.x == 0) st_relaxed_u64(mine_w, kInclusive | (uint64_t)(excl + tile_total));
    }
    if (threadIdx.x == 0) sh_prefix = excl;
  }
  __syncthreads();
  const uint32_t prefix = sh_prefix;
  const uint64_t tile_first = (uint64_t)tile * kTile;
  if (threadIdx.x == 0 && tile_first < n && tile_first + kTile >= n) *out.total_groups = prefix + tile_total;  // last tile

  bool overflow = false;
#pragma unroll
  for (int c = 0; c < kChunks; ++c) {
    const uint32_t base = tile * kTile + (uint32_t)c * (kThreads * 8) + threadIdx.x * 8u;
    uint32_t g = prefix + (c == 0 ? ex0 : ex1);
    uint32_t m = heads[c];
    while (m) {
      const int i = __ffs(m) - 1;
      m &= m - 1;
      const uint32_t j = base + i;
      uint32_t si = s[c][1], di = d[c][1], sp = s[c][0];
#pragma unroll
      for (int q = 1; q < 8; ++q)
        if (i == q) {
          si = s[c][q + 1];
          di = d[c][q + 1];
          sp = s[c][q];
        }
      if (g < out.group_capacity) {
        out.group_start[g] = j;
        out.group_delay[g] = (uint16_t)di;
      } else {
        overflow = true;
      }
      if (first_src[c] & (1u << i)) {
        const uint32_t lo = j == 0 ? 0u : sp + 1u;
        for (uint32_t node = lo; node <= si; ++node) {
          out.src_offsets[node] = j;
          out.group_ptr[node] = g;
        }
      }
      ++g;
    }
    if (cnt[c] > 0 && base + cnt[c] == n) {  // the last connection: nodes after its source, and the closing entries
      uint32_t sl = s[c][1];
#pragma unroll
      for (int q = 1; q < 8; ++q)
        if (cnt[c] == (uint32_t)q + 1) sl = s[c][q + 1];
      const uint32_t tg = prefix + tile_total;
      for (uint64_t node = (uint64_t)sl + 1; node <= out.n_nodes; ++node) {
        out.src_offsets[node] = n;
        out.group_ptr[node] = tg;
      }
    }
  }
  if (overflow) atomicOr(out.error, (uint32_t)NC_INDEX_STATIC_GROUPS);
}

// G_s = p_{s+1} - p_s
__global__ void __launch_bounds__(256) group_count_static_kernel(const uint32_t* __restrict__ group_ptr, uint32_t n_nodes,
                                                                uint32_t* __restrict__ group_count) {
  const uint64_t stride = (uint64_t)gridDim.x * 256u;
  for (uint64_t s = (uint64_t)blockIdx.x * 256u + threadIdx.x; s < n_nodes; s += stride) group_count[s] = group_ptr[s + 1] - group_ptr[s];
}

// ---- set-up: the device address of the scratch array, once per device ----
constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
unsigned long long* g_scratch_of[kMaxDevices] = {};

int fail_static(int code, char* err_msg, size_t err_cap, const char* what, cudaError_t e = cudaSuccess) {
  if (err_msg && err_cap) {
    if (e != cudaSuccess) snprintf(err_msg, err_cap, "nc_index_static: %s: %s", what, cudaGetErrorString(e));
    else snprintf(err_msg, err_cap, "nc_index_static: %s", what);
  }
  if (e != cudaSuccess) cudaGetLastError();  // leave no stale error for the caller's next check
  return code;
}

// Looks the address up with the CURRENT device current: a __device__ array exists once per device, each with its own
// address, and cudaGetSymbolAddress answers for the device that is current when it is called.
int scratch_of_current_device(unsigned long long** out, char* err_msg, size_t err_cap) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail_static(NC_ERR_CUDA, err_msg, err_cap, "cudaGetDevice", e);
  if (dev < 0 || dev >= kMaxDevices) return fail_static(NC_ERR_CAPACITY, err_msg, err_cap, "device ordinal above 63");
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_scratch_of[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_index_scratch);
    if (e != cudaSuccess || !p)
      return fail_static(NC_ERR_CUDA, err_msg, err_cap, "cudaGetSymbolAddress of the scratch array", e);
    g_scratch_of[dev] = static_cast<unsigned long long*>(p);
  }
  *out = g_scratch_of[dev];
  return NC_OK;
}

}  // namespace

extern "C" int nc_index_static(const uint32_t* d_source, const uint16_t* d_delay, uint64_t n, uint32_t n_nodes,
                               uint32_t* d_src_offsets, uint32_t* d_group_ptr, uint32_t* d_group_count,
                               uint32_t* d_group_start, uint16_t* d_group_delay, uint64_t group_capacity,
                               uint32_t* d_total_groups, uint32_t* d_error, void* cuda_stream, char* err_msg,
                               size_t err_cap) {
  if (n > NC_INDEX_STATIC_MAX_CONNECTIONS) {
    char what[256];
    snprintf(what, sizeof(what),
             "%llu connections are more than the %llu the built-in scratch array is sized for "
             "(NC_INDEX_STATIC_MAX_CONNECTIONS); use nc_finalize, which allocates",
             (unsigned long long)n, (unsigned long long)NC_INDEX_STATIC_MAX_CONNECTIONS);
    return fail_static(NC_ERR_CAPACITY, err_msg, err_cap, what);
  }
  if (!d_src_offsets || !d_group_ptr || !d_total_groups || !d_error)
    return fail_static(NC_ERR_INVALID_ARG, err_msg, err_cap, "d_src_offsets, d_group_ptr, d_total_groups and d_error must not be NULL");
  if (n > 0) {
    if (!d_source || !d_delay) return fail_static(NC_ERR_INVALID_ARG, err_msg, err_cap, "d_source / d_delay is NULL");
    if (((uintptr_t)d_source | (uintptr_t)d_delay) & 15u)
      return fail_static(NC_ERR_INVALID_ARG, err_msg, err_cap, "d_source and d_delay must be aligned to 16 bytes");
    if (n_nodes == 0) return fail_static(NC_ERR_INVALID_ARG, err_msg, err_cap, "connections without nodes");
    if (group_capacity > 0 && (!d_group_start || !d_group_delay))
      return fail_static(NC_ERR_INVALID_ARG, err_msg, err_cap, "group_capacity > 0 with a NULL group array");
  }
  unsigned long long* scratch = nullptr;
  const int rc = scratch_of_current_device(&scratch, err_msg, err_cap);  // first call on this device: the set-up
  if (rc != NC_OK) return rc;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  cudaError_t e = cudaMemsetAsync(d_error, 0, 4, stream);
  if (e != cudaSuccess) return fail_static(NC_ERR_CUDA, err_msg, err_cap, "clearing d_error", e);
  if (n == 0) {  // no connection, no group: every offset is 0
    e = cudaMemsetAsync(d_total_groups, 0, 4, stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_src_offsets, 0, ((size_t)n_nodes + 1) * 4, stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(d_group_ptr, 0, ((size_t)n_nodes + 1) * 4, stream);
    if (e == cudaSuccess && d_group_count && n_nodes) e = cudaMemsetAsync(d_group_count, 0, (size_t)n_nodes * 4, stream);
    if (e != cudaSuccess) return fail_static(NC_ERR_CUDA, err_msg, err_cap, "clearing the outputs of an empty index", e);
    return NC_OK;
  }
  const uint64_t tiles = (n + kTile - 1) / kTile;
  // The array still holds the previous call's status words and ticket: what this call uses must start at zero.
  e = cudaMemsetAsync(scratch, 0, tiles * 8, stream);
  if (e == cudaSuccess) e = cudaMemsetAsync(scratch + kMaxTiles, 0, 8, stream);
  if (e != cudaSuccess) return fail_static(NC_ERR_CUDA, err_msg, err_cap, "clearing the scratch array", e);
  Out out{d_src_offsets, d_group_ptr, d_group_start, d_group_delay, d_total_groups, d_error,
          (uint32_t)(group_capacity > n ? n : group_capacity), n_nodes};
  index_static_kernel<<<(unsigned)tiles, kThreads, 0, stream>>>(d_source, d_delay, (uint32_t)n,
                                                                 reinterpret_cast<uint64_t*>(scratch),
                                                                 reinterpret_cast<uint32_t*>(scratch + kMaxTiles), out);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail_static(NC_ERR_CUDA, err_msg, err_cap, "launching index_static_kernel", e);
  if (d_group_count) {
    const unsigned grid = (unsigned)((n_nodes + 255ull) / 256ull < 148ull * 16 ? (n_nodes + 255ull) / 256ull : 148ull * 16);
    group_count_static_kernel<<<grid, 256, 0, stream>>>(d_group_ptr, n_nodes, d_group_count);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail_static(NC_ERR_CUDA, err_msg, err_cap, "launching group_count_static_kernel", e);
  }
  return NC_OK;
}
