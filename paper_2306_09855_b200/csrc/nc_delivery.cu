// nc_delivery.cu -- spike delivery over the organised connections (include/nc_delivery.h).
//
// The paper keeps one queue per neuron and, every step, increments the time index of every buffered spike.  Here
// the buffered spikes of ALL neurons live in one flat device list of 16-byte entries (source, emission step, next
// group, multiplicity): the time index is `now - emission step`, so nothing is incremented, and one step is
//   advance_insert_kernel : one thread per buffered spike -- matured spikes append (group, multiplicity) to the
//                           spike array, spikes with groups left are re-appended to the other list (ping-pong),
//                           and the spikes emitted in this step are appended behind them (warp-aggregated atomics);
//   deliver_kernel        : one warp per spike-array entry, lanes over the connections of the group (coalesced
//                           reads of target and weight, one float atomic add per connection).
// Counts stay on the device: the host never waits inside a step.  Where the device supports cooperative launches the
// two kernels run as ONE launch per step (fused_step_kernel: a grid-wide barrier between them, the counters of the next
// step cleared behind it), which halves the cost of a step at biological rates, where a step is launch-bound.
#include "../../include/nc_delivery.h"

#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <cstddef>

#include <algorithm>
#include <cstdlib>
#include <new>

#include "nc_common.cuh"
#include "nc_internal.h"

using namespace nc;

namespace {

struct Counters {
  uint32_t n_live_a;   // entries of live list A
  uint32_t n_arr;      // entries of the spike array (two-kernel step; even steps of the fused step)
  uint32_t n_live_b;   // entries of live list B
  uint32_t n_arr_odd;  // entries of the spike array, odd steps of the fused step
  unsigned long long events, dropped, bad_nodes;
};
// the two-kernel step clears {n_arr, n_live_b} or {n_live_a, n_arr} with ONE 8-byte memset (nc_delivery_step)
static_assert(offsetof(Counters, n_live_a) == 0 && offsetof(Counters, n_arr) == 4 && offsetof(Counters, n_live_b) == 8,
              "nc_delivery_step resets two neighbouring counters at once");

struct StepParams {
  nc_organised_view v;
  const uint4* live_in;   // (source, emission step, next global group, multiplicity)
  uint4* live_out;
  const uint32_t* n_live_in;
  uint32_t* n_live_out;
  uint32_t* n_arr;
  uint2* arr;             // (global group, multiplicity)
  uint2* arr_range;       // (first, one past the last) organised position of the group's connections
  Counters* ctr;
  const uint32_t* new_nodes;
  const uint32_t* new_mult;
  uint32_t n_new, capacity, now;
};

// a slot for the lanes with want_a set and one for those with want_b set: two warp-aggregated reservations at once, both
// atomics issued before either result is waited for
__device__ __forceinline__ void warp_reserve2(uint32_t* counter_a, bool want_a, uint32_t* counter_b, bool want_b,
                                              uint32_t& slot_a, uint32_t& slot_b) {
  const uint32_t ma = __ballot_sync(0xffffffffu, want_a), mb = __ballot_sync(0xffffffffu, want_b);
  uint32_t base_a = 0, base_b = 0;
  if (ma && lane_id() == (uint32_t)(__ffs(ma) - 1)) base_a = atomicAdd(counter_a, (uint32_t)__popc(ma));
  if (mb && lane_id() == (uint32_t)(__ffs(mb) - 1)) base_b = atomicAdd(counter_b, (uint32_t)__popc(mb));
  base_a = __shfl_sync(0xffffffffu, base_a, ma ? __ffs(ma) - 1 : 0);
  base_b = __shfl_sync(0xffffffffu, base_b, mb ? __ffs(mb) - 1 : 0);
  slot_a = base_a + __popc(ma & lanemask_lt());
  slot_b = base_b + __popc(mb & lanemask_lt());
}

constexpr int kStepThreads = 256;

__device__ __forceinline__ void advance_insert_body(const StepParams& p) {
  const uint32_t n_live = min(*p.n_live_in, p.capacity);
  const uint32_t total = n_live + p.n_new;
  const uint32_t rounds = (total + gridDim.x * kStepThreads - 1) / (gridDim.x * kStepThreads);
  for (uint32_t r = 0; r < rounds; ++r) {  // whole warps stay in the loop: the ballots below need all lanes
    const uint32_t i = (r * gridDim.x + blockIdx.x) * kStepThreads + threadIdx.x;
    bool keep = false, mature = false, bad = false;
    uint4 sp = make_uint4(0u, 0u, 0u, 0u);
    uint32_t g_mature = 0;
    uint2 range = make_uint2(0u, 0u);
    if (i < n_live) {
      sp = p.live_in[i];
      const uint32_t end = p.v.group_ptr[sp.x + 1];
      // where the group's connections lie: fetched together with its delay, so that the delivery phase finds the
      // range in the spike array instead of chasing group -> group_start after the barrier
      range.x = p.v.group_start[sp.z];
      range.y = sp.z + 1 < p.v.total_groups ? p.v.group_start[sp.z + 1] : (uint32_t)p.v.n;
      // time index = steps since emission ("the time indexes of all the spikes are increased by one")
      if (p.v.group_delay[sp.z] == p.now - sp.y) {
        mature = true;
        g_mature = sp.z;
        sp.z += 1;  // "its connection group index is incremented by one unit"
      }
      keep = sp.z < end;
    } else if (i < total) {
      const uint32_t k = i - n_live;
      const uint32_t s = p.new_nodes[k], m = p.new_mult ? p.new_mult[k] : 1u;
      if (s >= p.v.n_nodes) {
        bad = true;
      } else {
        const uint32_t g0 = p.v.group_ptr[s], g1 = p.v.group_ptr[s + 1];
        keep = m != 0 && g0 < g1;  // a node without outgoing connections buffers nothing
        sp = make_uint4(s, p.now, g0, m);
      }
    }
    uint32_t a, o;
    warp_reserve2(p.n_arr, mature, p.n_live_out, keep, a, o);
    if (mature) {  // one entry per buffered spike at most: always fits
      p.arr[a] = make_uint2(g_mature, sp.w);
      p.arr_range[a] = range;
    }
    if (keep) {
      if (o < p.capacity) p.live_out[o] = sp;
      else atomicAdd(&p.ctr->dropped, 1ull);
    }
    if (bad) atomicAdd(&p.ctr->bad_nodes, 1ull);
  }
}

struct DeliverParams {
  nc_organised_view v;
  const uint32_t* n_arr;
  const uint2* arr;
  const uint2* arr_range;
  Counters* ctr;
  float* input;
  uint32_t capacity;
};

// BLOCKS: the organised connections live in the storage blocks (COPASS organisation); position c is entry c % B of
// block c / B, a group may straddle two blocks.
__global__ void __launch_bounds__(kStepThreads) advance_insert_kernel(const __grid_constant__ StepParams p) {
  advance_insert_body(p);
}

template <bool BLOCKS>
__device__ __forceinline__ void deliver_body(const DeliverParams& p) {
  const uint32_t n_arr = min(*p.n_arr, p.capacity);
  const uint32_t warps = gridDim.x * (256 / 32);
  unsigned long long ev = 0;
  for (uint32_t e = blockIdx.x * (256 / 32) + (threadIdx.x >> 5); e < n_arr; e += warps) {
    const uint2 ent = p.arr[e], range = p.arr_range[e];
    const uint32_t c0 = range.x, c1 = range.y;
    const float m = (float)ent.y;
    // kUnroll x 32 connections per round: all loads of a round are issued before the first add, so a large group
    // costs one memory latency per 256 connections instead of one per 32 (the largest groups of configs[2] have
    // several hundred connections and would otherwise set the duration of the whole step)
    constexpr int kUnroll = 16;
    for (uint32_t cb = c0 + lane_id(); cb < c1; cb += 32 * kUnroll) {
      uint32_t t[kUnroll];
      float w[kUnroll];
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) {
        const uint32_t c = cb + 32u * u;
        t[u] = 0xffffffffu;
        if (c < c1) {
          if (BLOCKS) {
            const uint64_t blk = c / p.v.block_size, slot = c - blk * p.v.block_size;
            const char* base = reinterpret_cast<const char*>(p.v.block_table[blk]);
            t[u] = reinterpret_cast<const uint32_t*>(base + p.v.off_target)[slot];
            w[u] = reinterpret_cast<const float*>(base + p.v.off_weight)[slot];
          } else {
            t[u] = p.v.target[c];
            w[u] = p.v.weight[c];
          }
        }
      }
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) {
        const uint32_t c = cb + 32u * u;
        if (c < c1) {
          const uint64_t in = p.v.port ? (uint64_t)p.v.port[c] * p.v.n_nodes + t[u] : t[u];  // input of (port, node)
          atomicAdd(p.input + in, w[u] * m);
        }
      }
    }
    ev += c1 - c0;
  }
  // one atomic per CTA on the event counter (thousands of warps finish within a few microseconds of one another)
  __shared__ unsigned long long cta_events;
  if (threadIdx.x == 0) cta_events = 0ull;
  __syncthreads();
  if (lane_id() == 0 && ev) atomicAdd(&cta_events, ev);
  __syncthreads();
  if (threadIdx.x == 0 && cta_events) atomicAdd(&p.ctr->events, cta_events);
}

template <bool BLOCKS>
__global__ void __launch_bounds__(256) deliver_kernel(const __grid_constant__ DeliverParams p) {
  deliver_body<BLOCKS>(p);
}

// One launch per step (cooperative): advance + insert, a grid-wide barrier, delivery.  The counters the NEXT step
// appends to are cleared here, after the barrier, when nobody reads them any more: the list counter this step
// consumed, and the other of the two spike-array counters (the host may still read this step's).
template <bool BLOCKS>
__global__ void __launch_bounds__(kStepThreads) fused_step_kernel(const __grid_constant__ StepParams sp,
                                                                 const __grid_constant__ DeliverParams dp,
                                                                 uint32_t* clear_a, uint32_t* clear_b) {
  advance_insert_body(sp);
  cooperative_groups::this_grid().sync();
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    *clear_a = 0u;
    *clear_b = 0u;
  }
  deliver_body<BLOCKS>(dp);
}

}  // namespace

struct nc_delivery {
  nc_context* ctx = nullptr;
  nc_organised_view v{};
  uint32_t capacity = 0, now = 0;
  int cur = 0;  // which live list is the input of the next step
  uint4* live[2] = {nullptr, nullptr};
  uint2* arr = nullptr;
  uint2* arr_range = nullptr;
  Counters* ctr = nullptr;
  int sms = 148;
  int coop_grid = 0;                  // > 0: one cooperative launch per step with at most this many CTAs
  uint32_t* last_arr_ctr = nullptr;   // counter of the spike array the last step filled
  bool attached = false;              // counted in the context (nc_destroy refuses while deliveries exist)
};

extern "C" {

int nc_delivery_create(nc_context* ctx, uint32_t capacity, nc_delivery** out) {
  if (!ctx || !out || capacity == 0) return NC_ERR_INVALID_ARG;
  *out = nullptr;
  nc_organised_view v{};
  int rc = nc_internal_organised_view(ctx, &v);
  if (rc != NC_OK) return rc;
  nc_delivery* d = new (std::nothrow) nc_delivery();
  if (!d) return NC_ERR_OOM;
  d->ctx = ctx;
  d->v = v;
  d->capacity = capacity;
  d->live[0] = (uint4*)nc_internal_alloc(ctx, (size_t)capacity * 16);
  d->live[1] = (uint4*)nc_internal_alloc(ctx, (size_t)capacity * 16);
  d->arr = (uint2*)nc_internal_alloc(ctx, (size_t)capacity * 8);
  d->arr_range = (uint2*)nc_internal_alloc(ctx, (size_t)capacity * 8);
  d->ctr = (Counters*)nc_internal_alloc(ctx, sizeof(Counters));
  if (!d->live[0] || !d->live[1] || !d->arr || !d->arr_range || !d->ctr) {
    nc_delivery_destroy(d);
    return nc_internal_fail(ctx, NC_ERR_OOM, "out of device memory for the spike buffers");
  }
  if (cudaMemsetAsync(d->ctr, 0, sizeof(Counters), v.stream) != cudaSuccess) {
    nc_delivery_destroy(d);
    return nc_internal_fail(ctx, NC_ERR_CUDA, "cudaMemsetAsync failed");
  }
  int dev = 0;
  if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&d->sms, cudaDevAttrMultiProcessorCount, dev);
  d->last_arr_ctr = &d->ctr->n_arr;
  // one cooperative launch per step when the device supports it (NC_DELIVERY_TWO_KERNELS=1 keeps the two-kernel step)
  const char* two = getenv("NC_DELIVERY_TWO_KERNELS");
  int coop = 0, per_sm = 0;
  if (!(two && atoi(two) != 0) && cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) == cudaSuccess && coop) {
    const cudaError_t e = v.block_table
                              ? cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fused_step_kernel<true>, kStepThreads, 0)
                              : cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fused_step_kernel<false>, kStepThreads, 0);
    if (e == cudaSuccess && per_sm > 0) d->coop_grid = d->sms * std::min(per_sm, 8);
  }
  cudaGetLastError();
  nc_internal_attach(ctx, +1);
  d->attached = true;
  *out = d;
  return NC_OK;
}

int nc_delivery_destroy(nc_delivery* d) {
  if (!d) return NC_OK;
  cudaStreamSynchronize(d->v.stream);
  nc_internal_free(d->ctx, d->live[0]);
  nc_internal_free(d->ctx, d->live[1]);
  nc_internal_free(d->ctx, d->arr);
  nc_internal_free(d->ctx, d->arr_range);
  nc_internal_free(d->ctx, d->ctr);
  if (d->attached) nc_internal_attach(d->ctx, -1);
  delete d;
  return NC_OK;
}

int nc_delivery_step(nc_delivery* d, const uint32_t* d_nodes, const uint32_t* d_mult, uint32_t n_new, float* d_input) {
  if (!d || !d_input || (n_new && !d_nodes)) return NC_ERR_INVALID_ARG;
  cudaStream_t st = d->v.stream;
  uint32_t* n_live_in = d->cur == 0 ? &d->ctr->n_live_a : &d->ctr->n_live_b;
  uint32_t* n_live_out = d->cur == 0 ? &d->ctr->n_live_b : &d->ctr->n_live_a;
  const uint32_t now = d->now + 1;  // committed only once the step has been launched
  const bool fused = d->coop_grid > 0;
  // fused step: two spike-array counters used in turn, each cleared by the step before (see fused_step_kernel)
  uint32_t* n_arr = fused && (now & 1u) ? &d->ctr->n_arr_odd : &d->ctr->n_arr;
  uint32_t* n_arr_next = fused && (now & 1u) ? &d->ctr->n_arr : &d->ctr->n_arr_odd;
  if (!fused) {
    // the spike array and the list that is written in this step start empty; they sit next to each other in Counters
    uint32_t* reset_from = d->cur == 0 ? &d->ctr->n_arr : &d->ctr->n_live_a;  // {n_arr, n_live_b} or {n_live_a, n_arr}
    if (cudaMemsetAsync(reset_from, 0, 8, st) != cudaSuccess) return nc_internal_fail(d->ctx, NC_ERR_CUDA, "cudaMemsetAsync failed");
  }
  StepParams sp{};
  sp.v = d->v;
  sp.live_in = d->live[d->cur];
  sp.live_out = d->live[1 - d->cur];
  sp.n_live_in = n_live_in;
  sp.n_live_out = n_live_out;
  sp.n_arr = n_arr;
  sp.arr = d->arr;
  sp.arr_range = d->arr_range;
  sp.ctr = d->ctr;
  sp.new_nodes = d_nodes;
  sp.new_mult = d_mult;
  sp.n_new = n_new;
  sp.capacity = d->capacity;
  sp.now = now;
  DeliverParams dp{};
  dp.v = d->v;
  dp.n_arr = n_arr;
  dp.arr = d->arr;
  dp.arr_range = d->arr_range;
  dp.ctr = d->ctr;
  dp.input = d_input;
  dp.capacity = d->capacity;
  // the number of buffered spikes is only known on the device: a fixed grid strides over them
  const uint64_t most = (uint64_t)d->capacity + n_new;
  const unsigned grid = (unsigned)std::max<uint64_t>(1, std::min<uint64_t>((most + kStepThreads - 1) / kStepThreads, (uint64_t)d->sms * 8));
  const unsigned dgrid = (unsigned)std::max<uint64_t>(1, std::min<uint64_t>(((uint64_t)d->capacity + 7) / 8, (uint64_t)d->sms * 8));
  if (fused) {
    const unsigned g = std::min<unsigned>(std::max(grid, dgrid), (unsigned)d->coop_grid);
    void* args[] = {(void*)&sp, (void*)&dp, (void*)&n_live_in, (void*)&n_arr_next};
    const cudaError_t e = d->v.block_table
                              ? cudaLaunchCooperativeKernel((void*)fused_step_kernel<true>, dim3(g), dim3(kStepThreads), args, 0, st)
                              : cudaLaunchCooperativeKernel((void*)fused_step_kernel<false>, dim3(g), dim3(kStepThreads), args, 0, st);
    if (e != cudaSuccess) return nc_internal_fail(d->ctx, NC_ERR_CUDA, cudaGetErrorString(e));
  } else {
    advance_insert_kernel<<<grid, kStepThreads, 0, st>>>(sp);
    if (d->v.block_table) deliver_kernel<true><<<dgrid, 256, 0, st>>>(dp);
    else deliver_kernel<false><<<dgrid, 256, 0, st>>>(dp);
  }
  if (cudaPeekAtLastError() != cudaSuccess)
    return nc_internal_fail(d->ctx, NC_ERR_CUDA, cudaGetErrorString(cudaGetLastError()));
  d->now = now;
  d->last_arr_ctr = n_arr;
  d->cur = 1 - d->cur;
  return NC_OK;
}

int nc_delivery_run(nc_delivery* d, uint32_t n_steps, const uint32_t* d_nodes, const uint32_t* d_mult,
                    const uint64_t* offsets, float* d_input) {
  if (!d || !offsets || !d_input) return NC_ERR_INVALID_ARG;
  for (uint32_t k = 0; k < n_steps; ++k) {
    if (offsets[k + 1] < offsets[k] || offsets[k + 1] - offsets[k] > 0xffffffffull) return NC_ERR_INVALID_ARG;
    const uint32_t n_new = (uint32_t)(offsets[k + 1] - offsets[k]);
    const int rc = nc_delivery_step(d, n_new ? d_nodes + offsets[k] : nullptr, (d_mult && n_new) ? d_mult + offsets[k] : nullptr,
                                    n_new, d_input);
    if (rc != NC_OK) return rc;
  }
  return NC_OK;
}

int nc_delivery_num_ports(nc_delivery* d, uint32_t* n_ports) {
  if (!d || !n_ports) return NC_ERR_INVALID_ARG;
  *n_ports = d->v.n_ports;
  return NC_OK;
}

int nc_delivery_read_spike_array(nc_delivery* d, uint32_t* group, uint32_t* mult, uint32_t cap, uint32_t* n) {
  if (!d || !n) return NC_ERR_INVALID_ARG;
  cudaStream_t st = d->v.stream;
  uint32_t cnt = 0;
  if (cudaMemcpyAsync(&cnt, d->last_arr_ctr, 4, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaStreamSynchronize(st) != cudaSuccess)
    return nc_internal_fail(d->ctx, NC_ERR_CUDA, "reading the spike array failed");
  *n = cnt;
  const uint32_t take = cnt < cap ? cnt : cap;
  if (take && group && mult) {
    uint2* tmp = new (std::nothrow) uint2[take];
    if (!tmp) return NC_ERR_OOM;
    cudaError_t e = cudaMemcpyAsync(tmp, d->arr, (size_t)take * 8, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    for (uint32_t i = 0; i < take && e == cudaSuccess; ++i) {
      group[i] = tmp[i].x;
      mult[i] = tmp[i].y;
    }
    delete[] tmp;
    if (e != cudaSuccess) return nc_internal_fail(d->ctx, NC_ERR_CUDA, cudaGetErrorString(e));
  }
  return NC_OK;
}

int nc_delivery_counts(nc_delivery* d, uint64_t* buffered, uint64_t* events, uint64_t* dropped, uint64_t* bad_nodes) {
  if (!d) return NC_ERR_INVALID_ARG;
  Counters h{};
  cudaStream_t st = d->v.stream;
  if (cudaMemcpyAsync(&h, d->ctr, sizeof(Counters), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
      cudaStreamSynchronize(st) != cudaSuccess)
    return nc_internal_fail(d->ctx, NC_ERR_CUDA, "reading the delivery counters failed");
  const uint32_t live = d->cur == 0 ? h.n_live_a : h.n_live_b;
  if (buffered) *buffered = live < d->capacity ? live : d->capacity;
  if (events) *events = h.events;
  if (dropped) *dropped = h.dropped;
  if (bad_nodes) *bad_nodes = h.bad_nodes;
  return NC_OK;
}

}  // extern "C"
