// nc_api.cu -- host side of libnc: the context, and the C ABI of include/nc.h.  No torch types, no CPU compute path.
// One translation unit, written in parts that are included below in this order:
//   nc_host_common.inl    error plumbing, device allocations (guard zones), timing spans, Eq. 1 block reservation, device scan
//   nc_host_organise.inl  the organisation paths over flat arrays (pairs, single-pass look-back, default count / scan / scatter, bulk-fed)
//   nc_host_copass.inl    host plan of the COPASS organisation inside the storage blocks
//   nc_host_index.inl     index construction, timings, device self-tests
//   nc_host_connect.inl   the connect path (rule validation, generator dispatch, pair-mask rules, flags, sharding) and nc_connect*
// and, in this file, nc_create / nc_destroy, nc_finalize, the getters and readers, and nc_internal.h.
#include "../../include/nc.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <unordered_map>
#include <vector>

#include "nc_common.cuh"
#include "nc_internal.h"
#include "nc_generate.cuh"
#include "nc_flags.cuh"
#include "nc_shard.cuh"
#include "nc_index.cuh"
#include "nc_sort.cuh"
#include "nc_sort_split.cuh"
#include "nc_sort_bulk.cuh"
#include "nc_sort_msd.cuh"
#include "nc_copass.cuh"
#include "../../include/nc_copass.h"

using namespace nc;

namespace {

constexpr uint64_t kMaxConns = 0xffffffffull;
constexpr double kZMax = 5.769;  // |z| <= sqrt(48 ln 2) = 5.7681 (D5/D6), rounded up (Q6)
constexpr int kSortThreads = 512;
constexpr int kSortItems = 16;

struct Span {
  int phase;
  bool is_pass;
  cudaEvent_t a, b;
};

inline uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }
inline uint32_t bit_width_u64(uint64_t v) {
  uint32_t b = 0;
  while (v) {
    ++b;
    v >>= 1;
  }
  return b;
}

}  // namespace

struct nc_context {
  nc_config cfg{};
  cudaStream_t stream = nullptr;
  int device = 0;
  uint64_t B = 0;
  double dt = 0, inv_dt = 0;
  std::string err;

  uint32_t n_nodes = 0;
  uint32_t n_proj = 0;
  uint64_t n_conns = 0;
  bool finalized = false;
  uint32_t max_delay_steps = 1;  // bound over all projections (Q6), sets the key's delay bits

  // storage blocks (D9)
  std::vector<void*> blocks;
  uint64_t* d_table = nullptr;
  size_t table_cap = 0;
  uint64_t off_tgt = 0, off_w = 0, off_d = 0, block_bytes = 0;
  uint64_t off_perm = 0;            // NC_FLAG_ORGANISE_COPASS: a fifth array per block (creation positions)
  bool organised_in_blocks = false; // nc_finalize left the organised connections in the storage blocks
  CopassTotals* d_copass_totals = nullptr;
  uint64_t copass_aux_bytes = 0, copass_moved = 0;
  uint8_t cur_port = 0, cur_group = 0;       // attributes in force for the next nc_connect*
  uint32_t rule_flags = 0;                   // NC_NO_AUTAPSES | NC_NO_MULTAPSES for the next nc_connect*
  bool sharded = false;                      // nc_set_shard: keep only connections whose target id is in the owned range
  uint32_t shard_first = 0, shard_count = 0;
  std::vector<void*> stage_blocks;           // sharded contexts: staging blocks, kept from call to call (released by nc_finalize)
  uint64_t* stage_table = nullptr;
  size_t stage_cap = 0;
  uint64_t stage_n = 0;                      // connections staged and not yet filtered (flush_shard)
  std::vector<std::pair<uint32_t, uint64_t>> stage_pending;  // (projection, its first staged position) of the staged calls
  std::vector<uint32_t> proj_first;          // creation position of the first connection of every projection
  std::vector<uint16_t> proj_attr;           // port | syn_group << 8 of every projection
  uint8_t* d_sorted_port = nullptr;          // port of every organised connection, built on first use by delivery
  bool broken = false;  // an in-place organisation failed half way: the connections are lost, only nc_destroy is left

  // allocations
  int atomic_rank = -1;         // NC_FLAG_SORT_BULK / _BUCKETS: -1 not decided yet, 0 ranks from ballots (default), 1 from returning shared atomics (NC_ATOMIC_RANK=1 and the device check passed)
  int attached = 0;             // delivery objects that allocate from this context (nc_destroy refuses while any exists)
  bool guard = false;           // NC_GUARD=1: every allocation sits between two 256-byte guard zones checked when it is freed
  uint64_t guard_violations = 0;
  std::unordered_map<void*, size_t> live;
  std::vector<void*> deferred;  // scratch to release at the next point the stream is known idle
  uint64_t bytes_in_use = 0, bytes_peak = 0;

  // sorted view + index
  uint32_t *s_src = nullptr, *s_tgt = nullptr, *perm = nullptr;
  float* s_w = nullptr;
  uint16_t* s_d = nullptr;
  uint32_t *src_offsets = nullptr, *group_count = nullptr, *group_ptr = nullptr, *group_start = nullptr;
  uint16_t* group_delay = nullptr;
  uint32_t total_groups = 0;
  uint64_t* d_total_groups = nullptr;  // device scalar; total_groups is fetched on first use (no sync in nc_finalize)
  uint32_t* d_index_error = nullptr;   // set by index_fused_kernel if its look-back ever gave up; read with total_groups
  bool total_groups_pending = false;
  uint32_t *out_degree = nullptr, *in_degree = nullptr, *d_max = nullptr;  // d_max: [2] device scalars
  bool have_in = false, have_out = false;
  uint32_t max_in = 0, max_out = 0;

  // stats / timing
  uint64_t launches = 0;
  uint32_t key_bits = 0, delay_bits = 0, sort_passes = 0;
  std::vector<Span> spans;
  bool gen_open = false;  // a span over consecutive generate launches is open (no events in between: they may overlap)
  cudaEvent_t gen_a = nullptr;
  nc_timings acc{};
};

#include "nc_host_common.inl"
#include "nc_host_organise.inl"
#include "nc_host_msd.inl"
#include "nc_host_copass.inl"
#include "nc_host_index.inl"


// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

int nc_create(const nc_config* cfg, nc_context** out) {
  if (!cfg || !out) return NC_ERR_INVALID_ARG;
  *out = nullptr;
  if (!(cfg->dt_ms > 0.0) || std::isinf(cfg->dt_ms)) return NC_ERR_INVALID_ARG;
  if ((cfg->mem.alloc == nullptr) != (cfg->mem.free == nullptr)) return NC_ERR_INVALID_ARG;
  int count = 0;
  if (cudaGetDeviceCount(&count) != cudaSuccess || count == 0) {
    cudaGetLastError();
    return NC_ERR_CUDA;  // no CPU fallback
  }
  int dev = cfg->device;
  if (dev < 0) {
    if (cudaGetDevice(&dev) != cudaSuccess) return NC_ERR_CUDA;
  } else {
    if (dev >= count || cudaSetDevice(dev) != cudaSuccess) return NC_ERR_CUDA;
  }
  nc_context* c = new (std::nothrow) nc_context();
  if (!c) return NC_ERR_OOM;
  c->cfg = *cfg;
  c->device = dev;
  c->stream = (cudaStream_t)cfg->cuda_stream;
  {
    const char* e = getenv("NC_GUARD");
    c->guard = e && atoi(e) != 0;
  }
  c->B = cfg->block_size ? cfg->block_size : (1ull << 24);  // Q10
  c->dt = cfg->dt_ms;
  c->inv_dt = 1.0 / cfg->dt_ms;  // Q5: computed once
  c->off_tgt = align_up(c->B * 4, 256);
  c->off_w = c->off_tgt + align_up(c->B * 4, 256);
  c->off_d = c->off_w + align_up(c->B * 4, 256);
  c->block_bytes = c->off_d + align_up(c->B * 2, 256);
  if (cfg->flags & NC_FLAG_ORGANISE_COPASS) {
    // a block must be able to hold its connections as five arrays (18 B each) and, while the block-sort runs,
    // as 16-byte records
    c->off_perm = c->block_bytes;
    c->block_bytes = std::max(c->off_perm + align_up(c->B * 4, 256), align_up(c->B * 16, 256));
  }
  c->d_max = (uint32_t*)dev_alloc(c, 8);
  if (!c->d_max) {
    delete c;
    return NC_ERR_OOM;
  }
  if (cudaMemsetAsync(c->d_max, 0, 8, c->stream) != cudaSuccess) {
    dev_free(c, c->d_max);
    delete c;
    return NC_ERR_CUDA;
  }
  *out = c;
  return NC_OK;
}

int nc_destroy(nc_context* c) {
  if (!c) return NC_OK;
  if (c->attached > 0)  // their buffers live in this context: destroying it first would leave them dangling
    return fail(c, NC_ERR_STATE, "nc_destroy: nc_delivery objects of this context still exist; destroy them first");
  gen_span_end(c);
  cudaStreamSynchronize(c->stream);
  for (Span& s : c->spans) {
    cudaEventDestroy(s.a);
    cudaEventDestroy(s.b);
  }
  release_deferred(c);
  std::vector<void*> all;
  for (auto& kv : c->live) all.push_back(kv.first);
  for (void* p : all) dev_free(c, p);
  const bool clean = c->guard_violations == 0;
  delete c;
  return clean ? NC_OK : NC_ERR_STATE;  // NC_GUARD=1: something wrote outside a buffer of the library
}

const char* nc_last_error(nc_context* c) { return c ? c->err.c_str() : "null context"; }

int nc_synchronize(nc_context* c) {
  if (!c) return NC_ERR_INVALID_ARG;
  return sync_stream(c);
}

int nc_create_population(nc_context* c, uint32_t n, uint32_t* first_id) {
  if (!c || !first_id || n == 0) return fail(c, NC_ERR_INVALID_ARG, "nc_create_population: bad argument");
  if (c->finalized) return fail(c, NC_ERR_STATE, "nc_create_population after nc_finalize");
  if ((uint64_t)c->n_nodes + n > 0xffffffffull) return fail(c, NC_ERR_CAPACITY, "more than 2^32-1 nodes");
  *first_id = c->n_nodes;  // D1
  c->n_nodes += n;
  return NC_OK;
}

#include "nc_host_connect.inl"

// A failed nc_finalize keeps nothing: the index and organised arrays it had assigned are released (kernels of the failed
// attempt may still run, hence the deferred release) so that a retry starts clean and nothing stays allocated twice.
static void drop_finalize_outputs(nc_context* c) {
  void** outs[] = {(void**)&c->src_offsets, (void**)&c->group_ptr, (void**)&c->group_count, (void**)&c->group_start,
                   (void**)&c->group_delay, (void**)&c->s_src,     (void**)&c->s_tgt,       (void**)&c->s_w,
                   (void**)&c->s_d,         (void**)&c->perm};
  for (void** o : outs) {
    dev_free_later(c, *o);
    *o = nullptr;
  }
}

int nc_finalize(nc_context* c) {
  if (!c) return NC_ERR_INVALID_ARG;
  if (c->broken) return fail(c, NC_ERR_STATE, "nc_finalize: a failed in-place organisation left this context without connections; destroy it");
  if (c->finalized) return fail(c, NC_ERR_STATE, "nc_finalize called twice");
  gen_span_end(c);
  {
    const int frc = flush_shard(c);
    if (frc != NC_OK) return frc;
  }
  for (void* b : c->stage_blocks) dev_free_later(c, b);  // a sharded context's staging is not needed any more
  c->stage_blocks.clear();
  dev_free_later(c, c->stage_table);
  c->stage_table = nullptr;
  c->stage_cap = 0;
  const uint32_t N = c->n_nodes;
  c->src_offsets = (uint32_t*)dev_alloc(c, ((size_t)N + 1) * 4);
  c->group_ptr = (uint32_t*)dev_alloc(c, ((size_t)N + 1) * 4);
  c->group_count = (uint32_t*)dev_alloc(c, (size_t)N * 4);
  if (!c->out_degree) c->out_degree = (uint32_t*)dev_alloc(c, (size_t)N * 4);
  if (!c->src_offsets || !c->group_ptr || !c->group_count || !c->out_degree) {
    drop_finalize_outputs(c);
    return fail(c, NC_ERR_OOM, "out of device memory for the index");
  }
  NC_CUDA(c, cudaMemsetAsync(c->d_max + 1, 0, 4, c->stream));

  // key-width plan: source bits from the node count, delay bits from the analytic bound (Q6)
  c->delay_bits = std::max(1u, bit_width_u64(c->max_delay_steps));
  const uint32_t src_bits = std::max(1u, bit_width_u64(N > 0 ? (uint64_t)N - 1 : 0));
  c->key_bits = src_bits + c->delay_bits;
  const PassPlan plan = plan_passes(c->key_bits);
  c->sort_passes = plan.n_passes;

  if (c->n_conns == 0) {
    NC_CUDA(c, cudaMemsetAsync(c->src_offsets, 0, ((size_t)N + 1) * 4, c->stream));
    NC_CUDA(c, cudaMemsetAsync(c->group_ptr, 0, ((size_t)N + 1) * 4, c->stream));
    if (N) {
      NC_CUDA(c, cudaMemsetAsync(c->group_count, 0, (size_t)N * 4, c->stream));
      NC_CUDA(c, cudaMemsetAsync(c->out_degree, 0, (size_t)N * 4, c->stream));
    }
    c->total_groups = 0;
    c->sort_passes = 0;
  } else {
    int rc;
    if (c->cfg.flags & NC_FLAG_ORGANISE_COPASS) {
      if (c->key_bits > 32) {
        drop_finalize_outputs(c);
        return fail(c, NC_ERR_CAPACITY, "COPASS organisation needs a (source, delay) key of at most 32 bits");
      }
      rc = organise_copass(c, plan);
    } else if (c->key_bits > 32) rc = sort_and_index<uint64_t>(c, plan);
    else if (c->cfg.flags & NC_FLAG_SORT_PAIRS) rc = sort_and_index<uint32_t>(c, plan);
    else if (c->cfg.flags & NC_FLAG_SORT_ONESWEEP) rc = sort_carry_and_index(c, plan);
    else if (c->cfg.flags & NC_FLAG_SORT_BUCKETS) rc = sort_msd_and_index(c);
    else rc = sort_split_and_index(c, plan);
    if (rc != NC_OK) {
      drop_finalize_outputs(c);
      return rc;
    }
  }
  c->finalized = true;
  c->have_out = true;
  return NC_OK;
}

int nc_num_connections(nc_context* c, uint64_t* n) {
  if (c && c->sharded && c->stage_n) {  // staged connect calls of a sharded context: filter them first
    const int frc = flush_shard(c);
    if (frc != NC_OK) return frc;
  }
  if (!c || !n) return NC_ERR_INVALID_ARG;
  *n = c->n_conns;  // pairwise_bernoulli already waited for its count inside nc_connect
  return NC_OK;
}

int nc_num_nodes(nc_context* c, uint32_t* n) {
  if (!c || !n) return NC_ERR_INVALID_ARG;
  *n = c->n_nodes;
  return NC_OK;
}

int nc_get_connections(nc_context* c, int sorted, nc_connections_view* out) {
  if (c && c->sharded && c->stage_n) {  // staged connect calls of a sharded context: filter them first
    const int frc = flush_shard(c);
    if (frc != NC_OK) return frc;
  }
  if (!c || !out) return NC_ERR_INVALID_ARG;
  std::memset(out, 0, sizeof(*out));
  out->n = c->n_conns;
  out->block_size = c->B;
  if (c->broken) return fail(c, NC_ERR_STATE, "a failed in-place organisation left this context without connections");
  if (sorted && !c->finalized) return fail(c, NC_ERR_STATE, "sorted view before nc_finalize");
  if (!sorted && c->organised_in_blocks)
    return fail(c, NC_ERR_STATE, "the creation-order view is gone: the blocks were organised in place (COPASS)");
  if (sorted && !c->organised_in_blocks) {
    out->source = c->s_src;
    out->target = c->s_tgt;
    out->weight = c->s_w;
    out->delay = c->s_d;
    out->perm = c->perm;
    return NC_OK;
  }
  if (sorted) {
    out->off_perm = c->off_perm;
    if (c->blocks.size() == 1) out->perm = (const uint32_t*)((char*)c->blocks[0] + c->off_perm);
  }
  out->n_blocks = c->blocks.size();
  out->blocks = c->blocks.data();
  out->off_source = 0;
  out->off_target = c->off_tgt;
  out->off_weight = c->off_w;
  out->off_delay = c->off_d;
  if (c->blocks.size() == 1) {
    char* b = (char*)c->blocks[0];
    out->source = (const uint32_t*)b;
    out->target = (const uint32_t*)(b + c->off_tgt);
    out->weight = (const float*)(b + c->off_w);
    out->delay = (const uint16_t*)(b + c->off_d);
  }
  return NC_OK;
}

int nc_get_index(nc_context* c, nc_index_view* out) {
  if (!c || !out) return NC_ERR_INVALID_ARG;
  if (!c->finalized) return fail(c, NC_ERR_STATE, "index before nc_finalize");
  int rc = ensure_total_groups(c);
  if (rc != NC_OK) return rc;
  out->src_offsets = c->src_offsets;
  out->group_count = c->group_count;
  out->group_ptr = c->group_ptr;
  out->group_start = c->group_start;
  out->group_delay = c->group_delay;
  out->n_nodes = c->n_nodes;
  out->total_groups = c->total_groups;
  return NC_OK;
}

int nc_degree_histogram(nc_context* c, int kind, const uint32_t** per_node_degree, uint32_t* max_degree) {
  if (c && c->sharded && c->stage_n) {  // staged connect calls of a sharded context: filter them first
    const int frc = flush_shard(c);
    if (frc != NC_OK) return frc;
  }
  if (!c || (kind != 0 && kind != 1)) return fail(c, NC_ERR_INVALID_ARG, "nc_degree_histogram: bad argument");
  const uint32_t N = c->n_nodes;
  bool& have = kind == 0 ? c->have_in : c->have_out;
  uint32_t*& deg = kind == 0 ? c->in_degree : c->out_degree;
  if (!have) {
    if (!deg) {
      deg = (uint32_t*)dev_alloc(c, (size_t)N * 4);
      if (!deg) return fail(c, NC_ERR_OOM, "out of device memory for the degree histogram");
    }
    Scope sc(c, NC_PHASE_DEGREE);
    if (N) NC_CUDA(c, cudaMemsetAsync(deg, 0, (size_t)N * 4, c->stream));
    NC_CUDA(c, cudaMemsetAsync(c->d_max + kind, 0, 4, c->stream));
    if (c->n_conns && N) {
      const unsigned grid = (unsigned)std::min<uint64_t>((c->n_conns + 255) / 256, 148ull * 32);
      degree_count_kernel<<<grid, 256, 0, c->stream>>>(make_map(c), c->n_conns, kind, deg);
      NC_LAUNCH_CHECK(c, "degree_count");
      max_u32_kernel<<<std::min<unsigned>((N + 255) / 256, 1024u), 256, 0, c->stream>>>(deg, N, c->d_max + kind);
      NC_LAUNCH_CHECK(c, "max_u32");
    }
    have = true;
  }
  if (per_node_degree) *per_node_degree = deg;
  if (max_degree) {
    NC_CUDA(c, cudaMemcpyAsync(max_degree, c->d_max + kind, 4, cudaMemcpyDeviceToHost, c->stream));
    int rc = sync_stream(c);
    if (rc != NC_OK) return rc;
  }
  return NC_OK;
}

int nc_get_stats(nc_context* c, nc_stats* out) {
  if (c && c->sharded && c->stage_n) {  // staged connect calls of a sharded context: filter them first
    const int frc = flush_shard(c);
    if (frc != NC_OK) return frc;
  }
  if (!c || !out) return NC_ERR_INVALID_ARG;
  out->kernel_launches = c->launches;
  out->bytes_in_use = c->bytes_in_use;
  out->bytes_peak = c->bytes_peak;
  out->n_blocks = c->blocks.size();
  out->n_projections = c->n_proj;
  out->key_bits = c->key_bits;
  out->sort_passes = c->sort_passes;
  out->delay_bits = c->delay_bits;
  return NC_OK;
}

int nc_get_timings(nc_context* c, nc_timings* out) {
  if (!c || !out) return NC_ERR_INVALID_ARG;
  if (!(c->cfg.flags & NC_FLAG_TIMING)) return fail(c, NC_ERR_STATE, "context was created without NC_FLAG_TIMING");
  int rc = collect_timings(c);
  if (rc != NC_OK) return rc;
  *out = c->acc;
  return NC_OK;
}

int nc_read_connections(nc_context* c, int sorted, uint64_t first, uint64_t count, uint32_t* source, uint32_t* target,
                        float* weight, uint16_t* delay, uint32_t* perm) {
  if (c && c->sharded && c->stage_n) {
    const int frc = flush_shard(c);
    if (frc != NC_OK) return frc;
  }
  if (!c) return NC_ERR_INVALID_ARG;
  if (first + count > c->n_conns) return fail(c, NC_ERR_INVALID_ARG, "nc_read_connections: range outside the connections");
  if (sorted && !c->finalized) return fail(c, NC_ERR_STATE, "sorted view before nc_finalize");
  if (c->broken) return fail(c, NC_ERR_STATE, "a failed in-place organisation left this context without connections");
  if (!sorted && c->organised_in_blocks)
    return fail(c, NC_ERR_STATE, "the creation-order view is gone: the blocks were organised in place (COPASS)");
  if (count == 0) return NC_OK;
  const cudaMemcpyKind k = cudaMemcpyDeviceToHost;
  if (sorted && !c->organised_in_blocks) {
    if (source) NC_CUDA(c, cudaMemcpyAsync(source, c->s_src + first, count * 4, k, c->stream));
    if (target) NC_CUDA(c, cudaMemcpyAsync(target, c->s_tgt + first, count * 4, k, c->stream));
    if (weight) NC_CUDA(c, cudaMemcpyAsync(weight, c->s_w + first, count * 4, k, c->stream));
    if (delay) NC_CUDA(c, cudaMemcpyAsync(delay, c->s_d + first, count * 2, k, c->stream));
    if (perm) NC_CUDA(c, cudaMemcpyAsync(perm, c->perm + first, count * 4, k, c->stream));
  } else {
    uint64_t pos = first, done = 0;
    while (done < count) {
      const uint64_t blk = pos / c->B, slot = pos % c->B;
      const uint64_t m = std::min(count - done, c->B - slot);
      char* b = (char*)c->blocks[blk];
      if (source) NC_CUDA(c, cudaMemcpyAsync(source + done, (uint32_t*)b + slot, m * 4, k, c->stream));
      if (target) NC_CUDA(c, cudaMemcpyAsync(target + done, (uint32_t*)(b + c->off_tgt) + slot, m * 4, k, c->stream));
      if (weight) NC_CUDA(c, cudaMemcpyAsync(weight + done, (float*)(b + c->off_w) + slot, m * 4, k, c->stream));
      if (delay) NC_CUDA(c, cudaMemcpyAsync(delay + done, (uint16_t*)(b + c->off_d) + slot, m * 2, k, c->stream));
      if (perm && sorted) NC_CUDA(c, cudaMemcpyAsync(perm + done, (uint32_t*)(b + c->off_perm) + slot, m * 4, k, c->stream));
      pos += m;
      done += m;
    }
  }
  return sync_stream(c);
}

int nc_set_connection_attributes(nc_context* c, uint8_t port, uint8_t syn_group) {
  if (!c) return NC_ERR_INVALID_ARG;
  if (c->finalized) return fail(c, NC_ERR_STATE, "nc_set_connection_attributes after nc_finalize");
  c->cur_port = port;
  c->cur_group = syn_group;
  return NC_OK;
}

int nc_read_connection_attributes(nc_context* c, int sorted, uint64_t first, uint64_t count, uint8_t* port,
                                  uint8_t* syn_group) {
  if (c && c->sharded && c->stage_n) {
    const int frc = flush_shard(c);
    if (frc != NC_OK) return frc;
  }
  if (!c) return NC_ERR_INVALID_ARG;
  if (c->broken) return fail(c, NC_ERR_STATE, "a failed in-place organisation left this context without connections");
  if (first + count > c->n_conns) return fail(c, NC_ERR_INVALID_ARG, "nc_read_connection_attributes: range outside the connections");
  if (sorted && !c->finalized) return fail(c, NC_ERR_STATE, "sorted view before nc_finalize");
  if (!sorted && c->organised_in_blocks)
    return fail(c, NC_ERR_STATE, "the creation-order view is gone: the blocks were organised in place (COPASS)");
  if (count == 0 || (!port && !syn_group)) return NC_OK;
  const uint32_t np = (uint32_t)c->proj_first.size();
  uint32_t* d_first = (uint32_t*)dev_alloc(c, (size_t)np * 4);
  uint16_t* d_attr = (uint16_t*)dev_alloc(c, (size_t)np * 2);
  uint8_t* d_port = port ? (uint8_t*)dev_alloc(c, count) : nullptr;
  uint8_t* d_group = syn_group ? (uint8_t*)dev_alloc(c, count) : nullptr;
  dev_free_later(c, d_first); dev_free_later(c, d_attr); dev_free_later(c, d_port); dev_free_later(c, d_group);
  if (!d_first || !d_attr || (port && !d_port) || (syn_group && !d_group))
    return fail(c, NC_ERR_OOM, "out of device memory in nc_read_connection_attributes");
  NC_CUDA(c, cudaMemcpyAsync(d_first, c->proj_first.data(), (size_t)np * 4, cudaMemcpyHostToDevice, c->stream));
  NC_CUDA(c, cudaMemcpyAsync(d_attr, c->proj_attr.data(), (size_t)np * 2, cudaMemcpyHostToDevice, c->stream));
  const uint32_t* perm = (sorted && !c->organised_in_blocks) ? c->perm : nullptr;
  const uint64_t perm_off = (sorted && c->organised_in_blocks) ? c->off_perm : 0;
  const unsigned grid = (unsigned)std::min<uint64_t>((count + 255) / 256, 148 * 16);
  attribute_lookup_kernel<<<grid, 256, 0, c->stream>>>(make_map(c), perm, perm_off, first, count, d_first, np, d_attr, d_port,
                                                       d_group);
  NC_LAUNCH_CHECK(c, "attribute_lookup");
  if (port) NC_CUDA(c, cudaMemcpyAsync(port, d_port, count, cudaMemcpyDeviceToHost, c->stream));
  if (syn_group) NC_CUDA(c, cudaMemcpyAsync(syn_group, d_group, count, cudaMemcpyDeviceToHost, c->stream));
  return sync_stream(c);
}

int nc_read_index(nc_context* c, uint32_t* src_offsets, uint32_t* group_count, uint32_t* group_ptr, uint32_t* group_start,
                  uint16_t* group_delay) {
  if (!c) return NC_ERR_INVALID_ARG;
  if (!c->finalized) return fail(c, NC_ERR_STATE, "index before nc_finalize");
  int rc0 = ensure_total_groups(c);
  if (rc0 != NC_OK) return rc0;
  const cudaMemcpyKind k = cudaMemcpyDeviceToHost;
  const size_t N = c->n_nodes, G = c->total_groups;
  if (src_offsets) NC_CUDA(c, cudaMemcpyAsync(src_offsets, c->src_offsets, (N + 1) * 4, k, c->stream));
  if (group_ptr) NC_CUDA(c, cudaMemcpyAsync(group_ptr, c->group_ptr, (N + 1) * 4, k, c->stream));
  if (group_count && N) NC_CUDA(c, cudaMemcpyAsync(group_count, c->group_count, N * 4, k, c->stream));
  if (group_start && G) NC_CUDA(c, cudaMemcpyAsync(group_start, c->group_start, G * 4, k, c->stream));
  if (group_delay && G) NC_CUDA(c, cudaMemcpyAsync(group_delay, c->group_delay, G * 2, k, c->stream));
  return sync_stream(c);
}

int nc_read_degree_histogram(nc_context* c, int kind, uint32_t* per_node_degree, uint32_t* max_degree) {
  const uint32_t* dev = nullptr;
  int rc = nc_degree_histogram(c, kind, &dev, max_degree);
  if (rc != NC_OK) return rc;
  if (per_node_degree && c->n_nodes)
    NC_CUDA(c, cudaMemcpyAsync(per_node_degree, dev, (size_t)c->n_nodes * 4, cudaMemcpyDeviceToHost, c->stream));
  return sync_stream(c);
}

int nc_copass_partition(nc_context* c, const uint32_t* keys, uint64_t n_keys, const uint32_t* start, const uint32_t* len,
                        uint32_t k, uint32_t m, uint32_t* m_out, nc_copass_info* info) {
  if (!c) return NC_ERR_INVALID_ARG;
  if (!keys || !start || !len || !m_out || k == 0) return fail(c, NC_ERR_INVALID_ARG, "nc_copass_partition: NULL argument");
  if (k > kCopassMaxBlocks) return fail(c, NC_ERR_CAPACITY, "nc_copass_partition: more than 4096 subarrays");
  if (n_keys > 0xffffffffull) return fail(c, NC_ERR_CAPACITY, "nc_copass_partition: more than 2^32 - 1 keys");
  uint64_t total = 0;
  for (uint32_t i = 0; i < k; ++i) {
    if ((uint64_t)start[i] + len[i] > n_keys) return fail(c, NC_ERR_INVALID_ARG, "nc_copass_partition: subarray outside keys");
    total += len[i];
  }
  if (m == 0 || (uint64_t)m >= total)
    return fail(c, NC_ERR_INVALID_ARG, "nc_copass_partition: 0 < m < sum of the subarray sizes is required (PAPER.md:464)");
  const size_t k1 = (size_t)k + 1;
  uint32_t* d_keys = (uint32_t*)dev_alloc(c, (size_t)n_keys * 4);
  uint32_t* st = (uint32_t*)dev_alloc(c, 7 * k1 * 4 + sizeof(CopassInfo));
  auto drop = [&]() {
    dev_free_later(c, d_keys);
    dev_free_later(c, st);
  };
  if (!d_keys || !st) {
    drop();
    return fail(c, NC_ERR_OOM, "out of device memory in nc_copass_partition");
  }
  uint32_t *d_start = st, *d_len = st + k1, *d_m = st + 2 * k1, *d_left = st + 3 * k1, *d_right = st + 4 * k1,
           *d_new_start = st + 5 * k1, *d_new_len = st + 6 * k1;
  CopassInfo* d_info = (CopassInfo*)(st + 7 * k1);
  NC_CUDA(c, cudaMemcpyAsync(d_keys, keys, (size_t)n_keys * 4, cudaMemcpyHostToDevice, c->stream));
  NC_CUDA(c, cudaMemcpyAsync(d_start, start, (size_t)k * 4, cudaMemcpyHostToDevice, c->stream));
  NC_CUDA(c, cudaMemcpyAsync(d_len, len, (size_t)k * 4, cudaMemcpyHostToDevice, c->stream));
  const size_t smem = 7 * k1 * 4;
  auto part = copass_partition_kernel<FlatKeys>;
  NC_CUDA(c, cudaFuncSetAttribute(part, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  part<<<1, kCopassThreads, smem, c->stream>>>(FlatKeys{d_keys}, k, m, d_start, d_len, 0u, d_m, d_left, d_right,
                                              d_new_start, d_new_len, d_info, nullptr, 0u, 0u);
  NC_LAUNCH_CHECK(c, "copass_partition");
  CopassInfo h{};
  NC_CUDA(c, cudaMemcpyAsync(m_out, d_m, (size_t)k * 4, cudaMemcpyDeviceToHost, c->stream));
  NC_CUDA(c, cudaMemcpyAsync(&h, d_info, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
  drop();
  const int rc = sync_stream(c);
  if (rc != NC_OK) return rc;
  if (info) {
    info->t = h.t;
    info->iterations = h.iterations;
    info->last_step = h.last_step;
  }
  return NC_OK;
}

int nc_get_copass_stats(nc_context* c, nc_copass_stats* out) {
  if (!c || !out) return NC_ERR_INVALID_ARG;
  if (!c->finalized || !(c->cfg.flags & NC_FLAG_ORGANISE_COPASS))
    return fail(c, NC_ERR_STATE, "nc_get_copass_stats: the context was not finalized under NC_FLAG_ORGANISE_COPASS");
  CopassTotals t{};
  if (c->d_copass_totals) {
    NC_CUDA(c, cudaMemcpyAsync(&t, c->d_copass_totals, sizeof(t), cudaMemcpyDeviceToHost, c->stream));
    const int rc = sync_stream(c);
    if (rc != NC_OK) return rc;
  }
  out->partitions = t.partitions;
  out->iterations = t.iterations;
  out->last_step_1 = t.last_step_1;
  out->last_step_2 = t.last_step_2;
  out->n_blocks = c->blocks.size();
  out->aux_bytes = c->copass_aux_bytes;
  out->records_moved = c->copass_moved;
  return NC_OK;
}

int nc_selftest_philox(nc_context* c, uint32_t n, const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
  if (!c || !ctr || !key || !out) return NC_ERR_INVALID_ARG;
  if (n == 0) return NC_OK;
  uint32_t* d_ctr = (uint32_t*)dev_alloc(c, (size_t)n * 16);
  uint32_t* d_key = (uint32_t*)dev_alloc(c, (size_t)n * 8);
  uint32_t* d_out = (uint32_t*)dev_alloc(c, (size_t)n * 16);
  if (!d_ctr || !d_key || !d_out) return fail(c, NC_ERR_OOM, "selftest: out of device memory");
  NC_CUDA(c, cudaMemcpyAsync(d_ctr, ctr, (size_t)n * 16, cudaMemcpyHostToDevice, c->stream));
  NC_CUDA(c, cudaMemcpyAsync(d_key, key, (size_t)n * 8, cudaMemcpyHostToDevice, c->stream));
  selftest_philox_kernel<<<(n + 127) / 128, 128, 0, c->stream>>>(n, d_ctr, d_key, d_out);
  NC_LAUNCH_CHECK(c, "selftest_philox");
  NC_CUDA(c, cudaMemcpyAsync(out, d_out, (size_t)n * 16, cudaMemcpyDeviceToHost, c->stream));
  int rc = sync_stream(c);
  dev_free(c, d_ctr);
  dev_free(c, d_key);
  dev_free(c, d_out);
  return rc;
}

namespace {
__global__ void poke_kernel(unsigned char* p) { *p = 0x11; }
}  // namespace

int nc_selftest_guard(nc_context* c, int offset, uint64_t* violations) {
  if (!c || !violations) return NC_ERR_INVALID_ARG;
  if (!c->guard) return fail(c, NC_ERR_STATE, "nc_selftest_guard: NC_GUARD was not set when the context was created");
  unsigned char* d = (unsigned char*)dev_alloc(c, 1000);
  if (!d) return fail(c, NC_ERR_OOM, "selftest: out of device memory");
  if (offset > 0) poke_kernel<<<1, 1, 0, c->stream>>>(d + 1024);  // first byte behind the body (1000 rounded up to 1024)
  if (offset < 0) poke_kernel<<<1, 1, 0, c->stream>>>(d - 1);
  const uint64_t before = c->guard_violations;
  dev_free(c, d);
  *violations = c->guard_violations - before;
  c->guard_violations = before;  // a deliberate poke is not a finding
  return NC_OK;
}

int nc_selftest_fastpath(nc_context* c, double out[4]) {
  if (!c || !out) return NC_ERR_INVALID_ARG;
  double* d = (double*)dev_alloc(c, 32);
  if (!d) return fail(c, NC_ERR_OOM, "selftest: out of device memory");
  NC_CUDA(c, cudaMemsetAsync(d, 0, 32, c->stream));
  selftest_fastpath_kernel<<<(1u << 24) / 256, 256, 0, c->stream>>>(d);
  NC_LAUNCH_CHECK(c, "selftest_fastpath");
  NC_CUDA(c, cudaMemcpyAsync(out, d, 32, cudaMemcpyDeviceToHost, c->stream));
  int rc = sync_stream(c);
  dev_free(c, d);
  return rc;
}

}  // extern "C"

// ---- nc_internal.h ----
int nc_internal_organised_view(nc_context* c, nc_organised_view* out) {
  if (!c || !out) return NC_ERR_INVALID_ARG;
  if (!c->finalized) return fail(c, NC_ERR_STATE, "the connections are not organised yet (nc_finalize)");
  int rc = ensure_total_groups(c);
  if (rc != NC_OK) return rc;
  std::memset(out, 0, sizeof(*out));
  if (c->organised_in_blocks) {
    out->block_table = c->d_table;
    out->block_size = c->B;
    out->off_target = c->off_tgt;
    out->off_weight = c->off_w;
  } else {
    out->target = c->s_tgt;
    out->weight = c->s_w;
  }
  // receptor ports: materialised once, only if some projection uses a port other than 0
  uint32_t max_port = 0;
  for (uint16_t a : c->proj_attr) max_port = std::max<uint32_t>(max_port, a & 0xffu);
  out->n_ports = max_port + 1;
  if (max_port > 0 && c->n_conns > 0) {
    if (!c->d_sorted_port) {
      const uint32_t np = (uint32_t)c->proj_first.size();
      uint32_t* d_first = (uint32_t*)dev_alloc(c, (size_t)np * 4);
      uint16_t* d_attr = (uint16_t*)dev_alloc(c, (size_t)np * 2);
      c->d_sorted_port = (uint8_t*)dev_alloc(c, c->n_conns);
      dev_free_later(c, d_first);
      dev_free_later(c, d_attr);
      if (!d_first || !d_attr || !c->d_sorted_port) return fail(c, NC_ERR_OOM, "out of device memory for the receptor ports");
      NC_CUDA(c, cudaMemcpyAsync(d_first, c->proj_first.data(), (size_t)np * 4, cudaMemcpyHostToDevice, c->stream));
      NC_CUDA(c, cudaMemcpyAsync(d_attr, c->proj_attr.data(), (size_t)np * 2, cudaMemcpyHostToDevice, c->stream));
      const unsigned grid = (unsigned)std::min<uint64_t>((c->n_conns + 255) / 256, 148 * 16);
      attribute_lookup_kernel<<<grid, 256, 0, c->stream>>>(make_map(c), c->organised_in_blocks ? nullptr : c->perm,
                                                           c->organised_in_blocks ? c->off_perm : 0, 0, c->n_conns, d_first,
                                                           np, d_attr, c->d_sorted_port, nullptr);
      NC_LAUNCH_CHECK(c, "attribute_lookup");
    }
    out->port = c->d_sorted_port;
  }
  out->group_ptr = c->group_ptr;
  out->group_start = c->group_start;
  out->group_delay = c->group_delay;
  out->n_nodes = c->n_nodes;
  out->total_groups = c->total_groups;
  out->n = c->n_conns;
  out->stream = c->stream;
  return NC_OK;
}
void* nc_internal_alloc(nc_context* c, size_t bytes) { return dev_alloc(c, bytes); }
void nc_internal_free(nc_context* c, void* p) { dev_free(c, p); }
int nc_internal_fail(nc_context* c, int code, const char* msg) { return fail(c, code, msg); }
void nc_internal_attach(nc_context* c, int delta) {
  if (c) c->attached += delta;
}
extern "C" uint64_t nc_internal_guard_violations(nc_context* c) { return c ? c->guard_violations : 0; }
