// nc_api.cu -- host side of libnc: context, planner (Eq. 1 block reservation, key-width plan),
// kernel launches and the C ABI of include/nc.h.  No torch types, no CPU compute path.
#include "../../include/nc.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
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

namespace {

int fail(nc_context* c, int code, const std::string& msg) {
  if (c) c->err = msg;
  return code;
}

#define NC_CUDA(ctx, call)                                                                      \
  do {                                                                                          \
    cudaError_t e_ = (call);                                                                    \
    if (e_ != cudaSuccess)                                                                      \
      return fail(ctx, NC_ERR_CUDA, std::string(#call) + ": " + cudaGetErrorString(e_));        \
  } while (0)

#define NC_LAUNCH_CHECK(ctx, name)                                                              \
  do {                                                                                          \
    (ctx)->launches++;                                                                          \
    cudaError_t e_ = cudaPeekAtLastError();                                                     \
    if (e_ != cudaSuccess)                                                                      \
      return fail(ctx, NC_ERR_CUDA, std::string("launch ") + name + ": " + cudaGetErrorString(e_)); \
  } while (0)

// Guard zones (NC_GUARD=1 in the environment; compute-sanitizer is not available on every box): an allocation of n bytes
// becomes 256 guard bytes | n bytes rounded up to 256 | 256 guard bytes, the guards filled with 0xA5 on the context's
// stream and compared when the allocation is freed.  A kernel that writes up to 256 bytes before or behind a buffer of
// the library is then counted (nc_internal_guard_violations) and reported on stderr instead of going unnoticed.
constexpr size_t kGuardBytes = 256;

void* dev_alloc(nc_context* c, size_t bytes) {
  if (bytes == 0) bytes = 256;
  const size_t body = c->guard ? (bytes + 255) / 256 * 256 : bytes;
  const size_t total = c->guard ? body + 2 * kGuardBytes : bytes;
  void* p = nullptr;
  if (c->cfg.mem.alloc) {
    p = c->cfg.mem.alloc(c->cfg.mem.user, total);
  } else {
    if (cudaMalloc(&p, total) != cudaSuccess) {
      cudaGetLastError();
      p = nullptr;
    }
  }
  if (p && c->guard) {
    cudaMemsetAsync(p, 0xA5, kGuardBytes, c->stream);
    cudaMemsetAsync((char*)p + kGuardBytes + body, 0xA5, kGuardBytes, c->stream);
    p = (char*)p + kGuardBytes;
  }
  if (p) {
    c->live[p] = bytes;
    c->bytes_in_use += bytes;
    c->bytes_peak = std::max(c->bytes_peak, c->bytes_in_use);
  }
  return p;
}

void dev_free(nc_context* c, void* p) {
  if (!p) return;
  size_t bytes = 0;
  auto it = c->live.find(p);
  if (it != c->live.end()) {
    bytes = it->second;
    c->bytes_in_use -= it->second;
    c->live.erase(it);
  }
  if (c->guard) {
    const size_t body = (bytes + 255) / 256 * 256;
    unsigned char g[2][kGuardBytes];
    cudaStreamSynchronize(c->stream);
    cudaMemcpy(g[0], (char*)p - kGuardBytes, kGuardBytes, cudaMemcpyDeviceToHost);
    cudaMemcpy(g[1], (char*)p + body, kGuardBytes, cudaMemcpyDeviceToHost);
    for (int side = 0; side < 2; ++side)
      for (size_t i = 0; i < kGuardBytes; ++i)
        if (g[side][i] != 0xA5) {
          ++c->guard_violations;
          fprintf(stderr, "libnc guard: byte %zu %s an allocation of %zu bytes was overwritten\n", side ? i : kGuardBytes - i,
                  side ? "behind" : "before", bytes);
          break;
        }
    p = (char*)p - kGuardBytes;
  }
  if (c->cfg.mem.alloc) {
    c->cfg.mem.free(c->cfg.mem.user, p);
  } else {
    cudaFree(p);
  }
}

// scratch that may still be read by enqueued kernels: released once the stream has been synchronised
void dev_free_later(nc_context* c, void* p) {
  if (p) c->deferred.push_back(p);
}
void release_deferred(nc_context* c) {
  for (void* p : c->deferred) dev_free(c, p);
  c->deferred.clear();
}

int sync_stream(nc_context* c) {
  NC_CUDA(c, cudaStreamSynchronize(c->stream));
  release_deferred(c);
  return NC_OK;
}

void gen_span_end(nc_context* c);

struct Scope {  // CUDA-event span around a phase (NC_FLAG_TIMING)
  nc_context* c;
  Span s{};
  bool on;
  Scope(nc_context* c_, int phase, bool is_pass = false) : c(c_), on((c_->cfg.flags & NC_FLAG_TIMING) != 0) {
    if (!on) return;
    gen_span_end(c);
    s.phase = phase;
    s.is_pass = is_pass;
    cudaEventCreate(&s.a);
    cudaEventCreate(&s.b);
    cudaEventRecord(s.a, c->stream);
  }
  ~Scope() {
    if (!on) return;
    cudaEventRecord(s.b, c->stream);
    c->spans.push_back(s);
  }
};

// Consecutive generate launches are timed as ONE span (first launch .. close), because an event between two of
// them would serialise kernels that are allowed to overlap (programmatic dependent launch).
void gen_span_begin(nc_context* c) {
  if (!(c->cfg.flags & NC_FLAG_TIMING) || c->gen_open) return;
  cudaEventCreate(&c->gen_a);
  cudaEventRecord(c->gen_a, c->stream);
  c->gen_open = true;
}
void gen_span_end(nc_context* c) {
  if (!c->gen_open) return;
  Span s{};
  s.phase = NC_PHASE_GENERATE;
  s.is_pass = false;
  s.a = c->gen_a;
  cudaEventCreate(&s.b);
  cudaEventRecord(s.b, c->stream);
  c->spans.push_back(s);
  c->gen_open = false;
}

BlockMap make_map(const nc_context* c) {
  BlockMap m{};
  m.table = c->d_table;
  m.B = c->B;
  m.off_tgt = c->off_tgt;
  m.off_w = c->off_w;
  m.off_d = c->off_d;
  if ((c->B & (c->B - 1)) == 0) {
    m.shift = bit_width_u64(c->B) - 1;
    m.magic = 0;
  } else {
    m.shift = 0xffffffffu;
    m.magic = (uint64_t)(((unsigned __int128)1 << 64) / c->B) + 1;
  }
  return m;
}

bool dist_ok(const nc_dist& d) {
  if (std::isnan(d.mean) || std::isnan(d.sd) || std::isnan(d.lo) || std::isnan(d.hi)) return false;
  if (std::isinf(d.mean) || std::isinf(d.sd)) return false;
  return d.sd >= 0.0 && d.lo <= d.hi;
}

// Q6: largest number of steps a projection's delay can take.
double delay_bound_steps(const nc_dist& d, double inv_dt) {
  double top = d.mean + kZMax * d.sd;
  if (top > d.hi) top = d.hi;
  if (top < d.lo) top = d.lo;
  return std::floor(top * inv_dt + 0.5);
}

SynConst make_syn(const nc_context* c, const nc_syn_spec& s) {
  SynConst k{};
  k.w_mean = (float)s.weight.mean;
  k.w_sd = (float)s.weight.sd;
  k.w_lo = (float)s.weight.lo;
  k.w_hi = (float)s.weight.hi;
  k.d_mean = (float)s.delay_ms.mean;
  k.d_sd = (float)s.delay_ms.sd;
  k.d_lo = (float)s.delay_ms.lo;
  k.d_hi = (float)s.delay_ms.hi;
  k.inv_dt = (float)c->inv_dt;
  // Guard band: the error of z1 (bounded in the kernel from r) enters x scaled
  // by sd / dt; 32 relative fp32 ulps of x cover the fp32 roundings of mean, sd, the bounds, 1/dt and of the
  // products; plus a small floor.
  const double scale = std::fabs(s.delay_ms.sd) * c->inv_dt;
  k.eps_a = (float)(scale * (double)kErrRa);
  k.eps_b = (float)(scale * ((double)kErrRb + (double)kErrTrig));
  k.eps_rel = (float)(32.0 / 16777216.0);
  k.eps_abs = (c->cfg.flags & NC_FLAG_EXACT_FP64) ? INFINITY : 1e-6f;
  k.dd_mean = s.delay_ms.mean;
  k.dd_sd = s.delay_ms.sd;
  k.dd_lo = s.delay_ms.lo;
  k.dd_hi = s.delay_ms.hi;
  k.dinv_dt = c->inv_dt;
  k.dw_mean = s.weight.mean;
  k.dw_sd = s.weight.sd;
  k.dw_lo = s.weight.lo;
  k.dw_hi = s.weight.hi;
  return k;
}

// Eq. 1: allocate floor((N_conns + N_newconns + B - 1) / B) - N_blocks new blocks and refresh
// the device-side table.  On failure nothing is kept.
int reserve_blocks(nc_context* c, uint64_t n_new) {
  const uint64_t want = (c->n_conns + n_new + c->B - 1) / c->B;
  const size_t have = c->blocks.size();
  if (want <= have) return NC_OK;
  std::vector<void*> fresh;
  for (uint64_t b = have; b < want; ++b) {
    void* p = dev_alloc(c, c->block_bytes);
    if (!p) {
      for (void* q : fresh) dev_free(c, q);
      return fail(c, NC_ERR_OOM, "out of device memory allocating a connection block");
    }
    fresh.push_back(p);
  }
  if (want > c->table_cap) {
    const size_t cap = std::max<size_t>(1024, (size_t)want * 2);
    uint64_t* t = (uint64_t*)dev_alloc(c, cap * sizeof(uint64_t));
    if (!t) {
      for (void* q : fresh) dev_free(c, q);
      return fail(c, NC_ERR_OOM, "out of device memory allocating the block table");
    }
    dev_free_later(c, c->d_table);  // earlier kernels may still read the old table
    c->d_table = t;
    c->table_cap = cap;
    c->blocks.insert(c->blocks.end(), fresh.begin(), fresh.end());
    NC_CUDA(c, cudaMemcpyAsync(c->d_table, c->blocks.data(), c->blocks.size() * sizeof(uint64_t),
                               cudaMemcpyHostToDevice, c->stream));
  } else {
    c->blocks.insert(c->blocks.end(), fresh.begin(), fresh.end());
    NC_CUDA(c, cudaMemcpyAsync(c->d_table + have, c->blocks.data() + have, (want - have) * sizeof(uint64_t),
                               cudaMemcpyHostToDevice, c->stream));
  }
  return NC_OK;
}

// Generation kernels write disjoint ranges, so consecutive launches may overlap: programmatic dependent launch
// lets the next kernel of the stream start while the previous one drains (each kernel waits for its predecessor
// before it exits, so completion stays in stream order).  NC_NO_PDL=1 in the environment disables it.
bool use_pdl() {
  static const bool on = [] {
    const char* e = getenv("NC_NO_PDL");
    return !(e && atoi(e) != 0);
  }();
  return on;
}

template <int RULE, bool ARR>
cudaError_t launch_generate_as(nc_context* c, const GenParams& p) {
  const uint64_t first_tile = p.pos0 / kGenTile;
  const uint64_t last_tile = (p.pos0 + p.n - 1) / kGenTile;
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)(last_tile - first_tile + 1));
  cfg.blockDim = dim3(kGenThreads);
  cfg.dynamicSmemBytes = 0;
  cfg.stream = c->stream;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = use_pdl() ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, generate_kernel<RULE, ARR>, p);
}

template <int RULE>
cudaError_t launch_generate(nc_context* c, const GenParams& p) {
  return (p.src_nodes || p.tgt_nodes) ? launch_generate_as<RULE, true>(c, p) : launch_generate_as<RULE, false>(c, p);
}

int device_scan(nc_context* c, const uint32_t* in, uint32_t* out, uint64_t n, uint32_t* partial, uint64_t* total) {
  const uint64_t chunks = (n + kScanChunk - 1) / kScanChunk;
  scan_reduce_kernel<<<(unsigned)chunks, kScanThreads, 0, c->stream>>>(in, n, partial);
  NC_LAUNCH_CHECK(c, "scan_reduce");
  scan_partials_kernel<<<1, kScanThreads, 0, c->stream>>>(partial, chunks, total);
  NC_LAUNCH_CHECK(c, "scan_partials");
  scan_downsweep_kernel<<<(unsigned)chunks, kScanThreads, 0, c->stream>>>(in, n, partial, out);
  NC_LAUNCH_CHECK(c, "scan_downsweep");
  return NC_OK;
}

// Pair-mask path: pairwise_bernoulli (trials = true), and -- reading A2 -- one_to_one / all_to_all with the equal-id
// pairs left out (trials = false: every pair accepted, then the autapses cleared).  self_tgt: device array for
// pair_mask_clear_autapses_kernel when node arrays are in use, NULL for ranges.
int connect_bernoulli(nc_context* c, GenParams gp, double p, uint32_t seed_lo, uint32_t seed_hi, bool trials = true,
                      bool one_to_one = false, bool no_autapses = false, const uint32_t* self_tgt = nullptr) {
  const uint64_t n_pairs = one_to_one ? (uint64_t)gp.n_src : (uint64_t)gp.n_src * gp.n_tgt;
  const uint64_t T = trials ? (uint64_t)std::floor(std::ldexp(p, 32)) : (1ull << 32);  // Q14
  if (T == 0) return NC_OK;                                    // realised probability 0: nothing to create
  const uint64_t n_tiles = (n_pairs + kBernTile - 1) / kBernTile;
  if (n_tiles > 0x7fffffffull) return fail(c, NC_ERR_CAPACITY, "pairwise_bernoulli: too many pairs for one call");
  const uint64_t n_words = (n_pairs + 31) / 32;
  const uint64_t chunks = (n_tiles + kScanChunk - 1) / kScanChunk;
  uint32_t* mask = (uint32_t*)dev_alloc(c, n_words * 4);
  uint32_t* tile_count = (uint32_t*)dev_alloc(c, n_tiles * 4);
  uint32_t* tile_off = (uint32_t*)dev_alloc(c, n_tiles * 4);
  uint32_t* partial = (uint32_t*)dev_alloc(c, chunks * 4);
  uint64_t* d_total = (uint64_t*)dev_alloc(c, 8);
  auto drop = [&]() {
    dev_free_later(c, mask); dev_free_later(c, tile_count); dev_free_later(c, tile_off);
    dev_free_later(c, partial); dev_free_later(c, d_total);
  };
  if (!mask || !tile_count || !tile_off || !partial || !d_total) {
    drop();
    return fail(c, NC_ERR_OOM, "out of device memory for pairwise_bernoulli scratch");
  }
  uint64_t total = 0;
  gen_span_end(c);
  {
    Scope sc(c, NC_PHASE_GENERATE);
    PairMaskParams pm{};
    pm.n_pairs = n_pairs;
    pm.n_src = gp.n_src;
    pm.n_tgt = gp.n_tgt;
    pm.s0 = gp.s0;
    pm.t0 = gp.t0;
    pm.one_to_one = one_to_one ? 1u : 0u;
    pm.self_tgt = self_tgt;
    pm.mask = mask;
    pm.tile_count = tile_count;
    if (trials) {
      BernParams bp{};
      bp.n_pairs = n_pairs;
      bp.threshold = T;
      bp.rng = make_philox_stream(seed_lo, seed_hi, c->n_proj, 1u);
      bp.mask = mask;
      bp.tile_count = tile_count;
      bernoulli_trials_kernel<<<(unsigned)n_tiles, kBernThreads, 0, c->stream>>>(bp);
      NC_LAUNCH_CHECK(c, "bernoulli_trials");
    } else {
      pair_mask_fill_kernel<<<(unsigned)n_tiles, kBernThreads, 0, c->stream>>>(pm);
      NC_LAUNCH_CHECK(c, "pair_mask_fill");
    }
    if (no_autapses) {
      pair_mask_clear_autapses_kernel<<<(gp.n_src + 255) / 256, 256, 0, c->stream>>>(pm);
      NC_LAUNCH_CHECK(c, "pair_mask_clear_autapses");
    }
    int rc = device_scan(c, tile_count, tile_off, n_tiles, partial, d_total);
    if (rc != NC_OK) {
      drop();
      return rc;
    }
    NC_CUDA(c, cudaMemcpyAsync(&total, d_total, 8, cudaMemcpyDeviceToHost, c->stream));
  }
  NC_CUDA(c, cudaStreamSynchronize(c->stream));  // the exact count decides the allocation
  release_deferred(c);  // the stream is idle: scratch of earlier calls (masks, tables) goes back before the blocks are reserved
  if (c->n_conns + total > kMaxConns) {
    drop();
    return fail(c, NC_ERR_CAPACITY, "more than 2^32-1 connections");
  }
  int rc = reserve_blocks(c, total);
  if (rc != NC_OK) {
    drop();
    return rc;
  }
  if (total > 0) {
    Scope sc(c, NC_PHASE_GENERATE);
    BernWriteParams wp{};
    wp.g = gp;
    wp.g.map = make_map(c);
    wp.g.pos0 = c->n_conns;
    wp.g.n = total;
    wp.n_pairs = n_pairs;
    wp.one_to_one = one_to_one ? 1u : 0u;
    wp.mask = mask;
    wp.tile_offset = tile_off;
    bernoulli_write_kernel<<<(unsigned)n_tiles, kBernThreads, 0, c->stream>>>(wp);
    NC_LAUNCH_CHECK(c, "bernoulli_write");
  }
  drop();
  c->n_conns += total;
  return NC_OK;
}

PassPlan plan_passes(uint32_t key_bits) {
  PassPlan pl{};
  pl.n_passes = (key_bits + kRadixBits - 1) / kRadixBits;
  uint32_t left = key_bits, shift = 0;
  for (uint32_t i = 0; i < pl.n_passes; ++i) {
    const uint32_t b = (left + (pl.n_passes - i) - 1) / (pl.n_passes - i);  // spread evenly, <= 8
    pl.shift[i] = shift;
    pl.bits[i] = b;
    shift += b;
    left -= b;
  }
  return pl;
}

template <typename KeyT>
int sort_and_index(nc_context* c, const PassPlan& plan) {
  using Smem = OnesweepSmem<KeyT, kSortThreads, kSortItems>;
  const uint32_t n = (uint32_t)c->n_conns;
  const uint32_t N = c->n_nodes;
  const uint64_t n_tiles = ((uint64_t)n + Smem::kTile - 1) / Smem::kTile;
  const BlockMap map = make_map(c);

  KeyT* keys[2] = {(KeyT*)dev_alloc(c, (size_t)n * sizeof(KeyT)),
                   plan.n_passes > 1 ? (KeyT*)dev_alloc(c, (size_t)n * sizeof(KeyT)) : nullptr};
  uint32_t* vals[2] = {(uint32_t*)dev_alloc(c, (size_t)n * 4),
                       plan.n_passes > 1 ? (uint32_t*)dev_alloc(c, (size_t)n * 4) : nullptr};
  uint32_t* ghist = (uint32_t*)dev_alloc(c, kMaxPasses * kRadix * 4);
  uint32_t* bin_start = (uint32_t*)dev_alloc(c, kMaxPasses * kRadix * 4);
  uint64_t* status = (uint64_t*)dev_alloc(c, n_tiles * kRadix * 8);
  uint32_t* tickets = (uint32_t*)dev_alloc(c, (kMaxPasses + 1) * 4);  // + the look-back error flag
  c->s_src = (uint32_t*)dev_alloc(c, (size_t)n * 4);
  c->s_tgt = (uint32_t*)dev_alloc(c, (size_t)n * 4);
  c->s_w = (float*)dev_alloc(c, (size_t)n * 4);
  c->s_d = (uint16_t*)dev_alloc(c, (size_t)n * 2);
  const uint64_t head_tiles = ((uint64_t)n + kHeadTile - 1) / kHeadTile;
  const uint64_t head_chunks = (head_tiles + kScanChunk - 1) / kScanChunk;
  uint32_t* tile_heads = (uint32_t*)dev_alloc(c, head_tiles * 4);
  uint32_t* tile_head_off = (uint32_t*)dev_alloc(c, head_tiles * 4);
  uint32_t* head_partial = (uint32_t*)dev_alloc(c, head_chunks * 4);
  uint64_t* d_total_groups = (uint64_t*)dev_alloc(c, 8);
  bool ok = keys[0] && vals[0] && ghist && bin_start && status && tickets && c->s_src && c->s_tgt && c->s_w &&
            c->s_d && tile_heads && tile_head_off && head_partial && d_total_groups;
  if (plan.n_passes > 1) ok = ok && keys[1] && vals[1];
  auto drop_scratch = [&](int final_buf) {
    for (int i = 0; i < 2; ++i) {
      dev_free_later(c, keys[i]);
      if (i != final_buf) dev_free_later(c, vals[i]);
    }
    dev_free_later(c, ghist); dev_free_later(c, bin_start); dev_free_later(c, status); dev_free_later(c, tickets);
    dev_free_later(c, tile_heads); dev_free_later(c, tile_head_off); dev_free_later(c, head_partial);
    dev_free_later(c, d_total_groups);
  };
  if (!ok) {
    drop_scratch(-1);
    return fail(c, NC_ERR_OOM, "out of device memory in nc_finalize");
  }

  // ---- a9: digit histograms of all passes + their exclusive scans ----
  {
    Scope sc(c, NC_PHASE_HISTOGRAM);
    NC_CUDA(c, cudaMemsetAsync(ghist, 0, kMaxPasses * kRadix * 4, c->stream));
    NC_CUDA(c, cudaMemsetAsync(tickets, 0, (kMaxPasses + 1) * 4, c->stream));
    NC_CUDA(c, cudaMemsetAsync(status, 0, n_tiles * kRadix * 8, c->stream));
    const unsigned grid = (unsigned)(((uint64_t)n + kHistThreads * kHistItems - 1) / (kHistThreads * kHistItems));
    if (c->B % 4 == 0) histogram_kernel<KeyT, true><<<grid, kHistThreads, 0, c->stream>>>(map, n, c->delay_bits, plan, ghist);
    else histogram_kernel<KeyT, false><<<grid, kHistThreads, 0, c->stream>>>(map, n, c->delay_bits, plan, ghist);
    NC_LAUNCH_CHECK(c, "histogram");
    bin_scan_kernel<<<plan.n_passes, kRadix, 0, c->stream>>>(ghist, bin_start);
    NC_LAUNCH_CHECK(c, "bin_scan");
  }

  // ---- a10: onesweep passes, ping-pong between the two buffers ----
  const size_t smem = sizeof(Smem);
  NC_CUDA(c, cudaFuncSetAttribute(onesweep_kernel<KeyT, true, kSortThreads, kSortItems>,
                                  cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  NC_CUDA(c, cudaFuncSetAttribute(onesweep_kernel<KeyT, false, kSortThreads, kSortItems>,
                                  cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int cur = 0;
  {
    Scope sc(c, NC_PHASE_SORT);
    for (uint32_t ps = 0; ps < plan.n_passes; ++ps) {
      Scope pass_sc(c, NC_PHASE_SORT, true);
      SortPassParams<KeyT> sp{};
      sp.map = map;
      sp.delay_bits = c->delay_bits;
      sp.n = n;
      const int dst = ps == 0 ? 0 : 1 - cur;
      sp.keys_in = ps == 0 ? nullptr : keys[cur];
      sp.vals_in = ps == 0 ? nullptr : vals[cur];
      sp.keys_out = keys[dst];
      sp.vals_out = vals[dst];
      sp.shift = plan.shift[ps];
      sp.bits = plan.bits[ps];
      sp.bin_start = bin_start + ps * kRadix;
      sp.status = status;
      sp.ticket = tickets + ps;
      sp.error_flag = tickets + kMaxPasses;
      sp.epoch = (uint64_t)(ps + 1) << 42;
      if (ps == 0) {
        onesweep_kernel<KeyT, true, kSortThreads, kSortItems><<<(unsigned)n_tiles, kSortThreads, smem, c->stream>>>(sp);
      } else {
        onesweep_kernel<KeyT, false, kSortThreads, kSortItems><<<(unsigned)n_tiles, kSortThreads, smem, c->stream>>>(sp);
      }
      NC_LAUNCH_CHECK(c, "onesweep");
      cur = dst;
    }
  }
  c->perm = vals[cur];

  // ---- a11: permutation apply ----
  {
    Scope sc(c, NC_PHASE_PERMUTE);
    const unsigned grid = (unsigned)(((uint64_t)n + kPermThreads - 1) / kPermThreads);
    permute_kernel<KeyT><<<grid, kPermThreads, 0, c->stream>>>(map, n, c->delay_bits, keys[cur], c->perm, c->s_src,
                                                              c->s_tgt, c->s_w, c->s_d);
    NC_LAUNCH_CHECK(c, "permute");
  }

  // ---- a12-a14: heads, scan, compaction, per-source offsets ----
  uint64_t total_groups = 0;
  uint32_t lookback_error = 0;
  {
    Scope sc(c, NC_PHASE_INDEX);
    head_count_kernel<<<(unsigned)head_tiles, kHeadThreads, 0, c->stream>>>(PackedKeys<KeyT>{keys[cur], c->delay_bits}, n, tile_heads);
    NC_LAUNCH_CHECK(c, "head_count");
    int rc = device_scan(c, tile_heads, tile_head_off, head_tiles, head_partial, d_total_groups);
    if (rc != NC_OK) return rc;
    NC_CUDA(c, cudaMemcpyAsync(&total_groups, d_total_groups, 8, cudaMemcpyDeviceToHost, c->stream));
    NC_CUDA(c, cudaMemcpyAsync(&lookback_error, tickets + kMaxPasses, 4, cudaMemcpyDeviceToHost, c->stream));
  }
  NC_CUDA(c, cudaStreamSynchronize(c->stream));  // total_groups sizes the group arrays
  release_deferred(c);
  if (lookback_error) {
    drop_scratch(cur);
    return fail(c, NC_ERR_CUDA, "onesweep look-back timed out");
  }
  c->total_groups = (uint32_t)total_groups;
  c->group_start = (uint32_t*)dev_alloc(c, (size_t)total_groups * 4);
  c->group_delay = (uint16_t*)dev_alloc(c, (size_t)total_groups * 2);
  if (!c->group_start || !c->group_delay) {
    drop_scratch(cur);
    return fail(c, NC_ERR_OOM, "out of device memory for the group arrays");
  }
  {
    Scope sc(c, NC_PHASE_INDEX);
    IndexOut io{c->src_offsets, c->group_ptr, c->group_start, c->group_delay, N};
    index_scatter_kernel<<<(unsigned)head_tiles, kHeadThreads, 0, c->stream>>>(PackedKeys<KeyT>{keys[cur], c->delay_bits}, n,
                                                                              tile_head_off, d_total_groups, io);
    NC_LAUNCH_CHECK(c, "index_scatter");
    index_finish_kernel<<<(N + 255) / 256, 256, 0, c->stream>>>(c->src_offsets, c->group_ptr, N, c->out_degree,
                                                               c->group_count, c->d_max + 1);
    NC_LAUNCH_CHECK(c, "index_finish");
  }
  drop_scratch(cur);
  return NC_OK;
}

// Record-carrying organisation step (keys of <= 32 bits): histogram, P onesweep passes that move whole
// connections, final pass writes the sorted SoA arrays; then the index over (source, delay).
// Launch shape of the record pass: 384 threads x 8 records, registers budgeted for 3 CTAs per SM, shared-memory
// peer masks (the best of the eight shapes tried on B200, profiles/r01_baseline.md).
struct RecShape {
  int threads, items;
};
constexpr RecShape kRecShapes[] = {{384, 8}};

int rec_variant() { return 0; }

template <bool FIRST, bool LAST, int THREADS, int ITEMS, int MIN_CTAS, int MATCH>
int launch_rec_pass_shape(nc_context* c, const SortRecParams& sp) {
  using Smem = OnesweepRecSmem<THREADS, ITEMS>;
  auto kern = onesweep_rec_kernel<FIRST, LAST, THREADS, ITEMS, MIN_CTAS, MATCH>;
  const uint64_t n_tiles = ((uint64_t)sp.n + Smem::kTile - 1) / Smem::kTile;
  NC_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem)));
  kern<<<(unsigned)n_tiles, THREADS, sizeof(Smem), c->stream>>>(sp);
  NC_LAUNCH_CHECK(c, "onesweep_rec");
  return NC_OK;
}

template <bool FIRST, bool LAST>
int launch_rec_pass(nc_context* c, const SortRecParams& sp, int /*variant*/) {
  return launch_rec_pass_shape<FIRST, LAST, 384, 8, 3, kMatchSmem>(c, sp);
}

int build_index_from_sorted(nc_context* c, uint32_t n, uint32_t* lookback_flag);

int sort_carry_and_index(nc_context* c, const PassPlan& plan) {
  const uint32_t n = (uint32_t)c->n_conns;
  const int variant = rec_variant();
  const uint64_t tile = (uint64_t)kRecShapes[variant].threads * kRecShapes[variant].items;
  const uint64_t n_tiles = ((uint64_t)n + tile - 1) / tile;
  const BlockMap map = make_map(c);
  const uint32_t P = plan.n_passes;

  uint4* recs[2] = {P > 1 ? (uint4*)dev_alloc(c, (size_t)n * 16) : nullptr,
                    P > 2 ? (uint4*)dev_alloc(c, (size_t)n * 16) : nullptr};
  uint32_t* ghist = (uint32_t*)dev_alloc(c, kMaxPasses * kRadix * 4);
  uint32_t* bin_start = (uint32_t*)dev_alloc(c, kMaxPasses * kRadix * 4);
  uint64_t* status = (uint64_t*)dev_alloc(c, n_tiles * kRadix * 8);
  uint32_t* tickets = (uint32_t*)dev_alloc(c, (kMaxPasses + 1) * 4);
  c->s_src = (uint32_t*)dev_alloc(c, (size_t)n * 4);
  c->s_tgt = (uint32_t*)dev_alloc(c, (size_t)n * 4);
  c->s_w = (float*)dev_alloc(c, (size_t)n * 4);
  c->s_d = (uint16_t*)dev_alloc(c, (size_t)n * 2);
  c->perm = (uint32_t*)dev_alloc(c, (size_t)n * 4);
  bool ok = ghist && bin_start && status && tickets && c->s_src && c->s_tgt && c->s_w && c->s_d && c->perm;
  if (P > 1) ok = ok && recs[0];
  if (P > 2) ok = ok && recs[1];
  auto drop_scratch = [&]() {
    dev_free_later(c, recs[0]); dev_free_later(c, recs[1]);
    dev_free_later(c, ghist); dev_free_later(c, bin_start); dev_free_later(c, status); dev_free_later(c, tickets);
  };
  if (!ok) {
    drop_scratch();
    return fail(c, NC_ERR_OOM, "out of device memory in nc_finalize");
  }
  {
    Scope sc(c, NC_PHASE_HISTOGRAM);
    NC_CUDA(c, cudaMemsetAsync(ghist, 0, kMaxPasses * kRadix * 4, c->stream));
    NC_CUDA(c, cudaMemsetAsync(tickets, 0, (kMaxPasses + 1) * 4, c->stream));
    NC_CUDA(c, cudaMemsetAsync(status, 0, n_tiles * kRadix * 8, c->stream));
    const unsigned grid = (unsigned)(((uint64_t)n + kHistThreads * kHistItems - 1) / (kHistThreads * kHistItems));
    if (c->B % 4 == 0) histogram_kernel<uint32_t, true><<<grid, kHistThreads, 0, c->stream>>>(map, n, c->delay_bits, plan, ghist);
    else histogram_kernel<uint32_t, false><<<grid, kHistThreads, 0, c->stream>>>(map, n, c->delay_bits, plan, ghist);
    NC_LAUNCH_CHECK(c, "histogram");
    bin_scan_kernel<<<P, kRadix, 0, c->stream>>>(ghist, bin_start);
    NC_LAUNCH_CHECK(c, "bin_scan");
  }
  {
    Scope sc(c, NC_PHASE_SORT);
    int cur = -1;
    for (uint32_t ps = 0; ps < P; ++ps) {
      Scope pass_sc(c, NC_PHASE_SORT, true);
      const bool first = ps == 0, last = ps + 1 == P;
      SortRecParams sp{};
      sp.map = map;
      sp.delay_bits = c->delay_bits;
      sp.n = n;
      const int dst = cur < 0 ? 0 : 1 - cur;
      sp.recs_in = first ? nullptr : recs[cur];
      sp.recs_out = last ? nullptr : recs[dst];
      sp.out_src = c->s_src;
      sp.out_tgt = c->s_tgt;
      sp.out_w = c->s_w;
      sp.out_d = c->s_d;
      sp.out_perm = c->perm;
      sp.shift = plan.shift[ps];
      sp.bits = plan.bits[ps];
      sp.bin_start = bin_start + ps * kRadix;
      sp.status = status;
      sp.ticket = tickets + ps;
      sp.error_flag = tickets + kMaxPasses;
      sp.epoch = (uint64_t)(ps + 1) << 42;
      int rc;
      if (first && last) rc = launch_rec_pass<true, true>(c, sp, variant);
      else if (first) rc = launch_rec_pass<true, false>(c, sp, variant);
      else if (last) rc = launch_rec_pass<false, true>(c, sp, variant);
      else rc = launch_rec_pass<false, false>(c, sp, variant);
      if (rc != NC_OK) return rc;
      cur = dst;
    }
  }
  int rc = build_index_from_sorted(c, n, tickets + kMaxPasses);
  drop_scratch();
  return rc;
}

// Default organisation step for keys of <= 32 bits (nc_sort_split.cuh): per digit pass, per-tile digit counts ->
// scan -> scatter of whole connections; the last pass writes the sorted SoA arrays; then the index.
struct SplitShape {
  int warps, items;
};
constexpr SplitShape kSplitShapes[] = {{8, 16}, {12, 8}};

int split_variant() {
  const char* e = getenv("NC_SPLIT_VARIANT");
  const int v = e ? atoi(e) : 0;
  return (v >= 0 && v < (int)(sizeof(kSplitShapes) / sizeof(kSplitShapes[0]))) ? v : 0;
}

template <bool FIRST, bool LAST, int WARPS, int ITEMS, int MIN_CTAS, int MATCH>
int launch_scatter_match(nc_context* c, const ScatterParams& sp, uint32_t n_tiles) {
  using Smem = ScatterSmem<WARPS, ITEMS, MATCH == kMatchSmem>;
  auto kern = scatter_pass_kernel<FIRST, LAST, WARPS, ITEMS, MIN_CTAS, MATCH>;
  NC_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem)));
  kern<<<n_tiles, WARPS * 32, sizeof(Smem), c->stream>>>(sp);
  NC_LAUNCH_CHECK(c, "scatter_pass");
  return NC_OK;
}

template <bool FIRST, bool LAST, int WARPS, int ITEMS, int MIN_CTAS>
int launch_scatter_shape(nc_context* c, const ScatterParams& sp, uint32_t n_tiles) {
  return launch_scatter_match<FIRST, LAST, WARPS, ITEMS, MIN_CTAS, kMatchBallot>(c, sp, n_tiles);
}

template <bool FIRST, bool LAST>
int launch_scatter_pass(nc_context* c, const ScatterParams& sp, uint32_t n_tiles, int variant) {
  switch (variant) {
    case 1: return launch_scatter_shape<FIRST, LAST, 12, 8, 3>(c, sp, n_tiles);
    default: return launch_scatter_shape<FIRST, LAST, 8, 16, 2>(c, sp, n_tiles);
  }
}

// NC_FLAG_SORT_BULK: the same pass as a persistent kernel fed by cp.async.bulk (nc_sort_bulk.cuh), one CTA per SM.
template <bool FIRST, bool LAST>
int launch_scatter_bulk(nc_context* c, const ScatterParams& sp, uint32_t n_tiles) {
  auto kern = scatter_bulk_kernel<FIRST, LAST>;
  NC_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(BulkSmem)));
  int sms = 0;
  NC_CUDA(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device));
  kern<<<std::min<uint32_t>(n_tiles, (uint32_t)sms), kBulkWarps * 32, sizeof(BulkSmem), c->stream>>>(sp, n_tiles);
  NC_LAUNCH_CHECK(c, "scatter_bulk");
  return NC_OK;
}

int sort_split_and_index(nc_context* c, const PassPlan& plan) {
  const uint32_t n = (uint32_t)c->n_conns;
  const bool bulk = (c->cfg.flags & NC_FLAG_SORT_BULK) != 0;
  const int variant = bulk ? 0 : split_variant();  // the bulk kernel works on the tiles of shape 0
  const uint32_t kSplitTile = (uint32_t)kSplitShapes[variant].warps * 32u * (uint32_t)kSplitShapes[variant].items;
  const uint32_t n_tiles = (uint32_t)(((uint64_t)n + kSplitTile - 1) / kSplitTile);
  const uint32_t n_chunks = (n_tiles + kScanChunkTiles - 1) / kScanChunkTiles;
  const BlockMap map = make_map(c);
  const uint32_t P = plan.n_passes;

  uint4* recs[2] = {P > 1 ? (uint4*)dev_alloc(c, (size_t)n * 16) : nullptr,
                    P > 2 ? (uint4*)dev_alloc(c, (size_t)n * 16) : nullptr};
  uint8_t* dig = P > 1 ? (uint8_t*)dev_alloc(c, (size_t)n) : nullptr;
  uint16_t* counts = (uint16_t*)dev_alloc(c, (size_t)n_tiles * kRadix * 2);
  uint32_t* offs = (uint32_t*)dev_alloc(c, (size_t)n_tiles * kRadix * 4);
  uint32_t* chunk = (uint32_t*)dev_alloc(c, (size_t)n_chunks * kRadix * 4);
  c->s_src = (uint32_t*)dev_alloc(c, (size_t)n * 4);
  c->s_tgt = (uint32_t*)dev_alloc(c, (size_t)n * 4);
  c->s_w = (float*)dev_alloc(c, (size_t)n * 4);
  c->s_d = (uint16_t*)dev_alloc(c, (size_t)n * 2);
  c->perm = (uint32_t*)dev_alloc(c, (size_t)n * 4);
  bool ok = counts && offs && chunk && c->s_src && c->s_tgt && c->s_w && c->s_d && c->perm;
  if (P > 1) ok = ok && recs[0] && dig;
  if (P > 2) ok = ok && recs[1];
  auto drop_scratch = [&]() {
    dev_free_later(c, recs[0]); dev_free_later(c, recs[1]); dev_free_later(c, dig);
    dev_free_later(c, counts); dev_free_later(c, offs); dev_free_later(c, chunk);
  };
  if (!ok) {
    drop_scratch();
    return fail(c, NC_ERR_OOM, "out of device memory in nc_finalize");
  }
  int cur = -1;
  for (uint32_t ps = 0; ps < P; ++ps) {
    const bool first = ps == 0, last = ps + 1 == P;
    {
      Scope sc(c, NC_PHASE_HISTOGRAM);
      if (first) {
        if (c->B % 4 == 0)
          tile_count_first_kernel<true><<<n_tiles, kCountThreads, 0, c->stream>>>(map, n, kSplitTile, c->delay_bits,
                                                                                plan.shift[0], plan.bits[0], counts);
        else
          tile_count_first_kernel<false><<<n_tiles, kCountThreads, 0, c->stream>>>(map, n, kSplitTile, c->delay_bits,
                                                                                 plan.shift[0], plan.bits[0], counts);
      } else {
        tile_count_bytes_kernel<<<(n_tiles + kCountTilesPerCta - 1) / kCountTilesPerCta, kCountThreads, 0, c->stream>>>(
            dig, n, kSplitTile, n_tiles, counts);
      }
      NC_LAUNCH_CHECK(c, "tile_count");
      chunk_total_kernel<<<n_chunks, kRadix, 0, c->stream>>>(counts, n_tiles, chunk);
      NC_LAUNCH_CHECK(c, "chunk_total");
      chunk_scan_kernel<<<1, kRadix * kChunkScanSegs, 0, c->stream>>>(chunk, n_chunks);
      NC_LAUNCH_CHECK(c, "chunk_scan");
      tile_offsets_kernel<<<n_chunks, kRadix, 0, c->stream>>>(counts, n_tiles, chunk, offs);
      NC_LAUNCH_CHECK(c, "tile_offsets");
    }
    {
      Scope sc(c, NC_PHASE_SORT);
      Scope pass_sc(c, NC_PHASE_SORT, true);
      ScatterParams sp{};
      sp.map = map;
      sp.delay_bits = c->delay_bits;
      sp.n = n;
      const int dst = cur < 0 ? 0 : 1 - cur;
      sp.recs_in = first ? nullptr : recs[cur];
      sp.recs_out = last ? nullptr : recs[dst];
      sp.dig_out = dig;
      sp.out_src = c->s_src;
      sp.out_tgt = c->s_tgt;
      sp.out_w = c->s_w;
      sp.out_d = c->s_d;
      sp.out_perm = c->perm;
      sp.shift = plan.shift[ps];
      sp.bits = plan.bits[ps];
      sp.next_shift = last ? 0 : plan.shift[ps + 1];
      sp.next_bits = last ? 0 : plan.bits[ps + 1];
      sp.offs = offs;
      int rc;
      static_assert(kBulkTile == 8 * 32 * 16, "the bulk kernel shares the tiles (and their offsets) of split shape 0");
      const bool bulk_first = bulk && c->B % kBulkTile == 0;  // a tile of the first pass must lie inside one block
      if (first && last) rc = bulk_first ? launch_scatter_bulk<true, true>(c, sp, n_tiles) : launch_scatter_pass<true, true>(c, sp, n_tiles, variant);
      else if (first) rc = bulk_first ? launch_scatter_bulk<true, false>(c, sp, n_tiles) : launch_scatter_pass<true, false>(c, sp, n_tiles, variant);
      else if (last) rc = bulk ? launch_scatter_bulk<false, true>(c, sp, n_tiles) : launch_scatter_pass<false, true>(c, sp, n_tiles, variant);
      else rc = bulk ? launch_scatter_bulk<false, false>(c, sp, n_tiles) : launch_scatter_pass<false, false>(c, sp, n_tiles, variant);
      if (rc != NC_OK) return rc;
      cur = dst;
    }
  }
  int rc = build_index_from_sorted(c, n, nullptr);
  drop_scratch();
  return rc;
}

// ---------------------------------------------------------------------------------------------------------------
// COPASS organisation (NC_FLAG_ORGANISE_COPASS; nc_copass.cuh): the connections are sorted inside
// their storage blocks with auxiliary memory of a few blocks instead of two more copies of everything.
// ---------------------------------------------------------------------------------------------------------------
constexpr uint32_t kCopassChunkTiles = 32;  // tiles per scan chunk: a block has few thousand tiles, keep the chunks short
struct CopassScratch {
  uint4* buf[2];   // intermediate records of the radix passes (one block each)
  uint8_t* dig;    // next-pass digit per record
  uint16_t* counts;
  uint32_t* offs;
  uint32_t* chunk;
};

// The underlying sort: stable radix passes over n <= B records.  Input: one storage block in its
// creation-order layout (from_storage; map addresses it as block 0; pos_base = its first creation position) or an
// array of records.  Output: n records at `out`.
int copass_sort_records(nc_context* c, const PassPlan& plan, const CopassScratch& sc, bool from_storage,
                        const BlockMap& map, uint32_t pos_base, const uint4* in, uint32_t n, uint4* out,
                        bool have_first_digits = false, char* final_block = nullptr) {
  // final_block: the last pass writes the block's final five arrays there instead of records at `out`
  const uint32_t kTile = (uint32_t)kSplitShapes[0].warps * 32u * (uint32_t)kSplitShapes[0].items;
  const uint32_t n_tiles = (n + kTile - 1) / kTile;
  const uint32_t n_chunks = (n_tiles + kCopassChunkTiles - 1) / kCopassChunkTiles;
  const uint32_t P = plan.n_passes;
  const uint4* cur_in = in;
  for (uint32_t ps = 0; ps < P; ++ps) {
    const bool storage = from_storage && ps == 0, last = ps + 1 == P;
    {
      Scope scp(c, NC_PHASE_HISTOGRAM);
      if (storage) {
        if (c->B % 4 == 0)
          tile_count_first_kernel<true><<<n_tiles, kCountThreads, 0, c->stream>>>(map, n, kTile, c->delay_bits,
                                                                                plan.shift[0], plan.bits[0], sc.counts);
        else
          tile_count_first_kernel<false><<<n_tiles, kCountThreads, 0, c->stream>>>(map, n, kTile, c->delay_bits,
                                                                                 plan.shift[0], plan.bits[0], sc.counts);
      } else if (ps == 0 && !have_first_digits) {
        tile_count_recs_kernel<<<n_tiles, kCountThreads, 0, c->stream>>>(in, n, kTile, plan.shift[0], plan.bits[0],
                                                                        sc.counts);
      } else {
        // a block has a few thousand tiles: two per CTA fill the machine, eight would leave most SMs idle
        tile_count_bytes_kernel<<<(n_tiles + 1) / 2, kCountThreads, 0, c->stream>>>(sc.dig, n, kTile, n_tiles, sc.counts, 2u);
      }
      NC_LAUNCH_CHECK(c, "tile_count");
      chunk_total_kernel<<<n_chunks, kRadix, 0, c->stream>>>(sc.counts, n_tiles, sc.chunk, kCopassChunkTiles);
      NC_LAUNCH_CHECK(c, "chunk_total");
      chunk_scan_kernel<<<1, kRadix * kChunkScanSegs, 0, c->stream>>>(sc.chunk, n_chunks);
      NC_LAUNCH_CHECK(c, "chunk_scan");
      tile_offsets_kernel<<<n_chunks, kRadix, 0, c->stream>>>(sc.counts, n_tiles, sc.chunk, sc.offs, kCopassChunkTiles);
      NC_LAUNCH_CHECK(c, "tile_offsets");
    }
    {
      Scope scp(c, NC_PHASE_SORT);
      Scope pass_sc(c, NC_PHASE_SORT, true);
      ScatterParams sp{};
      sp.map = map;
      sp.delay_bits = c->delay_bits;
      sp.n = n;
      sp.pos_base = pos_base;
      sp.recs_in = storage ? nullptr : cur_in;
      sp.recs_out = last ? out : sc.buf[ps & 1];
      sp.dig_out = sc.dig;
      const bool to_arrays = last && final_block != nullptr && !storage;
      if (to_arrays) {
        sp.out_src = (uint32_t*)final_block;
        sp.out_tgt = (uint32_t*)(final_block + c->off_tgt);
        sp.out_w = (float*)(final_block + c->off_w);
        sp.out_d = (uint16_t*)(final_block + c->off_d);
        sp.out_perm = (uint32_t*)(final_block + c->off_perm);
      }
      sp.shift = plan.shift[ps];
      sp.bits = plan.bits[ps];
      sp.next_shift = last ? 0 : plan.shift[ps + 1];
      sp.next_bits = last ? 0 : plan.bits[ps + 1];
      sp.offs = sc.offs;
      const int rc = storage     ? launch_scatter_pass<true, false>(c, sp, n_tiles, 0)
                     : to_arrays ? launch_scatter_pass<false, true>(c, sp, n_tiles, 0)
                                 : launch_scatter_pass<false, false>(c, sp, n_tiles, 0);
      if (rc != NC_OK) return rc;
      cur_in = sp.recs_out;
    }
  }
  return NC_OK;
}

// Extraction by hole filling (the default under NC_FLAG_ORGANISE_COPASS; DESIGN.md 8d "what differs").  The paper
// extracts output block b from the logical subarrays left by extraction b-1 and then shifts everything to the right
// (Fig. 6 C-E), i.e. ~k/2 copies of all connections.  Two observations remove the shift:
//  1. the left partitions of extraction b are the part of the first (b+1) B elements (in the stable order) that is
//     not among the first b B: all k-1 partitions can be taken on the ORIGINAL sorted blocks with m = (b+1) B, they
//     do not depend on one another and run as k-1 CTAs of one launch;
//  2. "the subarrays do not need to be stored in contiguous locations": a subarray is kept as a list of
//     extents.  Output block b is gathered into the spare block and sorted there; then ONE block (the one with the
//     most holes) is emptied into the holes the left partitions left in the other blocks and becomes the next spare.
//     Per extraction ~2 B records move instead of everything to the right of block b.
// The host reads the (k-1) k partition sizes once, plans every copy from them, uploads the commands and enqueues
// the rest without waiting again.  `spare` is the free physical block on entry and on return; c->blocks / d_table
// are rewritten at the end.
struct CopassExtent {
  uint32_t lo, hi;  // sorted positions [lo, hi) of the original block
  uint32_t phys;    // physical position (block id * B + slot) of element lo
};

int copass_extract_fill(nc_context* c, const PassPlan& plan, const CopassScratch& sc, void*& spare, uint32_t* st,
                        bool* blocks_are_final) {
  const uint32_t n = (uint32_t)c->n_conns;
  const uint64_t B = c->B;
  const uint32_t k = (uint32_t)c->blocks.size();
  const size_t k1 = (size_t)k + 1;  // (k + 1) B < 2^32 was checked before anything was rewritten
  auto block_n = [&](uint32_t b) { return (uint32_t)std::min<uint64_t>(B, (uint64_t)n - (uint64_t)b * B); };

  // ---- Fig. 6C for every output block at once ----
  uint32_t* part = (uint32_t*)dev_alloc(c, (size_t)(k - 1) * k * 4);  // m_i of every partition
  uint64_t* d_phys = (uint64_t*)dev_alloc(c, k1 * 8);
  std::vector<void*> phys(c->blocks.begin(), c->blocks.end());
  phys.push_back(spare);
  auto drop = [&]() {
    dev_free_later(c, part);
    dev_free_later(c, d_phys);
  };
  if (!part || !d_phys) {
    drop();
    return fail(c, NC_ERR_OOM, "out of device memory in nc_finalize (COPASS organisation)");
  }
  uint32_t *start = st, *len = st + k1;
  std::vector<uint32_t> M((size_t)(k - 1) * k);
  {
    Scope scp(c, NC_PHASE_COPASS);
    copass_init_subarrays_kernel<<<(k + 255) / 256, 256, 0, c->stream>>>(start, len, k, (uint32_t)B, n);
    NC_LAUNCH_CHECK(c, "copass_init_subarrays");
    const size_t smem = 7 * k1 * 4;
    auto kern = copass_partition_kernel<RecKeys>;
    NC_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    kern<<<k - 1, kCopassThreads, smem, c->stream>>>(RecKeys{make_map(c)}, k, (uint32_t)B, start, len, 0u, part, nullptr,
                                                    nullptr, nullptr, nullptr, nullptr, c->d_copass_totals, (uint32_t)B,
                                                    k);
    NC_LAUNCH_CHECK(c, "copass_partition");
    NC_CUDA(c, cudaMemcpyAsync(M.data(), part, (size_t)(k - 1) * k * 4, cudaMemcpyDeviceToHost, c->stream));
    NC_CUDA(c, cudaMemcpyAsync(d_phys, phys.data(), k1 * 8, cudaMemcpyHostToDevice, c->stream));
  }
  NC_CUDA(c, cudaStreamSynchronize(c->stream));  // the one wait of the organisation step: the plan needs the m_i
  release_deferred(c);

  // ---- plan (host): extents of every original block, holes per physical block, copy commands per step ----
  struct Step {
    size_t g0, g1, e0, e1;  // command ranges: gather into the spare block, evacuation of the victim
    uint32_t g_total, e_total, target;  // target = physical id the output block is assembled in
  };
  std::vector<uint32_t> cs, cd, cp;  // commands: source position, destination position, prefix inside the launch
  std::vector<Step> steps(k);
  std::vector<std::vector<CopassExtent>> ext(k);
  std::vector<std::vector<std::pair<uint32_t, uint32_t>>> holes(k + 1);  // per physical block: (position, length)
  std::vector<char> is_final(k + 1, 0);
  std::vector<uint32_t> final_of(k), prev(k, 0);
  for (uint32_t i = 0; i < k; ++i) ext[i].push_back(CopassExtent{0u, block_n(i), (uint32_t)((uint64_t)i * B)});
  if (block_n(k - 1) < B) holes[k - 1].push_back({(uint32_t)((uint64_t)(k - 1) * B + block_n(k - 1)), (uint32_t)(B - block_n(k - 1))});
  uint32_t F = k;
  for (uint32_t b = 0; b < k; ++b) {
    Step& sp = steps[b];
    sp.g0 = cs.size();
    sp.target = F;
    uint32_t at = 0;
    for (uint32_t i = 0; i < k; ++i) {  // left partitions in subarray order: ties stay in creation order
      const uint32_t cut = b + 1 < k ? M[(size_t)b * k + i] : block_n(i);
      if (cut < prev[i] || cut > block_n(i)) return fail(c, NC_ERR_CUDA, "COPASS plan: partition sizes are not nested");
      uint32_t need = cut - prev[i];
      prev[i] = cut;
      size_t used = 0;
      while (need > 0) {
        if (used >= ext[i].size()) return fail(c, NC_ERR_CUDA, "COPASS plan: a subarray ran out of extents");
        CopassExtent& x = ext[i][used];
        const uint32_t take = std::min(need, x.hi - x.lo);
        cs.push_back(x.phys);
        cd.push_back((uint32_t)((uint64_t)F * B) + at);
        cp.push_back(at);
        holes[x.phys / B].push_back({x.phys, take});
        at += take;
        x.lo += take;
        x.phys += take;
        need -= take;
        if (x.lo == x.hi) ++used;
      }
      ext[i].erase(ext[i].begin(), ext[i].begin() + used);
    }
    sp.g1 = cs.size();
    sp.g_total = at;
    if (at != block_n(b)) return fail(c, NC_ERR_CUDA, "COPASS plan: the left partitions do not add up to the block");
    final_of[b] = F;
    is_final[F] = 1;
    sp.e0 = sp.e1 = cs.size();
    sp.e_total = 0;
    if (b + 1 == k) break;
    // the victim: the block with the most free room; what lives in it moves into the holes of the others
    uint32_t V = 0xffffffffu;
    uint64_t best = 0;
    std::vector<uint64_t> room(k + 1, 0);
    for (uint32_t p = 0; p <= k; ++p) {
      if (is_final[p]) continue;
      for (auto& h : holes[p]) room[p] += h.second;
      if (V == 0xffffffffu || room[p] > best) {
        V = p;
        best = room[p];
      }
    }
    uint32_t hp = 0;      // physical block whose holes are being filled
    size_t hi_ = 0;       // index into holes[hp]
    uint32_t h_used = 0;  // how much of that hole is taken
    auto next_hole = [&]() -> bool {  // advance to a hole with room outside V and the final blocks
      for (;;) {
        if (hp > k) return false;
        if (hp == V || is_final[hp] || hi_ >= holes[hp].size()) {
          ++hp;
          hi_ = 0;
          h_used = 0;
          continue;
        }
        if (h_used >= holes[hp][hi_].second) {
          ++hi_;
          h_used = 0;
          continue;
        }
        return true;
      }
    };
    uint32_t moved = 0;
    for (uint32_t i = 0; i < k; ++i) {
      std::vector<CopassExtent> out;
      out.reserve(ext[i].size() + 4);
      for (const CopassExtent& x0 : ext[i]) {
        if (x0.phys / B != V) {
          out.push_back(x0);
          continue;
        }
        CopassExtent x = x0;
        while (x.lo < x.hi) {
          if (!next_hole()) return fail(c, NC_ERR_CUDA, "COPASS plan: no hole left for a live piece");
          auto& h = holes[hp][hi_];
          const uint32_t take = std::min(x.hi - x.lo, h.second - h_used);
          cs.push_back(x.phys);
          cd.push_back(h.first + h_used);
          cp.push_back(moved);
          out.push_back(CopassExtent{x.lo, x.lo + take, h.first + h_used});
          moved += take;
          h_used += take;
          x.lo += take;
          x.phys += take;
        }
      }
      ext[i].swap(out);
    }
    // holes that were used up to (hp, hi_, h_used) are gone; the rest stay
    for (uint32_t p = 0; p <= k; ++p) {
      if (p == V || is_final[p]) continue;
      auto& hs = holes[p];
      if (p < hp) {
        hs.clear();
      } else if (p == hp) {
        std::vector<std::pair<uint32_t, uint32_t>> rest;
        if (hi_ < hs.size()) {
          if (h_used < hs[hi_].second) rest.push_back({hs[hi_].first + h_used, hs[hi_].second - h_used});
          rest.insert(rest.end(), hs.begin() + hi_ + 1, hs.end());
        }
        hs.swap(rest);
      }
    }
    holes[V].clear();
    sp.e1 = cs.size();
    sp.e_total = moved;
    F = V;
  }
  // the spare block at the end: the one physical block that holds no output block
  uint32_t last_free = 0;
  for (uint32_t p = 0; p <= k; ++p)
    if (!is_final[p]) last_free = p;

  // ---- upload the commands and enqueue everything ----
  const size_t n_cmds = cs.size();
  uint32_t* d_cmd = (uint32_t*)dev_alloc(c, std::max<size_t>(1, n_cmds) * 12);
  if (!d_cmd) {
    drop();
    return fail(c, NC_ERR_OOM, "out of device memory for the COPASS copy commands");
  }
  dev_free_later(c, d_cmd);
  uint32_t *d_cs = d_cmd, *d_cd = d_cmd + n_cmds, *d_cp = d_cmd + 2 * n_cmds;
  NC_CUDA(c, cudaMemcpyAsync(d_cs, cs.data(), n_cmds * 4, cudaMemcpyHostToDevice, c->stream));
  NC_CUDA(c, cudaMemcpyAsync(d_cd, cd.data(), n_cmds * 4, cudaMemcpyHostToDevice, c->stream));
  NC_CUDA(c, cudaMemcpyAsync(d_cp, cp.data(), n_cmds * 4, cudaMemcpyHostToDevice, c->stream));
  BlockMap pm = make_map(c);
  pm.table = d_phys;
  const uint32_t per_cta = kGatherThreads * kGatherItems;
  for (uint32_t b = 0; b < k; ++b) {
    const Step& sp = steps[b];
    uint4* target = (uint4*)phys[sp.target];
    {
      Scope scp(c, NC_PHASE_COPASS);
      // Fig. 6D: left partitions -> the spare block (which is the auxiliary array)
      copass_segcopy_kernel<<<(sp.g_total + per_cta - 1) / per_cta, kGatherThreads, 0, c->stream>>>(
          pm, d_cs + sp.g0, d_cd + sp.g0, d_cp + sp.g0, (uint32_t)(sp.g1 - sp.g0), sp.g_total, sc.dig, plan.shift[0],
          (1u << plan.bits[0]) - 1u);
      NC_LAUNCH_CHECK(c, "copass_gather_left");
      if (sp.e_total) {  // instead of Fig. 6E: empty the victim into the holes
        copass_segcopy_kernel<<<(sp.e_total + per_cta - 1) / per_cta, kGatherThreads, 0, c->stream>>>(
            pm, d_cs + sp.e0, d_cd + sp.e0, d_cp + sp.e0, (uint32_t)(sp.e1 - sp.e0), sp.e_total, nullptr, 0u, 0u);
        NC_LAUNCH_CHECK(c, "copass_fill_holes");
      }
    }
    // Fig. 6F: sorted where it stands -- the passes go through the scratch and the last one writes the block's
    // final arrays (an output block is never touched again); with a single pass the records come back as records
    uint4* out = plan.n_passes > 1 ? target : sc.buf[0];
    int rc = copass_sort_records(c, plan, sc, false, pm, 0, target, sp.g_total, out, true,
                                 plan.n_passes > 1 ? (char*)target : nullptr);
    if (rc != NC_OK) return rc;
    if (out != target)
      NC_CUDA(c, cudaMemcpyAsync(target, out, (size_t)sp.g_total * 16, cudaMemcpyDeviceToDevice, c->stream));
  }
  *blocks_are_final = plan.n_passes > 1;
  for (const Step& sp : steps) c->copass_moved += (uint64_t)sp.g_total + sp.e_total;
  for (uint32_t b = 0; b < k; ++b) c->blocks[b] = phys[final_of[b]];
  spare = phys[last_free];
  NC_CUDA(c, cudaMemcpyAsync(c->d_table, c->blocks.data(), (size_t)k * 8, cudaMemcpyHostToDevice, c->stream));
  drop();
  return NC_OK;
}

int organise_copass(nc_context* c, const PassPlan& plan) {
  const uint32_t n = (uint32_t)c->n_conns;
  const uint64_t B = c->B;
  const uint32_t k = (uint32_t)c->blocks.size();
  if (k > kCopassMaxBlocks)
    return fail(c, NC_ERR_CAPACITY, "COPASS organisation handles at most 4096 storage blocks: raise block_size");
  if (k > 1 && !(c->cfg.flags & NC_FLAG_COPASS_SHIFT) && (uint64_t)(k + 1) * B > 0xffffffffull)
    return fail(c, NC_ERR_CAPACITY, "COPASS organisation: (blocks + 1) x block_size must stay below 2^32");
  const uint32_t big = (uint32_t)std::min<uint64_t>(B, n);  // the largest block (Eq. A3)
  const uint32_t kTile = (uint32_t)kSplitShapes[0].warps * 32u * (uint32_t)kSplitShapes[0].items;
  const uint32_t max_tiles = (big + kTile - 1) / kTile;
  const uint32_t max_chunks = (max_tiles + kCopassChunkTiles - 1) / kCopassChunkTiles;
  auto block_n = [&](uint32_t b) { return (uint32_t)std::min<uint64_t>(B, (uint64_t)n - (uint64_t)b * B); };

  const uint64_t bytes_before = c->bytes_in_use;
  void* spare = dev_alloc(c, c->block_bytes);                       // the free block of Fig. 6E
  // the auxiliary array (Eq. A3); with hole filling the spare block is the auxiliary array
  uint4* aux = (k > 1 && (c->cfg.flags & NC_FLAG_COPASS_SHIFT)) ? (uint4*)dev_alloc(c, (size_t)big * 16) : nullptr;
  CopassScratch sc{};
  const bool shift = (c->cfg.flags & NC_FLAG_COPASS_SHIFT) != 0;
  sc.buf[0] = (plan.n_passes > 1 || (!shift && k > 1)) ? (uint4*)dev_alloc(c, (size_t)big * 16) : nullptr;
  sc.buf[1] = plan.n_passes > 2 ? (uint4*)dev_alloc(c, (size_t)big * 16) : nullptr;
  sc.dig = (uint8_t*)dev_alloc(c, (size_t)big);
  sc.counts = (uint16_t*)dev_alloc(c, (size_t)max_tiles * kRadix * 2);
  sc.offs = (uint32_t*)dev_alloc(c, (size_t)max_tiles * kRadix * 4);
  sc.chunk = (uint32_t*)dev_alloc(c, (size_t)max_chunks * kRadix * 4);
  // partition state: two (start[k+1], len[k]) sets used in turn, m_i, left_prefix[k+1], right_src[k], what it did
  const size_t k1 = (size_t)k + 1;
  uint32_t* st = (uint32_t*)dev_alloc(c, (7 * k1) * 4 + sizeof(CopassInfo));
  if (!c->d_copass_totals) c->d_copass_totals = (CopassTotals*)dev_alloc(c, sizeof(CopassTotals));
  auto drop = [&]() {
    dev_free_later(c, spare); dev_free_later(c, aux); dev_free_later(c, sc.buf[0]); dev_free_later(c, sc.buf[1]);
    dev_free_later(c, sc.dig); dev_free_later(c, sc.counts); dev_free_later(c, sc.offs); dev_free_later(c, sc.chunk);
    dev_free_later(c, st);
  };
  bool ok = spare && sc.dig && sc.counts && sc.offs && sc.chunk && st && c->d_copass_totals && (k == 1 || !shift || aux);
  if (plan.n_passes > 1 || (!shift && k > 1)) ok = ok && sc.buf[0];
  if (plan.n_passes > 2) ok = ok && sc.buf[1];
  if (!ok) {
    drop();
    return fail(c, NC_ERR_OOM, "out of device memory in nc_finalize (COPASS organisation)");
  }
  c->copass_aux_bytes = c->bytes_in_use - bytes_before;
  NC_CUDA(c, cudaMemsetAsync(c->d_copass_totals, 0, sizeof(CopassTotals), c->stream));
  uint32_t* start[2] = {st, st + 2 * k1};
  uint32_t* len[2] = {st + k1, st + 3 * k1};
  uint32_t* m_out = st + 4 * k1;
  uint32_t* left_prefix = st + 5 * k1;
  uint32_t* right_src = st + 6 * k1;
  CopassInfo* info = (CopassInfo*)(st + 7 * k1);

  // block b takes the place of the spare block (whose memory the caller has just filled) and becomes the spare
  auto swap_with_spare = [&](uint32_t b) -> int {
    std::swap(c->blocks[b], spare);
    copass_poke_kernel<<<1, 1, 0, c->stream>>>(c->d_table, b, (uint64_t)c->blocks[b], 0xffffffffu, 0);
    NC_LAUNCH_CHECK(c, "copass_poke");
    return NC_OK;
  };
  const BlockMap map = make_map(c);
  int rc;

  // Fig. 6B: every block sorted on its own, creation-order layout -> records.  From here on the blocks are being
  // rewritten: a failure leaves no usable connections behind.
  c->broken = true;
  for (uint32_t b = 0; b < k; ++b) {
    BlockMap one = map;
    one.table = c->d_table + b;
    rc = copass_sort_records(c, plan, sc, true, one, (uint32_t)((uint64_t)b * B), nullptr, block_n(b), (uint4*)spare);
    if (rc != NC_OK) return rc;
    if ((rc = swap_with_spare(b)) != NC_OK) return rc;
  }
  bool blocks_are_final = false;
  if (k > 1 && !shift) {
    if ((rc = copass_extract_fill(c, plan, sc, spare, st, &blocks_are_final)) != NC_OK) return rc;
  } else if (k > 1) {
    {
      Scope scp(c, NC_PHASE_COPASS);
      copass_init_subarrays_kernel<<<(k + 255) / 256, 256, 0, c->stream>>>(start[0], len[0], k, (uint32_t)B, n);
      NC_LAUNCH_CHECK(c, "copass_init_subarrays");
    }
    const size_t part_smem = 7 * k1 * 4, gather_smem = (2 * k1) * 4;
    auto part = copass_partition_kernel<RecKeys>;
    NC_CUDA(c, cudaFuncSetAttribute(part, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)part_smem));
    NC_CUDA(c, cudaFuncSetAttribute(copass_gather_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gather_smem));
    const uint32_t per_cta = kGatherThreads * kGatherItems;
    int cur = 0;
    for (uint32_t b = 0; b + 1 < k; ++b) {
      const uint32_t N_b = (uint32_t)B;  // every block but the last is full
      const uint32_t new_base = (uint32_t)((uint64_t)(b + 1) * B);
      {
        Scope scp(c, NC_PHASE_COPASS);
        // Fig. 6C
        part<<<1, kCopassThreads, part_smem, c->stream>>>(RecKeys{map}, k, N_b, start[cur], len[cur], new_base, m_out,
                                                         left_prefix, right_src, start[1 - cur], len[1 - cur], info,
                                                         c->d_copass_totals, 0u, 0u);
        NC_LAUNCH_CHECK(c, "copass_partition");
        // Fig. 6D
        c->copass_moved += N_b;
        copass_gather_kernel<<<(N_b + per_cta - 1) / per_cta, kGatherThreads, gather_smem, c->stream>>>(
            map, k, left_prefix, start[cur], 0u, N_b, aux, sc.dig, plan.shift[0], (1u << plan.bits[0]) - 1u);
        NC_LAUNCH_CHECK(c, "copass_gather_left");
        // Fig. 6E, last destination block first: everything a block receives lies at or before it
        for (uint32_t j = k - 1; j > b; --j) {
          const uint32_t cnt = block_n(j);
          c->copass_moved += cnt;
          copass_gather_kernel<<<(cnt + per_cta - 1) / per_cta, kGatherThreads, gather_smem, c->stream>>>(
              map, k, start[1 - cur], right_src, (uint32_t)((uint64_t)j * B), cnt, (uint4*)spare, nullptr, 0u, 0u);
          NC_LAUNCH_CHECK(c, "copass_shift");
          if ((rc = swap_with_spare(j)) != NC_OK) return rc;
        }
      }
      // Fig. 6F: the auxiliary array, sorted, into block b (all of whose old content has moved)
      rc = copass_sort_records(c, plan, sc, false, map, 0, aux, N_b, (uint4*)c->blocks[b], true);
      if (rc != NC_OK) return rc;
      cur = 1 - cur;
    }
    // the last block: what is left is its content (reading C5); its k ascending pieces are merged by the sort
    rc = copass_sort_records(c, plan, sc, false, map, 0, (const uint4*)c->blocks[k - 1], block_n(k - 1), (uint4*)spare);
    if (rc != NC_OK) return rc;
    if ((rc = swap_with_spare(k - 1)) != NC_OK) return rc;
  }
  // records -> source / target / weight / delay / creation position arrays of the block
  if (!blocks_are_final) {
    Scope scp(c, NC_PHASE_PERMUTE);
    for (uint32_t b = 0; b < k; ++b) {
      char* o = (char*)spare;
      const uint32_t cnt = block_n(b);
      copass_unpack_kernel<<<std::min<uint32_t>((cnt + 255) / 256, 148 * 16), 256, 0, c->stream>>>(
          (const uint4*)c->blocks[b], cnt, c->delay_bits, (uint32_t*)o, (uint32_t*)(o + c->off_tgt),
          (float*)(o + c->off_w), (uint16_t*)(o + c->off_d), (uint32_t*)(o + c->off_perm));
      NC_LAUNCH_CHECK(c, "copass_unpack");
      if ((rc = swap_with_spare(b)) != NC_OK) return rc;
    }
  }
  c->copass_aux_bytes = c->bytes_in_use - bytes_before;  // nothing of the scratch has been released yet
  c->organised_in_blocks = true;
  c->broken = false;  // the blocks hold the organised connections
  rc = build_index_from_sorted(c, n, nullptr);
  drop();
  return rc;
}

// a12-a14 over the final source / delay arrays.
// NC_INDEX_FUSED=1 selects the single-read index (index_fused_kernel: count, look-back across tiles and write in one kernel).
// Measured on B200, configs[2]: 1.16 - 1.20 ms against 0.72 ms for count / scan / scatter (two streaming reads at 8 CTAs per
// SM): a tile cannot write before the tiles before it have counted, so each CTA sits through one load latency, two block
// scans and a look-back with nothing to overlap them (tiles of 4096 with 1184 in flight and tiles of 16384 with 148 in
// flight measure the same).  Kept selectable and parity-tested; not the default.
bool index_fused() {
  const char* e = getenv("NC_INDEX_FUSED");
  return e && atoi(e) != 0;
}

int build_index_from_sorted(nc_context* c, uint32_t n, uint32_t* lookback_flag) {
  const uint32_t N = c->n_nodes;
  const uint64_t head_tiles = ((uint64_t)n + kHeadTile - 1) / kHeadTile;
  const uint64_t head_chunks = (head_tiles + kScanChunk - 1) / kScanChunk;
  uint32_t* tile_heads = (uint32_t*)dev_alloc(c, head_tiles * 4);
  uint32_t* tile_head_off = (uint32_t*)dev_alloc(c, head_tiles * 4);
  uint32_t* head_partial = (uint32_t*)dev_alloc(c, head_chunks * 4);
  if (!c->d_total_groups) c->d_total_groups = (uint64_t*)dev_alloc(c, 16);  // total_groups | index error flag
  auto drop = [&]() {
    dev_free_later(c, tile_heads); dev_free_later(c, tile_head_off); dev_free_later(c, head_partial);
  };
  if (!tile_heads || !tile_head_off || !head_partial || !c->d_total_groups) {
    drop();
    return fail(c, NC_ERR_OOM, "out of device memory for the index scratch");
  }
  // A group is a distinct (source, delay) pair, so total_groups <= min(n, N_nodes * max delay).  When that bound
  // is small next to the connections themselves the group arrays are sized by it and nc_finalize never waits for
  // the device; otherwise the exact count is read back first.
  const uint64_t bound = std::min<uint64_t>(n, (uint64_t)N * c->max_delay_steps);
  const bool presize = !lookback_flag && bound * 6 <= std::max<uint64_t>((uint64_t)n * 2, 1u << 20);
  const SoAKeys keys{c->s_src, c->s_d, 16u};
  const BlockKeys block_keys{make_map(c), 16u};
  if (presize && !c->organised_in_blocks && index_fused()) {
    // one read of the keys: heads counted, chained across tiles by look-back and written by the same kernel
    const uint64_t tiles = ((uint64_t)n + kFusedTile - 1) / kFusedTile;
    uint64_t* status = (uint64_t*)dev_alloc(c, tiles * 8 + 16);  // [tiles] status words | ticket | error flag
    c->group_start = (uint32_t*)dev_alloc(c, (size_t)bound * 4);
    c->group_delay = (uint16_t*)dev_alloc(c, (size_t)bound * 2);
    drop();
    dev_free_later(c, status);
    if (!status || !c->group_start || !c->group_delay) return fail(c, NC_ERR_OOM, "out of device memory for the index");
    uint32_t* ticket = reinterpret_cast<uint32_t*>(status + tiles);
    c->d_index_error = reinterpret_cast<uint32_t*>(c->d_total_groups + 1);  // read back together with total_groups
    Scope sc(c, NC_PHASE_INDEX);
    NC_CUDA(c, cudaMemsetAsync(status, 0, tiles * 8 + 16, c->stream));
    NC_CUDA(c, cudaMemsetAsync(c->d_index_error, 0, 4, c->stream));
    IndexOut io{c->src_offsets, c->group_ptr, c->group_start, c->group_delay, N};
    index_fused_kernel<<<(unsigned)tiles, kFusedThreads, 0, c->stream>>>(c->s_src, c->s_d, n, status, ticket, c->d_total_groups,
                                                                     c->d_index_error, io);
    NC_LAUNCH_CHECK(c, "index_fused");
    index_finish_kernel<<<(N + 255) / 256, 256, 0, c->stream>>>(c->src_offsets, c->group_ptr, N, c->out_degree,
                                                               c->group_count, c->d_max + 1);
    NC_LAUNCH_CHECK(c, "index_finish");
    c->total_groups_pending = true;
    return NC_OK;
  }
  {
    Scope sc(c, NC_PHASE_INDEX);
    if (c->organised_in_blocks)
      head_count_kernel<<<(unsigned)head_tiles, kHeadThreads, 0, c->stream>>>(block_keys, n, tile_heads);
    else
      head_count_kernel<<<(unsigned)head_tiles, kHeadThreads, 0, c->stream>>>(keys, n, tile_heads);
    NC_LAUNCH_CHECK(c, "head_count");
    int rc = device_scan(c, tile_heads, tile_head_off, head_tiles, head_partial, c->d_total_groups);
    if (rc != NC_OK) return rc;
  }
  uint64_t cap = bound;
  if (!presize) {
    uint64_t total_groups = 0;
    uint32_t lookback_error = 0;
    NC_CUDA(c, cudaMemcpyAsync(&total_groups, c->d_total_groups, 8, cudaMemcpyDeviceToHost, c->stream));
    if (lookback_flag) NC_CUDA(c, cudaMemcpyAsync(&lookback_error, lookback_flag, 4, cudaMemcpyDeviceToHost, c->stream));
    NC_CUDA(c, cudaStreamSynchronize(c->stream));  // total_groups sizes the group arrays
    release_deferred(c);
    if (lookback_error) {
      drop();
      return fail(c, NC_ERR_CUDA, "onesweep look-back timed out");
    }
    c->total_groups = (uint32_t)total_groups;
    cap = total_groups;
  } else {
    c->total_groups_pending = true;
  }
  c->group_start = (uint32_t*)dev_alloc(c, (size_t)cap * 4);
  c->group_delay = (uint16_t*)dev_alloc(c, (size_t)cap * 2);
  if (!c->group_start || !c->group_delay) {
    drop();
    return fail(c, NC_ERR_OOM, "out of device memory for the group arrays");
  }
  {
    Scope sc(c, NC_PHASE_INDEX);
    IndexOut io{c->src_offsets, c->group_ptr, c->group_start, c->group_delay, N};
    if (c->organised_in_blocks)
      index_scatter_kernel<<<(unsigned)head_tiles, kHeadThreads, 0, c->stream>>>(block_keys, n, tile_head_off,
                                                                                  c->d_total_groups, io);
    else
      index_scatter_soa_kernel<<<(unsigned)head_tiles, kHeadThreads, 0, c->stream>>>(c->s_src, c->s_d, n, tile_head_off,
                                                                                      c->d_total_groups, io);
    NC_LAUNCH_CHECK(c, "index_scatter");
    index_finish_kernel<<<(N + 255) / 256, 256, 0, c->stream>>>(c->src_offsets, c->group_ptr, N, c->out_degree,
                                                               c->group_count, c->d_max + 1);
    NC_LAUNCH_CHECK(c, "index_finish");
  }
  drop();
  return NC_OK;
}

// total_groups when nc_finalize did not wait for it.
int ensure_total_groups(nc_context* c) {
  if (!c->total_groups_pending) return NC_OK;
  uint64_t total_groups = 0;
  uint32_t index_error = 0;
  NC_CUDA(c, cudaMemcpyAsync(&total_groups, c->d_total_groups, 8, cudaMemcpyDeviceToHost, c->stream));
  if (c->d_index_error) NC_CUDA(c, cudaMemcpyAsync(&index_error, c->d_index_error, 4, cudaMemcpyDeviceToHost, c->stream));
  int rc = sync_stream(c);
  if (rc != NC_OK) return rc;
  if (index_error) return fail(c, NC_ERR_CUDA, "index look-back timed out");
  c->total_groups = (uint32_t)total_groups;
  c->total_groups_pending = false;
  return NC_OK;
}

int collect_timings(nc_context* c) {
  gen_span_end(c);
  int rc = sync_stream(c);
  if (rc != NC_OK) return rc;
  for (Span& s : c->spans) {
    float ms = 0.f;
    cudaEventElapsedTime(&ms, s.a, s.b);
    if (s.is_pass) {
      c->acc.sort_pass_ms += ms;
      c->acc.sort_passes += 1;
    } else {
      c->acc.ms[s.phase] += ms;
    }
    cudaEventDestroy(s.a);
    cudaEventDestroy(s.b);
  }
  c->spans.clear();
  return NC_OK;
}

// ---- self-test kernels ----
__global__ void selftest_philox_kernel(uint32_t n, const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const Philox4 r = philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1]);
  out[4 * i] = r.x;
  out[4 * i + 1] = r.y;
  out[4 * i + 2] = r.z;
  out[4 * i + 3] = r.w;
}

__device__ void atomic_max_double(double* addr, double v) {  // v >= 0: bit patterns order like the values
  atomicMax(reinterpret_cast<unsigned long long*>(addr), (unsigned long long)__double_as_longlong(v));
}

__global__ void selftest_fastpath_kernel(double* out /* [4] */) {
  const uint32_t v = blockIdx.x * blockDim.x + threadIdx.x;  // 0 .. 2^24-1
  const uint32_t word = v << 8;
  const float r2c = fmaxf(fast_r2(word), 1e-30f);
  const float inv_r = rsqrt_approx(r2c);
  const float r32 = r2c * inv_r;
  const double u1 = (double)(v + 1u) * (1.0 / 16777216.0);
  const double r64 = sqrt(-2.0 * log(u1));
  const double dr = fabs((double)r32 - r64);
  // ratio of the actual error of r to the bound the guard band assumes, evaluated with the kernel's own r, 1/r
  const double bound = (double)kErrRa * (double)inv_r + (double)kErrRb * (double)r32;
  double e0 = dr / bound;  // u1 = 1: r32 = 1e-15 instead of 0, far inside the (then infinite) bound
  double e3 = dr;  // absolute error of r: the weight error is sd_w * (dr + r * dcos)
  float sn, cs;
  fast_sincos_shifted(word, sn, cs);  // sin, cos of (theta - pi) = -sin, -cos of theta
  sn = -sn;
  cs = -cs;
  const double th = 6.283185307179586 * ((double)v * (1.0 / 16777216.0));
  double e1 = fabs((double)sn - sin(th)) / (double)kErrTrig, e2 = fabs((double)cs - cos(th)) / (double)kErrTrig;
  for (int d = 16; d > 0; d >>= 1) {
    e0 = fmax(e0, __shfl_xor_sync(0xffffffffu, e0, d));
    e1 = fmax(e1, __shfl_xor_sync(0xffffffffu, e1, d));
    e2 = fmax(e2, __shfl_xor_sync(0xffffffffu, e2, d));
    e3 = fmax(e3, __shfl_xor_sync(0xffffffffu, e3, d));
  }
  if ((threadIdx.x & 31) == 0) {
    atomic_max_double(out + 0, e0);
    atomic_max_double(out + 1, e1);
    atomic_max_double(out + 2, e2);
    atomic_max_double(out + 3, e3);
  }
}

}  // namespace

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

// src_nodes / tgt_nodes: HOST arrays of src.count / tgt.count node ids, or NULL for the consecutive range
static int connect_core(nc_context* c, const uint32_t* src_nodes, nc_range src, const uint32_t* tgt_nodes, nc_range tgt,
                        nc_rule rule, const nc_rule_params* params, const nc_syn_spec* syn, uint64_t seed,
                        const float* weights = nullptr, const double* delays_ms = nullptr, uint64_t n_values = 0,
                        bool with_values = false) {
  if (!c) return NC_ERR_INVALID_ARG;
  if (c->broken) return fail(c, NC_ERR_STATE, "nc_connect: a failed in-place organisation left this context without connections; destroy it");
  if (c->finalized) return fail(c, NC_ERR_STATE, "nc_connect after nc_finalize");
  if (!params || !syn) return fail(c, NC_ERR_INVALID_ARG, "nc_connect: null params");
  if (src.count == 0 || tgt.count == 0) return fail(c, NC_ERR_INVALID_ARG, "nc_connect: empty node range");
  if (src_nodes) src.first = 0;
  if (tgt_nodes) tgt.first = 0;
  if ((!src_nodes && (uint64_t)src.first + src.count > c->n_nodes) ||
      (!tgt_nodes && (uint64_t)tgt.first + tgt.count > c->n_nodes))
    return fail(c, NC_ERR_INVALID_ARG, "nc_connect: node range outside the created nodes");
  for (uint32_t k = 0; src_nodes && k < src.count; ++k)
    if (src_nodes[k] >= c->n_nodes) return fail(c, NC_ERR_INVALID_ARG, "nc_connect_nodes: source id outside the created nodes");
  for (uint32_t k = 0; tgt_nodes && k < tgt.count; ++k)
    if (tgt_nodes[k] >= c->n_nodes) return fail(c, NC_ERR_INVALID_ARG, "nc_connect_nodes: target id outside the created nodes");
  if (!dist_ok(syn->weight) || !dist_ok(syn->delay_ms))
    return fail(c, NC_ERR_INVALID_ARG, "nc_connect: bad distribution (sd < 0, lo > hi or NaN)");
  const uint64_t K = params->degree_or_total;
  uint64_t n_new = 0;
  switch (rule) {
    case NC_ONE_TO_ONE:
      if (src.count != tgt.count) return fail(c, NC_ERR_INVALID_ARG, "one_to_one needs N_sources == N_targets");
      n_new = src.count;
      break;
    case NC_ALL_TO_ALL:
      n_new = (uint64_t)src.count * tgt.count;
      break;
    case NC_FIXED_OUTDEGREE:
      if (K > kMaxConns) return fail(c, NC_ERR_CAPACITY, "out-degree too large");
      n_new = (uint64_t)src.count * K;
      break;
    case NC_FIXED_INDEGREE:
      if (K > kMaxConns) return fail(c, NC_ERR_CAPACITY, "in-degree too large");
      n_new = (uint64_t)tgt.count * K;
      break;
    case NC_FIXED_TOTAL_NUMBER:
      n_new = K;
      break;
    case NC_PAIRWISE_BERNOULLI:
      if (!(params->p >= 0.0 && params->p <= 1.0)) return fail(c, NC_ERR_INVALID_ARG, "p outside [0, 1]");
      break;
    default:
      return fail(c, NC_ERR_INVALID_ARG, "unknown rule");
  }
  if (rule != NC_PAIRWISE_BERNOULLI && n_new > kMaxConns) return fail(c, NC_ERR_CAPACITY, "more than 2^32-1 connections");
  double bound = delay_bound_steps(syn->delay_ms, c->inv_dt);
  if (bound > 65535.0) return fail(c, NC_ERR_CAPACITY, "delay can exceed 65535 steps");
  if (with_values) {  // one value per connection
    if (!weights && !delays_ms) return fail(c, NC_ERR_INVALID_ARG, "nc_connect_values: no value array given");
    if (rule == NC_PAIRWISE_BERNOULLI)
      return fail(c, NC_ERR_INVALID_ARG, "nc_connect_values: pairwise_bernoulli has no connection count known beforehand");
    if (n_values != n_new)
      return fail(c, NC_ERR_INVALID_ARG, "nc_connect_values: the arrays must have one entry per connection of the rule");
    for (uint64_t i = 0; weights && i < n_values; ++i)
      if (std::isnan(weights[i])) return fail(c, NC_ERR_INVALID_ARG, "nc_connect_values: NaN weight");
    for (uint64_t i = 0; delays_ms && i < n_values; ++i) {
      if (!std::isfinite(delays_ms[i])) return fail(c, NC_ERR_INVALID_ARG, "nc_connect_values: delay not finite");
      const double steps = std::floor(delays_ms[i] * c->inv_dt + 0.5);
      if (steps > 65535.0) return fail(c, NC_ERR_CAPACITY, "nc_connect_values: a delay exceeds 65535 steps");
      if (steps > bound) bound = steps;  // the key's delay bits must hold it
    }
  }
  if (rule != NC_PAIRWISE_BERNOULLI && c->n_conns + n_new > kMaxConns)
    return fail(c, NC_ERR_CAPACITY, "more than 2^32-1 connections");

  // ---- autapses / multapses prohibited (readings A1-A6): checks that need no device work ----
  const uint32_t rflags = c->rule_flags;
  const bool no_aut = (rflags & NC_NO_AUTAPSES) != 0, no_mult = (rflags & NC_NO_MULTAPSES) != 0;
  std::vector<uint32_t> self_host;  // A2: per source its equal-id target index; A5: per fixed node its index among the partners
  bool need_self = false;
  if (rflags) {
    if (with_values && no_aut && (rule == NC_ONE_TO_ONE || rule == NC_ALL_TO_ALL))
      return fail(c, NC_ERR_INVALID_ARG, "nc_connect_values: without autapses the number of connections of this rule is not known beforehand");
    if (rule == NC_FIXED_TOTAL_NUMBER && no_mult)
      return fail(c, NC_ERR_INVALID_ARG, "fixed_total_number cannot prohibit multapses (reading A6)");
    for (int side = 0; side < 2; ++side) {  // A1: node arrays must not repeat an id
      const uint32_t* a = side ? tgt_nodes : src_nodes;
      if (!a) continue;
      std::vector<uint32_t> v(a, a + (side ? tgt.count : src.count));
      std::sort(v.begin(), v.end());
      if (std::adjacent_find(v.begin(), v.end()) != v.end())
        return fail(c, NC_ERR_INVALID_ARG, "nc_connect_nodes: a node array repeats an id while autapses or multapses are prohibited");
    }
    // index of a node id among the sources (side 0) or targets (side 1), or kNoIndex
    std::unordered_map<uint32_t, uint32_t> where[2];
    for (int side = 0; side < 2; ++side) {
      const uint32_t* a = side ? tgt_nodes : src_nodes;
      const uint32_t cnt = side ? tgt.count : src.count;
      for (uint32_t k = 0; a && k < cnt; ++k) where[side][a[k]] = k;
    }
    auto find_in = [&](int side, uint32_t id) -> uint32_t {
      const uint32_t* a = side ? tgt_nodes : src_nodes;
      const nc_range r = side ? tgt : src;
      if (!a) return (id >= r.first && (uint64_t)id < (uint64_t)r.first + r.count) ? id - r.first : kNoIndex;
      auto it = where[side].find(id);
      return it == where[side].end() ? kNoIndex : it->second;
    };
    auto id_of = [&](int side, uint32_t k) -> uint32_t {
      const uint32_t* a = side ? tgt_nodes : src_nodes;
      return a ? a[k] : (side ? tgt.first : src.first) + k;
    };
    const bool arrays = src_nodes || tgt_nodes;
    if (rule == NC_FIXED_INDEGREE || rule == NC_FIXED_OUTDEGREE) {
      const int fixed_side = rule == NC_FIXED_INDEGREE ? 1 : 0, part_side = 1 - fixed_side;
      const uint32_t n_fixed = fixed_side ? tgt.count : src.count, n_part = part_side ? tgt.count : src.count;
      bool any_self = false;
      if (no_aut) {
        if (arrays) {
          self_host.resize(n_fixed);
          for (uint32_t f = 0; f < n_fixed; ++f) {
            self_host[f] = find_in(part_side, id_of(fixed_side, f));
            any_self = any_self || self_host[f] != kNoIndex;
          }
          need_self = no_mult;  // only the permutation (A5) needs the index on the device; the redraws compare ids
        } else {
          const uint64_t a0 = fixed_side ? tgt.first : src.first, b0 = part_side ? tgt.first : src.first;
          any_self = a0 < b0 + n_part && b0 < a0 + n_fixed;  // the ranges overlap
        }
      }
      const uint64_t M_min = (uint64_t)n_part - (any_self ? 1 : 0);
      if (no_mult ? K > M_min : (K > 0 && M_min == 0))
        return fail(c, NC_ERR_INVALID_ARG, "more distinct partners asked for than the rule allows (readings A3, A5)");
    } else if (rule == NC_FIXED_TOTAL_NUMBER) {
      if (no_aut && K > 0 && src.count == 1 && tgt.count == 1 && id_of(0, 0) == id_of(1, 0))
        return fail(c, NC_ERR_INVALID_ARG, "fixed_total_number: the only pair is an autapse");
    } else if (no_aut && arrays) {  // A2 with node arrays: which target index carries each source's id
      self_host.resize(src.count);
      for (uint32_t k = 0; k < src.count; ++k) self_host[k] = find_in(1, id_of(0, k));
      need_self = true;
    }
  }

  GenParams gp{};
  gp.pos0 = c->n_conns;
  gp.n = n_new;
  gp.s0 = src.first;
  gp.n_src = src.count;
  gp.t0 = tgt.first;
  gp.n_tgt = tgt.count;
  gp.K = (uint32_t)K;
  gp.div = rule == NC_ALL_TO_ALL ? tgt.count : (rule == NC_FIXED_INDEGREE || rule == NC_FIXED_OUTDEGREE) ? (uint32_t)K : 1u;
  gp.div_magic = make_div_magic(gp.div);
  const uint32_t seed_lo = (uint32_t)(seed & 0xffffffffull), seed_hi = (uint32_t)(seed >> 32);
  gp.rng = make_philox_stream(seed_lo, seed_hi, c->n_proj, 0u);  // D2: synapse stream
  gp.syn = make_syn(c, *syn);
  // explicit node arrays: copied into library-owned device memory, released once the stream has been synchronised
  for (int side = 0; side < 2; ++side) {
    const uint32_t* host = side == 0 ? src_nodes : tgt_nodes;
    if (!host) continue;
    const size_t bytes = (size_t)(side == 0 ? src.count : tgt.count) * sizeof(uint32_t);
    uint32_t* dev = (uint32_t*)dev_alloc(c, bytes);
    if (!dev) return fail(c, NC_ERR_OOM, "out of device memory for a node array");
    dev_free_later(c, dev);
    NC_CUDA(c, cudaMemcpyAsync(dev, host, bytes, cudaMemcpyHostToDevice, c->stream));
    (side == 0 ? gp.src_nodes : gp.tgt_nodes) = dev;
  }

  uint32_t* d_self = nullptr;
  if (need_self) {
    d_self = (uint32_t*)dev_alloc(c, self_host.size() * 4);
    if (!d_self) return fail(c, NC_ERR_OOM, "out of device memory for the self-index array");
    dev_free_later(c, d_self);
    NC_CUDA(c, cudaMemcpyAsync(d_self, self_host.data(), self_host.size() * 4, cudaMemcpyHostToDevice, c->stream));
  }
  const bool pair_rule = rule == NC_PAIRWISE_BERNOULLI || rule == NC_ONE_TO_ONE || rule == NC_ALL_TO_ALL;
  if (rule == NC_PAIRWISE_BERNOULLI || (no_aut && pair_rule)) {
    // reading A2: under NC_NO_AUTAPSES one_to_one and all_to_all also go through the pair mask (count, reserve, ordered write)
    int rc = connect_bernoulli(c, gp, params->p, seed_lo, seed_hi, rule == NC_PAIRWISE_BERNOULLI, rule == NC_ONE_TO_ONE, no_aut,
                               d_self);
    if (rc != NC_OK) return rc;
    if (need_self) {
      rc = sync_stream(c);  // self_host is read by the upload
      if (rc != NC_OK) return rc;
    }
  } else if (rflags && !pair_rule && n_new > 0) {
    // readings A3-A5: the random-partner rules under the flags
    int rc = reserve_blocks(c, n_new);
    if (rc != NC_OK) return rc;
    gp.map = make_map(c);
    gen_span_end(c);
    {
      Scope sc(c, NC_PHASE_GENERATE);
      FlagGenParams fp{};
      fp.g = gp;
      fp.rule = rule == NC_FIXED_INDEGREE ? (uint32_t)kFixedIndegree
                                          : rule == NC_FIXED_OUTDEGREE ? (uint32_t)kFixedOutdegree : (uint32_t)kFixedTotalNumber;
      fp.flags = rflags;
      fp.seed_lo = seed_lo;
      fp.seed_hi = seed_hi;
      fp.proj = c->n_proj;
      fp.self_idx = d_self;
      const unsigned grid = (unsigned)std::min<uint64_t>((n_new + 255) / 256, 148 * 32);
      generate_flagged_kernel<<<grid, 256, 0, c->stream>>>(fp);
      NC_LAUNCH_CHECK(c, "generate_flagged");
    }
    if (with_values) {
      float* d_w = weights ? (float*)dev_alloc(c, (size_t)n_new * 4) : nullptr;
      double* d_d = delays_ms ? (double*)dev_alloc(c, (size_t)n_new * 8) : nullptr;
      dev_free_later(c, d_w);
      dev_free_later(c, d_d);
      if ((weights && !d_w) || (delays_ms && !d_d)) return fail(c, NC_ERR_OOM, "out of device memory for the value arrays");
      if (d_w) NC_CUDA(c, cudaMemcpyAsync(d_w, weights, (size_t)n_new * 4, cudaMemcpyHostToDevice, c->stream));
      if (d_d) NC_CUDA(c, cudaMemcpyAsync(d_d, delays_ms, (size_t)n_new * 8, cudaMemcpyHostToDevice, c->stream));
      const unsigned vgrid = (unsigned)std::min<uint64_t>((n_new + 255) / 256, 148 * 16);
      set_values_kernel<<<vgrid, 256, 0, c->stream>>>(gp.map, gp.pos0, n_new, d_w, d_d, c->inv_dt);
      NC_LAUNCH_CHECK(c, "set_values");
    }
    c->n_conns += n_new;
    if (need_self) {
      rc = sync_stream(c);
      if (rc != NC_OK) return rc;
    }
  } else if (n_new > 0) {
    int rc = reserve_blocks(c, n_new);
    if (rc != NC_OK) return rc;
    gp.map = make_map(c);
    {
      gen_span_begin(c);
      cudaError_t e;
      switch (rule) {
        case NC_ONE_TO_ONE: e = launch_generate<kOneToOne>(c, gp); break;
        case NC_ALL_TO_ALL: e = launch_generate<kAllToAll>(c, gp); break;
        case NC_FIXED_INDEGREE: e = launch_generate<kFixedIndegree>(c, gp); break;
        case NC_FIXED_OUTDEGREE: e = launch_generate<kFixedOutdegree>(c, gp); break;
        default: e = launch_generate<kFixedTotalNumber>(c, gp); break;
      }
      if (e != cudaSuccess) return fail(c, NC_ERR_CUDA, std::string("launch generate: ") + cudaGetErrorString(e));
      NC_LAUNCH_CHECK(c, "generate");
    }
    if (with_values) {
      float* d_w = weights ? (float*)dev_alloc(c, (size_t)n_new * 4) : nullptr;
      double* d_d = delays_ms ? (double*)dev_alloc(c, (size_t)n_new * 8) : nullptr;
      dev_free_later(c, d_w);
      dev_free_later(c, d_d);
      if ((weights && !d_w) || (delays_ms && !d_d)) return fail(c, NC_ERR_OOM, "out of device memory for the value arrays");
      if (d_w) NC_CUDA(c, cudaMemcpyAsync(d_w, weights, (size_t)n_new * 4, cudaMemcpyHostToDevice, c->stream));
      if (d_d) NC_CUDA(c, cudaMemcpyAsync(d_d, delays_ms, (size_t)n_new * 8, cudaMemcpyHostToDevice, c->stream));
      const unsigned grid = (unsigned)std::min<uint64_t>((n_new + 255) / 256, 148 * 16);
      set_values_kernel<<<grid, 256, 0, c->stream>>>(gp.map, gp.pos0, n_new, d_w, d_d, c->inv_dt);
      NC_LAUNCH_CHECK(c, "set_values");
    }
    c->n_conns += n_new;
  }
  if (src_nodes || tgt_nodes || with_values) {
    // nc.h: the host arrays are copied DURING the call.  From page-locked memory cudaMemcpyAsync returns before the copy
    // has run, so wait here; this also releases the device copies (and any older scratch) right away.
    const int rc = sync_stream(c);
    if (rc != NC_OK) return rc;
  }
  c->n_proj += 1;
  c->proj_first.push_back((uint32_t)gp.pos0);
  c->proj_attr.push_back((uint16_t)(c->cur_port | (c->cur_group << 8)));
  if (bound > (double)c->max_delay_steps) c->max_delay_steps = (uint32_t)bound;
  c->have_in = c->have_out = false;
  return NC_OK;
}

// Reading S1 (nc_set_shard): connect calls run in full into staging blocks; flush_shard then keeps what this shard owns
// (nc_shard.cuh).  Calls are batched -- the filter runs when kShardFlush connections are staged, at nc_finalize and before
// anything reads the storage -- so a network of many small projections costs one wait per batch, not one per call.
constexpr uint64_t kShardFlush = 1ull << 28;  // 3.8 GB of staged connections

static int flush_shard(nc_context* c) {
  if (!c->sharded || c->stage_n == 0) {
    c->stage_pending.clear();
    return NC_OK;
  }
  const uint64_t n_full = c->stage_n;
  const uint64_t tiles = (n_full + kOwnTile - 1) / kOwnTile;
  const uint64_t chunks = (tiles + kScanChunk - 1) / kScanChunk;
  const size_t n_q = c->stage_pending.size();
  uint32_t* tile_count = (uint32_t*)dev_alloc(c, tiles * 4);
  uint32_t* tile_off = (uint32_t*)dev_alloc(c, tiles * 4);
  uint32_t* partial = (uint32_t*)dev_alloc(c, chunks * 4);
  uint64_t* d_total = (uint64_t*)dev_alloc(c, 8);
  uint64_t* d_query = (uint64_t*)dev_alloc(c, (n_q + 1) * 16);  // [n_q] staged start positions | [n_q] owned connections before each
  auto drop = [&]() {
    dev_free_later(c, tile_count); dev_free_later(c, tile_off); dev_free_later(c, partial); dev_free_later(c, d_total);
    dev_free_later(c, d_query);
  };
  if (!tile_count || !tile_off || !partial || !d_total || !d_query) {
    drop();
    return fail(c, NC_ERR_OOM, "out of device memory for the shard filter");
  }
  ShardFilterParams fp{};
  fp.stage = make_map(c);
  fp.stage.table = c->stage_table;
  fp.n = n_full;
  fp.first = c->shard_first;
  fp.count = c->shard_count;
  fp.tile_count = tile_count;
  fp.tile_offset = tile_off;
  uint64_t total = 0;
  std::vector<uint64_t> starts(n_q), before(n_q);
  for (size_t k = 0; k < n_q; ++k) starts[k] = c->stage_pending[k].second;
  gen_span_end(c);
  {
    Scope sc(c, NC_PHASE_GENERATE);
    owned_count_kernel<<<(unsigned)tiles, kOwnThreads, 0, c->stream>>>(fp);
    NC_LAUNCH_CHECK(c, "owned_count");
    int rc = device_scan(c, tile_count, tile_off, tiles, partial, d_total);
    if (rc != NC_OK) {
      drop();
      return rc;
    }
    if (n_q) {
      NC_CUDA(c, cudaMemcpyAsync(d_query, starts.data(), n_q * 8, cudaMemcpyHostToDevice, c->stream));
      owned_before_kernel<<<(unsigned)((n_q + 7) / 8), 256, 0, c->stream>>>(fp, d_query, (uint32_t)n_q, d_query + n_q);
      NC_LAUNCH_CHECK(c, "owned_before");
      NC_CUDA(c, cudaMemcpyAsync(before.data(), d_query + n_q, n_q * 8, cudaMemcpyDeviceToHost, c->stream));
    }
    NC_CUDA(c, cudaMemcpyAsync(&total, d_total, 8, cudaMemcpyDeviceToHost, c->stream));
  }
  NC_CUDA(c, cudaStreamSynchronize(c->stream));  // the exact count decides the allocation
  if (c->n_conns + total > kMaxConns) {
    drop();
    return fail(c, NC_ERR_CAPACITY, "more than 2^32-1 connections in this shard");
  }
  int rc = reserve_blocks(c, total);
  if (rc != NC_OK) {
    drop();
    return rc;
  }
  if (total > 0) {
    Scope sc(c, NC_PHASE_GENERATE);
    fp.store = make_map(c);
    fp.pos0 = c->n_conns;
    owned_copy_kernel<<<(unsigned)tiles, kOwnThreads, 0, c->stream>>>(fp);
    NC_LAUNCH_CHECK(c, "owned_copy");
  }
  for (size_t k = 0; k < n_q; ++k)  // a projection starts where the first connection kept from it (or after it) went
    c->proj_first[c->stage_pending[k].first] = (uint32_t)(c->n_conns + before[k]);
  c->n_conns += total;
  c->stage_n = 0;
  c->stage_pending.clear();
  drop();
  return NC_OK;
}

static int connect_impl(nc_context* c, const uint32_t* src_nodes, nc_range src, const uint32_t* tgt_nodes, nc_range tgt,
                        nc_rule rule, const nc_rule_params* params, const nc_syn_spec* syn, uint64_t seed,
                        const float* weights = nullptr, const double* delays_ms = nullptr, uint64_t n_values = 0,
                        bool with_values = false) {
  if (!c || !c->sharded || c->broken || c->finalized)  // not sharded, or let the ordinary path report the state
    return connect_core(c, src_nodes, src, tgt_nodes, tgt, rule, params, syn, seed, weights, delays_ms, n_values, with_values);
  // swap in the staging storage: the generators append the full projection behind what is already staged
  std::vector<void*> real_blocks;
  real_blocks.swap(c->blocks);
  c->blocks.swap(c->stage_blocks);
  uint64_t* real_table = c->d_table;
  const size_t real_cap = c->table_cap;
  const uint64_t real_n = c->n_conns;
  c->d_table = c->stage_table;
  c->table_cap = c->stage_cap;
  c->n_conns = c->stage_n;
  const uint32_t proj_before = c->n_proj;
  const uint64_t stage_start = c->stage_n;
  const int rc = connect_core(c, src_nodes, src, tgt_nodes, tgt, rule, params, syn, seed, weights, delays_ms, n_values, with_values);
  c->stage_blocks.swap(c->blocks);
  c->stage_table = c->d_table;
  c->stage_cap = c->table_cap;
  c->stage_n = c->n_conns;
  c->blocks.swap(real_blocks);
  c->d_table = real_table;
  c->table_cap = real_cap;
  c->n_conns = real_n;
  if (rc != NC_OK) return rc;
  if (c->n_proj > proj_before) c->stage_pending.push_back({proj_before, stage_start});
  return c->stage_n >= kShardFlush ? flush_shard(c) : NC_OK;
}

int nc_set_shard(nc_context* c, uint32_t first, uint32_t count) {
  if (!c) return NC_ERR_INVALID_ARG;
  if (c->finalized || c->n_conns || c->n_proj) return fail(c, NC_ERR_STATE, "nc_set_shard: only before the first nc_connect*");
  if (c->cfg.flags & NC_FLAG_ORGANISE_COPASS) {}  // any organisation works: the filter runs before it
  c->sharded = true;
  c->shard_first = first;
  c->shard_count = count;
  return NC_OK;
}

int nc_set_rule_flags(nc_context* c, uint32_t flags) {
  if (!c) return NC_ERR_INVALID_ARG;
  if (flags & ~(uint32_t)(NC_NO_AUTAPSES | NC_NO_MULTAPSES)) return fail(c, NC_ERR_INVALID_ARG, "nc_set_rule_flags: unknown flag");
  if (c->finalized) return fail(c, NC_ERR_STATE, "nc_set_rule_flags after nc_finalize");
  c->rule_flags = flags;
  return NC_OK;
}

int nc_connect(nc_context* c, nc_range src, nc_range tgt, nc_rule rule, const nc_rule_params* params,
               const nc_syn_spec* syn, uint64_t seed) {
  return connect_impl(c, nullptr, src, nullptr, tgt, rule, params, syn, seed);
}

int nc_connect_nodes(nc_context* c, const uint32_t* src_nodes, uint32_t n_src, nc_range src, const uint32_t* tgt_nodes,
                     uint32_t n_tgt, nc_range tgt, nc_rule rule, const nc_rule_params* params, const nc_syn_spec* syn,
                     uint64_t seed) {
  if (src_nodes) src = nc_range{0u, n_src};
  if (tgt_nodes) tgt = nc_range{0u, n_tgt};
  return connect_impl(c, src_nodes, src, tgt_nodes, tgt, rule, params, syn, seed);
}

int nc_connect_values(nc_context* c, const uint32_t* src_nodes, uint32_t n_src, nc_range src, const uint32_t* tgt_nodes,
                      uint32_t n_tgt, nc_range tgt, nc_rule rule, const nc_rule_params* params, const nc_syn_spec* syn,
                      uint64_t seed, const float* weights, const double* delays_ms, uint64_t n_values) {
  if (src_nodes) src = nc_range{0u, n_src};
  if (tgt_nodes) tgt = nc_range{0u, n_tgt};
  return connect_impl(c, src_nodes, src, tgt_nodes, tgt, rule, params, syn, seed, weights, delays_ms, n_values, true);
}

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
extern "C" uint64_t nc_internal_guard_violations(nc_context* c) { return c ? c->guard_violations : 0; }
