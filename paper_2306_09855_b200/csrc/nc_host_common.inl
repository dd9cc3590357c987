// nc_host_common.inl -- host helpers of libnc: error plumbing, device allocations with guard zones, timing spans, the
// block map, Eq. 1 block reservation, generator launches, the device-wide scan.
// Part of the single translation unit nc_api.cu (included there, in order; not compiled on its own).

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


}  // namespace

