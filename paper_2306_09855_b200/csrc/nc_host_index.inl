// nc_host_index.inl -- index construction over the organised keys, timings, device self-test kernels.
// Part of the single translation unit nc_api.cu (included there, in order; not compiled on its own).

namespace {

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

