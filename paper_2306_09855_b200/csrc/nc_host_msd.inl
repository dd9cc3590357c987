// nc_host_msd.inl -- nc_finalize's bucket-first organisation path (NC_FLAG_SORT_BUCKETS, kernels in nc_sort_msd.cuh).
// Part of the single translation unit nc_api.cu (included there, in order; not compiled on its own).

namespace {

constexpr int kMsdMaxLanes = 4;
constexpr uint64_t kMsdSlotCapRecords = 4ull << 20;  // 64 MB of records; a larger bucket goes to lane 0's own slot

// The CUDA streams the buckets are spread over: created once per device and process, shared by every context (work of two
// contexts on them is ordered by the events each finalize records, like any two users of a stream).
cudaStream_t msd_lane_stream(int device, int lane) {
  static std::mutex mu;
  static std::map<std::pair<int, int>, cudaStream_t> pool;
  std::lock_guard<std::mutex> lock(mu);
  auto it = pool.find({device, lane});
  if (it != pool.end()) return it->second;
  cudaStream_t s = nullptr;
  if (cudaStreamCreateWithFlags(&s, cudaStreamNonBlocking) != cudaSuccess) {
    cudaGetLastError();
    return nullptr;
  }
  pool[{device, lane}] = s;
  return s;
}

template <typename F>
struct AtExit {  // runs f when the scope is left, whichever return leaves it
  F f;
  ~AtExit() { f(); }
};
template <typename F>
AtExit(F) -> AtExit<F>;

struct MsdLane {
  cudaStream_t st = nullptr;
  uint4* tmp[2] = {nullptr, nullptr};    // intermediate records of the bucket being sorted (the second one: three or more passes)
  uint8_t* dig[2] = {nullptr, nullptr};  // next pass's digit of each
  uint16_t* counts = nullptr;
  uint32_t* chunk_base = nullptr;
  uint64_t cap = 0;  // records
};

template <bool LAST, int MODE>
int launch_scatter_bucket(nc_context* c, const ScatterParams& sp, uint32_t n_tiles, cudaStream_t st) {
  using Smem = ScatterSmem<8, 16, false>;
  auto kern = scatter_pass_kernel<false, LAST, 8, 16, 2, kMatchBallot, MODE>;
  kern<<<n_tiles, 8 * 32, sizeof(Smem), st>>>(sp);
  NC_LAUNCH_CHECK(c, "scatter_pass (bucket)");
  return NC_OK;
}

bool msd_force_lanes() {  // experiments: per-bucket launches even where the persistent kernel applies
  const char* e = getenv("NC_BUCKET_LANES");
  return e && atoi(e) >= 1;
}

int msd_lanes_wanted(uint64_t slot_records) {
  const char* e = getenv("NC_BUCKET_LANES");
  if (e && atoi(e) >= 1 && atoi(e) <= kMsdMaxLanes) return atoi(e);
  return slot_records * 16 <= (24ull << 20) ? 3 : 2;  // what fits the L2 together (membench `ring`)
}

int sort_msd_and_index(nc_context* c) {
  using Smem = ScatterSmem<8, 16, false>;
  constexpr uint32_t kTile = 8 * 32 * 16;
  const uint32_t n = (uint32_t)c->n_conns;
  const uint32_t N = c->n_nodes;
  const uint32_t db = c->delay_bits;
  const uint32_t n_tiles = (uint32_t)(((uint64_t)n + kTile - 1) / kTile);
  const uint32_t n_chunks = (n_tiles + kScanChunkTiles - 1) / kScanChunkTiles;
  const BlockMap map = make_map(c);

  // ---- the bucket map and, from it, the key bits left to sort inside a bucket ----
  const uint64_t mul64 = (1ull << 40) / std::max<uint32_t>(N, 1u);
  const uint32_t mul = (uint32_t)std::min<uint64_t>(mul64, 0xffffffffull);
  uint32_t s_min[kRadix + 1];  // smallest source of every bucket: bucket(s) >= b  <=>  s * mul >= b * 2^32
  for (uint32_t b = 0; b < (uint32_t)kRadix; ++b)
    s_min[b] = (uint32_t)std::min<uint64_t>(N, (((uint64_t)b << 32) + mul - 1) / mul);
  s_min[kRadix] = N;
  uint32_t w_max = 1;
  std::vector<uint32_t> key_base(kRadix);
  for (uint32_t b = 0; b < (uint32_t)kRadix; ++b) {
    w_max = std::max(w_max, s_min[b + 1] - s_min[b]);
    key_base[b] = (uint32_t)((uint64_t)s_min[b] << db);  // wraps only for buckets past the last node, which stay empty
  }
  const uint32_t rel_bits = std::max(1u, bit_width_u64(((uint64_t)w_max << db) - 1));
  const PassPlan plan = plan_passes(rel_bits);
  const uint32_t PB = plan.n_passes;
  c->sort_passes = 1 + PB;

  uint4* recs = (uint4*)dev_alloc(c, (size_t)n * 16);
  uint8_t* dig = (uint8_t*)dev_alloc(c, (size_t)n + 16);
  uint16_t* counts = (uint16_t*)dev_alloc(c, (size_t)n_tiles * kRadix * 2);
  uint32_t* offs = (uint32_t*)dev_alloc(c, (size_t)n_tiles * kRadix * 4);
  uint32_t* chunk = (uint32_t*)dev_alloc(c, (size_t)n_chunks * kRadix * 4);
  uint32_t* d_key_base = (uint32_t*)dev_alloc(c, kRadix * 4);
  uint32_t* done = (uint32_t*)dev_alloc(c, kMsdMaxLanes * 4);
  c->s_src = (uint32_t*)dev_alloc(c, (size_t)n * 4);
  c->s_tgt = (uint32_t*)dev_alloc(c, (size_t)n * 4);
  c->s_w = (float*)dev_alloc(c, (size_t)n * 4);
  c->s_d = (uint16_t*)dev_alloc(c, (size_t)n * 2);
  c->perm = (uint32_t*)dev_alloc(c, (size_t)n * 4);
  MsdLane lanes[kMsdMaxLanes];
  bool scratch_dropped = false;
  auto drop_scratch = [&]() {
    if (scratch_dropped) return;
    scratch_dropped = true;
    dev_free_later(c, recs); dev_free_later(c, dig); dev_free_later(c, counts); dev_free_later(c, offs);
    dev_free_later(c, chunk); dev_free_later(c, d_key_base); dev_free_later(c, done);
    for (MsdLane& l : lanes) {
      dev_free_later(c, l.tmp[0]); dev_free_later(c, l.tmp[1]); dev_free_later(c, l.dig[0]); dev_free_later(c, l.dig[1]);
      dev_free_later(c, l.counts); dev_free_later(c, l.chunk_base);
    }
  };
  // Every way out of this function -- the error returns in the middle of the bucket loop as well -- first makes c->stream wait
  // for what was queued on the lane streams, then hands the scratch back.  The lane streams are process-wide: without the
  // join, what nc_finalize does on c->stream after a failure (releasing s_src / s_tgt / perm) could overtake lane kernels
  // that still write to them.
  AtExit lane_guard{[&]() {
    for (MsdLane& l : lanes) {
      if (!l.st) continue;
      cudaEvent_t ev = nullptr;
      bool joined = false;
      if (cudaEventCreateWithFlags(&ev, cudaEventDisableTiming) == cudaSuccess) {
        joined = cudaEventRecord(ev, l.st) == cudaSuccess && cudaStreamWaitEvent(c->stream, ev, 0) == cudaSuccess;
        cudaEventDestroy(ev);
      }
      if (!joined) {
        cudaStreamSynchronize(l.st);
        cudaGetLastError();
      }
    }
    drop_scratch();
  }};
  if (!recs || !dig || !counts || !offs || !chunk || !d_key_base || !done || !c->s_src || !c->s_tgt || !c->s_w || !c->s_d ||
      !c->perm) {
    return fail(c, NC_ERR_OOM, "out of device memory in nc_finalize");
  }
  cudaStream_t side = msd_lane_stream(c->device, 0);
  if (!side) {
    drop_scratch();
    return fail(c, NC_ERR_CUDA, "could not create the streams of the bucket-first organisation");
  }
  cudaEvent_t ev_scan = nullptr, ev_a = nullptr;
  NC_CUDA(c, cudaEventCreateWithFlags(&ev_scan, cudaEventDisableTiming));
  NC_CUDA(c, cudaEventCreateWithFlags(&ev_a, cudaEventDisableTiming));
  struct EventGuard {
    cudaEvent_t &a, &b;
    ~EventGuard() {
      if (a) cudaEventDestroy(a);
      if (b) cudaEventDestroy(b);
    }
  } guard{ev_scan, ev_a};

  // ---- pass A: counts and scan; the bucket sizes travel to the host while the scatter runs ----
  uint32_t h_start[kRadix + 1];
  {
    Scope sc(c, NC_PHASE_HISTOGRAM);
    NC_CUDA(c, cudaMemsetAsync(done, 0, kMsdMaxLanes * 4, c->stream));
    NC_CUDA(c, cudaMemcpyAsync(d_key_base, key_base.data(), kRadix * 4, cudaMemcpyHostToDevice, c->stream));
    if (c->B % 4 == 0)
      msd_tile_count_first_kernel<true><<<n_tiles, kCountThreads, 0, c->stream>>>(map, n, kTile, mul, counts);
    else
      msd_tile_count_first_kernel<false><<<n_tiles, kCountThreads, 0, c->stream>>>(map, n, kTile, mul, counts);
    NC_LAUNCH_CHECK(c, "tile_count (buckets)");
    chunk_total_kernel<<<n_chunks, kRadix, 0, c->stream>>>(counts, n_tiles, chunk);
    NC_LAUNCH_CHECK(c, "chunk_total");
    chunk_scan_kernel<<<1, kRadix * kChunkScanSegs, 0, c->stream>>>(chunk, n_chunks);
    NC_LAUNCH_CHECK(c, "chunk_scan");
    NC_CUDA(c, cudaEventRecord(ev_scan, c->stream));
    tile_offsets_kernel<<<n_chunks, kRadix, 0, c->stream>>>(counts, n_tiles, chunk, offs);
    NC_LAUNCH_CHECK(c, "tile_offsets");
  }
  {
    Scope sc(c, NC_PHASE_SORT);
    Scope pass_sc(c, NC_PHASE_SORT, true);
    ScatterParams sp{};
    sp.map = map;
    sp.delay_bits = db;
    sp.n = n;
    sp.recs_out = recs;
    sp.dig_out = dig;
    sp.next_shift = plan.shift[0];
    sp.next_bits = plan.bits[0];
    sp.offs = offs;
    sp.msd_mul = mul;
    sp.key_base_tab = d_key_base;
    auto kern = scatter_pass_kernel<true, false, 8, 16, 2, kMatchBallot, 1>;
    NC_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem)));
    kern<<<n_tiles, 8 * 32, sizeof(Smem), c->stream>>>(sp);
    NC_LAUNCH_CHECK(c, "scatter_pass (into buckets)");
    NC_CUDA(c, cudaEventRecord(ev_a, c->stream));
  }
  // first output position of every bucket = the scanned totals of chunk 0
  NC_CUDA(c, cudaStreamWaitEvent(side, ev_scan, 0));
  NC_CUDA(c, cudaMemcpyAsync(h_start, chunk, kRadix * 4, cudaMemcpyDeviceToHost, side));
  NC_CUDA(c, cudaStreamSynchronize(side));
  h_start[kRadix] = n;

  uint64_t max_all = 0, max_fit = 0;
  uint32_t n_buckets = 0;
  for (uint32_t b = 0; b < (uint32_t)kRadix; ++b) {
    const uint64_t sz = h_start[b + 1] - h_start[b];
    if (!sz) continue;
    ++n_buckets;
    max_all = std::max(max_all, sz);
    if (sz <= kMsdSlotCapRecords) max_fit = std::max(max_fit, sz);
  }

  // ---- pass B, two in-bucket passes and buckets that fit the slots: one persistent kernel ----
  if (PB == 2 && max_all <= kMsdSlotCapRecords && !msd_force_lanes()) {
    const uint64_t tiles_cap = (max_all + kBsTile - 1) / kBsTile, chunks_cap = (tiles_cap + kSegChunkTiles - 1) / kSegChunkTiles;
    const uint32_t nb = n_buckets;
    // descriptor block: bstart[nb] | bsize[nb] | bkey[nb] | round_first[nb + 4]
    std::vector<uint32_t> desc((size_t)4 * nb + 4);
    uint32_t* bstart = desc.data();
    uint32_t* bsize = bstart + nb;
    uint32_t* bkey = bsize + nb;
    uint32_t* round_first = bkey + nb;
    {
      uint32_t i = 0;
      for (uint32_t b = 0; b < (uint32_t)kRadix; ++b) {
        const uint32_t sz = h_start[b + 1] - h_start[b];
        if (!sz) continue;
        bstart[i] = h_start[b];
        bsize[i] = sz;
        bkey[i] = key_base[b];
        ++i;
      }
    }
    uint32_t n_items = 0;
    for (uint32_t r = 0; r < nb + 3; ++r) {
      round_first[r] = n_items;
      for (uint32_t seg = 0; seg < 4; ++seg) {
        if (r < seg || r - seg >= nb) continue;
        const uint32_t tiles = (bsize[r - seg] + kBsTile - 1) / kBsTile;
        n_items += (seg & 1) ? tiles : (tiles + kSegChunkTiles - 1) / kSegChunkTiles;
      }
    }
    round_first[nb + 3] = n_items;

    uint32_t* d_desc = (uint32_t*)dev_alloc(c, desc.size() * 4);
    uint32_t* d_sync = (uint32_t*)dev_alloc(c, ((size_t)nb * kBsSyncWords + 4) * 4);  // per-bucket counters | ticket
    uint4* slot_recs = (uint4*)dev_alloc(c, (size_t)kBsSlots * max_all * 16);
    uint8_t* slot_dig = (uint8_t*)dev_alloc(c, (size_t)kBsSlots * (max_all + 16));
    uint16_t* slot_counts = (uint16_t*)dev_alloc(c, (size_t)2 * kBsSlots * chunks_cap * kSegChunkTiles * kRadix * 2);
    uint32_t* slot_chunk = (uint32_t*)dev_alloc(c, (size_t)2 * kBsSlots * chunks_cap * kRadix * 4);
    auto drop_b = [&]() {
      dev_free_later(c, d_desc); dev_free_later(c, d_sync); dev_free_later(c, slot_recs); dev_free_later(c, slot_dig);
      dev_free_later(c, slot_counts); dev_free_later(c, slot_chunk);
    };
    if (!d_desc || !d_sync || !slot_recs || !slot_dig || !slot_counts || !slot_chunk) {
      drop_b();
      drop_scratch();
      return fail(c, NC_ERR_OOM, "out of device memory in nc_finalize");
    }
    using BsSmem = ScatterSmem<kBsWarps, kBsItems, false>;
    BucketSortParams bp{};
    bp.recs = recs;
    bp.dig = dig;
    for (int k = 0; k < kBsSlots; ++k) {
      bp.slot[k] = slot_recs + (size_t)k * max_all;
      bp.slot_dig[k] = slot_dig + (size_t)k * (max_all + 16);
      for (int ps = 0; ps < 2; ++ps) {
        bp.counts[ps][k] = slot_counts + ((size_t)ps * kBsSlots + k) * chunks_cap * kSegChunkTiles * kRadix;
        bp.chunk_base[ps][k] = slot_chunk + ((size_t)ps * kBsSlots + k) * chunks_cap * kRadix;
      }
    }
    bp.out_src = c->s_src;
    bp.out_tgt = c->s_tgt;
    bp.out_w = c->s_w;
    bp.out_d = c->s_d;
    bp.out_perm = c->perm;
    bp.bstart = d_desc;
    bp.bsize = d_desc + nb;
    bp.bkey = d_desc + 2 * (size_t)nb;
    bp.round_first = d_desc + 3 * (size_t)nb;
    bp.sync = d_sync;
    bp.ticket = d_sync + (size_t)nb * kBsSyncWords;
    bp.nb = nb;
    bp.n_items = n_items;
    bp.delay_bits = db;
    for (int ps = 0; ps < 2; ++ps) {
      bp.shift[ps] = plan.shift[ps];
      bp.bits[ps] = plan.bits[ps];
    }
    {
      Scope sc(c, NC_PHASE_SORT);
      Scope pass_sc(c, NC_PHASE_SORT, true);
      NC_CUDA(c, cudaMemcpyAsync(d_desc, desc.data(), desc.size() * 4, cudaMemcpyHostToDevice, c->stream));
      NC_CUDA(c, cudaMemsetAsync(d_sync, 0, ((size_t)nb * kBsSyncWords + 4) * 4, c->stream));
      int arc = atomic_rank_usable(c);  // once per context: may ranks come from returning shared atomics on this device?
      if (arc != NC_OK) return arc;
      auto kern = c->atomic_rank ? bucket_sort_kernel<true> : bucket_sort_kernel<false>;
      NC_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(BsSmem)));
      int per_sm = 0, sms = 0;
      NC_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kBsThreads, sizeof(BsSmem)));
      NC_CUDA(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device));
      uint32_t grid = std::min<uint32_t>(n_items, (uint32_t)std::max(1, per_sm) * (uint32_t)sms);
      if (const char* e = getenv("NC_BUCKET_GRID")) grid = std::max(1, std::min<int>(atoi(e), (int)grid));  // experiments
      // NC_BUCKET_DEBUG=1: thread 0 of every CTA reports where its cycles went (profiles/r02_buckets.md); waits for the kernel
      unsigned long long* d_prof = getenv("NC_BUCKET_DEBUG") ? (unsigned long long*)dev_alloc(c, (size_t)grid * 64) : nullptr;
      bp.prof = d_prof;
      kern<<<grid, kBsThreads, sizeof(BsSmem), c->stream>>>(bp);
      NC_LAUNCH_CHECK(c, "bucket_sort");
      if (d_prof) {
        std::vector<unsigned long long> h((size_t)grid * 8);
        cudaStreamSynchronize(c->stream);
        cudaMemcpy(h.data(), d_prof, h.size() * 8, cudaMemcpyDeviceToHost);
        dev_free(c, d_prof);
        double sum[8] = {0};
        for (uint32_t g = 0; g < grid; ++g)
          for (int k = 0; k < 8; ++k) sum[k] += (double)h[(size_t)g * 8 + k];
        fprintf(stderr, "bucket_sort: grid %u items %u | per CTA mean kcycles: blocked %.0f (%.0f times) scatter1 %.0f scatter2 %.0f count %.0f (%.0f items) "
                "| scatter items %.0f | total %.0f\n", grid, n_items, sum[0] / grid / 1e3, sum[5] / grid, sum[1] / grid / 1e3, sum[2] / grid / 1e3,
                sum[3] / grid / 1e3, sum[6] / grid, sum[4] / grid, sum[7] / grid / 1e3);
      }
    }
    int rc = build_index_from_sorted(c, n, nullptr);
    drop_b();
    drop_scratch();
    return rc;
  }

  // ---- otherwise: the buckets spread over lanes (CUDA streams), one slot per lane sized by the largest bucket it will see ----
  const int n_lanes = max_fit == 0 ? 1 : std::max(1, std::min<int>(msd_lanes_wanted(max_fit), (int)n_buckets));
  for (int q = 0; q < n_lanes; ++q) {
    MsdLane& l = lanes[q];
    l.st = msd_lane_stream(c->device, q);
    l.cap = q == 0 ? max_all : max_fit;
    if (!l.st) {
      drop_scratch();
      return fail(c, NC_ERR_CUDA, "could not create the streams of the bucket-first organisation");
    }
    const uint64_t tiles = (l.cap + kTile - 1) / kTile, chunks = (tiles + kSegChunkTiles - 1) / kSegChunkTiles;
    bool ok = true;
    for (uint32_t k = 0; k < std::min(PB - 1, 2u); ++k) {
      l.tmp[k] = (uint4*)dev_alloc(c, (size_t)l.cap * 16);
      l.dig[k] = (uint8_t*)dev_alloc(c, (size_t)l.cap + 16);
      ok = ok && l.tmp[k] && l.dig[k];
    }
    l.counts = (uint16_t*)dev_alloc(c, (size_t)chunks * kSegChunkTiles * kRadix * 2);
    l.chunk_base = (uint32_t*)dev_alloc(c, (size_t)chunks * kRadix * 4);
    if (!ok || !l.counts || !l.chunk_base) {
      drop_scratch();
      return fail(c, NC_ERR_OOM, "out of device memory in nc_finalize");
    }
  }
  {
    auto k2 = scatter_pass_kernel<false, false, 8, 16, 2, kMatchBallot, 2>;
    auto k2l = scatter_pass_kernel<false, true, 8, 16, 2, kMatchBallot, 2>;
    auto k3 = scatter_pass_kernel<false, false, 8, 16, 2, kMatchBallot, 3>;
    auto k3l = scatter_pass_kernel<false, true, 8, 16, 2, kMatchBallot, 3>;
    NC_CUDA(c, cudaFuncSetAttribute(k2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem)));
    NC_CUDA(c, cudaFuncSetAttribute(k2l, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem)));
    NC_CUDA(c, cudaFuncSetAttribute(k3, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem)));
    NC_CUDA(c, cudaFuncSetAttribute(k3l, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(Smem)));
  }

  // ---- pass B: every bucket sorted on its own, inside the L2 ----
  {
    Scope sc(c, NC_PHASE_SORT);
    Scope pass_sc(c, NC_PHASE_SORT, true);
    for (int q = 0; q < n_lanes; ++q) NC_CUDA(c, cudaStreamWaitEvent(lanes[q].st, ev_a, 0));
    int next_lane = 0;
    for (uint32_t b = 0; b < (uint32_t)kRadix; ++b) {
      const uint32_t start = h_start[b], sz = h_start[b + 1] - h_start[b];
      if (!sz) continue;
      int q = 0;  // an oversized bucket: only lane 0's slot holds it
      if (sz <= max_fit) {
        q = next_lane;
        next_lane = (next_lane + 1) % n_lanes;
      }
      MsdLane& l = lanes[q];
      const uint32_t tiles = (sz + kTile - 1) / kTile, chunks = (tiles + kSegChunkTiles - 1) / kSegChunkTiles;
      for (uint32_t ps = 0; ps < PB; ++ps) {
        const bool last = ps + 1 == PB;
        const uint8_t* dig_in = ps == 0 ? dig + start : l.dig[(ps - 1) & 1];
        seg_count_scan_kernel<<<chunks, kSegThreads, 0, l.st>>>(dig_in, sz, kTile, l.counts, l.chunk_base, done + q);
        NC_LAUNCH_CHECK(c, "seg_count_scan");
        ScatterParams sp{};
        sp.delay_bits = db;
        sp.n = sz;
        sp.recs_in = ps == 0 ? recs + start : l.tmp[(ps - 1) & 1];
        sp.recs_out = last ? nullptr : l.tmp[ps & 1];
        sp.dig_out = last ? nullptr : l.dig[ps & 1];
        sp.out_src = c->s_src + start;
        sp.out_tgt = c->s_tgt + start;
        sp.out_w = c->s_w + start;
        sp.out_d = c->s_d + start;
        sp.out_perm = c->perm + start;
        sp.shift = plan.shift[ps];
        sp.bits = plan.bits[ps];
        sp.next_shift = last ? 0 : plan.shift[ps + 1];
        sp.next_bits = last ? 0 : plan.bits[ps + 1];
        sp.key_base = key_base[b];
        sp.counts = l.counts;
        sp.chunk_base = l.chunk_base;
        int rc;
        if (ps == 0) rc = last ? launch_scatter_bucket<true, 2>(c, sp, tiles, l.st) : launch_scatter_bucket<false, 2>(c, sp, tiles, l.st);
        else rc = last ? launch_scatter_bucket<true, 3>(c, sp, tiles, l.st) : launch_scatter_bucket<false, 3>(c, sp, tiles, l.st);
        if (rc != NC_OK) return rc;
      }
    }
    for (int q = 0; q < n_lanes; ++q) {
      cudaEvent_t ev = nullptr;
      NC_CUDA(c, cudaEventCreateWithFlags(&ev, cudaEventDisableTiming));
      cudaError_t e1 = cudaEventRecord(ev, lanes[q].st);
      cudaError_t e2 = cudaStreamWaitEvent(c->stream, ev, 0);
      cudaEventDestroy(ev);
      if (e1 != cudaSuccess || e2 != cudaSuccess) return fail(c, NC_ERR_CUDA, "joining the bucket streams failed");
    }
  }
  int rc = build_index_from_sorted(c, n, nullptr);
  drop_scratch();
  return rc;
}

}  // namespace
