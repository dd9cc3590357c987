// nc_host_organise.inl -- nc_finalize's organisation paths over flat arrays: the (key, position) pairs sort, the
// single-pass look-back variant and the default count / scan / scatter passes (also in their bulk-fed form).
// Part of the single translation unit nc_api.cu (included there, in order; not compiled on its own).

namespace {

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
// Launch shapes of the scatter pass, NC_SPLIT_VARIANT=k in the environment (measured on B200): 0 the default,
// 2 CTAs x 8 warps x 16 records; 1 three CTAs x 12 warps x 8 records (tiles of 3072); 2 one CTA x 16 warps x 16 records (tiles of
// 8192: 512-byte runs, but one CTA's phases do not overlap).
struct SplitShape {
  int warps, items;
};
constexpr SplitShape kSplitShapes[] = {{8, 16}, {12, 8}, {16, 16}};

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
    case 2: return launch_scatter_shape<FIRST, LAST, 16, 16, 1>(c, sp, n_tiles);
    default: return launch_scatter_shape<FIRST, LAST, 8, 16, 2>(c, sp, n_tiles);
  }
}

// NC_FLAG_SORT_BULK: the same pass as a persistent kernel fed by cp.async.bulk (nc_sort_bulk.cuh), one CTA per SM.
// Ranks among equal digits come from ballots (defined behaviour) unless NC_ATOMIC_RANK=1 asks for the faster form that takes
// them from the return values of one shared atomicAdd per record.  That form rests on same-address lanes of one instruction
// being served in ascending lane order, which no document promises: it is therefore never a default, and even when asked for
// it is only used after atomic_lane_order_kernel has seen the order hold on this device (once per context; a sampling check,
// not a proof -- a stable sort is only guaranteed with ballots).
int atomic_rank_usable(nc_context* c) {
  if (c->atomic_rank >= 0) return NC_OK;
  const char* e = getenv("NC_ATOMIC_RANK");
  if (!(e && atoi(e) != 0)) {
    c->atomic_rank = 0;
    return NC_OK;
  }
  uint32_t* d = (uint32_t*)dev_alloc(c, 4);
  if (!d) return fail(c, NC_ERR_OOM, "out of device memory");
  uint32_t bad = 1;
  NC_CUDA(c, cudaMemsetAsync(d, 0, 4, c->stream));
  atomic_lane_order_kernel<<<296, 256, 0, c->stream>>>(d, 256);
  NC_LAUNCH_CHECK(c, "atomic_lane_order");
  NC_CUDA(c, cudaMemcpyAsync(&bad, d, 4, cudaMemcpyDeviceToHost, c->stream));
  NC_CUDA(c, cudaStreamSynchronize(c->stream));
  dev_free(c, d);
  c->atomic_rank = bad == 0 ? 1 : 0;
  return NC_OK;
}

template <bool FIRST, bool LAST>
int launch_scatter_bulk(nc_context* c, const ScatterParams& sp, uint32_t n_tiles) {
  int rc = atomic_rank_usable(c);
  if (rc != NC_OK) return rc;
  int sms = 0;
  NC_CUDA(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device));
  const uint32_t grid = std::min<uint32_t>(n_tiles, (uint32_t)sms);
  if (c->atomic_rank) {
    auto kern = scatter_bulk_kernel<FIRST, LAST, true>;
    NC_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(BulkSmem)));
    kern<<<grid, kBulkWarps * 32, sizeof(BulkSmem), c->stream>>>(sp, n_tiles);
  } else {
    auto kern = scatter_bulk_kernel<FIRST, LAST, false>;
    NC_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(BulkSmem)));
    kern<<<grid, kBulkWarps * 32, sizeof(BulkSmem), c->stream>>>(sp, n_tiles);
  }
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


}  // namespace

