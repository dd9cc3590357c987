// nc_host_copass.inl -- host plan of the COPASS organisation inside the storage blocks.
// Part of the single translation unit nc_api.cu (included there, in order; not compiled on its own).

namespace {

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

}  // namespace

