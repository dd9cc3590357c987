// nc_host_connect.inl -- the connect path: pairwise_bernoulli / pair-mask rules, rule validation and generator dispatch
// (connect_core), autapse / multapse flags, sharded contexts (staging + owner filter), and the nc_connect* entry points.
// Part of the single translation unit nc_api.cu (included there, inside extern "C"; not compiled on its own).

}  // extern "C" (reopened below)
namespace {

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
      if (T < (1ull << 32)) bernoulli_trials_kernel<true><<<(unsigned)n_tiles, kBernThreads, 0, c->stream>>>(bp);
      else bernoulli_trials_kernel<false><<<(unsigned)n_tiles, kBernThreads, 0, c->stream>>>(bp);
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

}  // namespace
extern "C" {

// src_nodes / tgt_nodes: HOST arrays of src.count / tgt.count node ids, or NULL for the consecutive range
static int connect_core(nc_context* c, const uint32_t* src_nodes, nc_range src, const uint32_t* tgt_nodes, nc_range tgt,
                        nc_rule rule, const nc_rule_params* params, const nc_syn_spec* syn, uint64_t seed,
                        const float* weights = nullptr, const double* delays_ms = nullptr, uint64_t n_values = 0,
                        bool with_values = false, bool sub = false, uint64_t sub_first = 0, uint64_t sub_count = 0,
                        uint32_t sub_w = 0, uint32_t sub_off = 0) {
  // sub: create only connections sub_first .. sub_first + sub_count - 1 of the call (a shard's owned index sub-range; the
  // caller guarantees a rule whose indexes it may cut, no value arrays, no rule flags).  sub_w > 0 (all_to_all only): the
  // sub_count = N_src * sub_w connections whose target is one of columns sub_off .. sub_off + sub_w - 1 instead, row by row
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
  if (sub) n_new = sub_count;  // every check above was made on the whole call
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
  gp.i_first = sub ? (uint32_t)sub_first : 0u;
  gp.s0 = src.first;
  gp.n_src = src.count;
  gp.t0 = tgt.first;
  gp.n_tgt = tgt.count;
  gp.K = (uint32_t)K;
  gp.div = rule == NC_ALL_TO_ALL ? (sub_w ? sub_w : tgt.count) : (rule == NC_FIXED_INDEGREE || rule == NC_FIXED_OUTDEGREE) ? (uint32_t)K : 1u;
  gp.sub_w = rule == NC_ALL_TO_ALL ? sub_w : 0u;
  gp.sub_off = sub_off;
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
        case NC_ALL_TO_ALL: e = gp.sub_w ? launch_generate<kAllToAllSub>(c, gp) : launch_generate<kAllToAll>(c, gp); break;
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
  // (all_to_all, whose owned part is a strip of columns, follows below.)
  // Rules whose target is the slow deterministic coordinate of the index (one_to_one: t = t0 + i; fixed_indegree:
  // t = t0 + i div K) over a target RANGE: the connections this shard owns are one contiguous index sub-range of the call,
  // generated directly into the storage -- no staging, no filter, no redundant draws ("each GPU generates the
  // index sub-range whose deterministic coordinate it owns").
  if ((rule == NC_ONE_TO_ONE || rule == NC_FIXED_INDEGREE) && !tgt_nodes && !with_values && c->rule_flags == 0 && params &&
      tgt.count > 0 && (uint64_t)tgt.first + tgt.count <= c->n_nodes) {
    const uint64_t own_lo = std::max<uint64_t>(c->shard_first, tgt.first);
    const uint64_t own_hi = std::min<uint64_t>((uint64_t)c->shard_first + c->shard_count, (uint64_t)tgt.first + tgt.count);
    const uint64_t per = rule == NC_ONE_TO_ONE ? 1 : params->degree_or_total;
    const uint64_t first = own_hi > own_lo ? (own_lo - tgt.first) * per : 0, count = own_hi > own_lo ? (own_hi - own_lo) * per : 0;
    const int rc = flush_shard(c);  // what is staged comes before this call in creation order
    if (rc != NC_OK) return rc;
    return connect_core(c, src_nodes, src, tgt_nodes, tgt, rule, params, syn, seed, nullptr, nullptr, 0, false, true, first, count);
  }
  // all_to_all over a target RANGE: the owned connections are the strip of owned target columns of every row, generated
  // directly with the full call's indexes for the random numbers (kAllToAllSub) -- no staging, no filter, no redundant draws
  if (rule == NC_ALL_TO_ALL && !tgt_nodes && !with_values && c->rule_flags == 0 && params && src.count > 0 && tgt.count > 0 &&
      (uint64_t)tgt.first + tgt.count <= c->n_nodes) {
    const uint64_t own_lo = std::max<uint64_t>(c->shard_first, tgt.first);
    const uint64_t own_hi = std::min<uint64_t>((uint64_t)c->shard_first + c->shard_count, (uint64_t)tgt.first + tgt.count);
    const uint32_t w = own_hi > own_lo ? (uint32_t)(own_hi - own_lo) : 0u;
    const int rc = flush_shard(c);  // what is staged comes before this call in creation order
    if (rc != NC_OK) return rc;
    return connect_core(c, src_nodes, src, tgt_nodes, tgt, rule, params, syn, seed, nullptr, nullptr, 0, false, true, 0,
                        (uint64_t)src.count * w, w, w ? (uint32_t)(own_lo - tgt.first) : 0u);
  }
  // swap in the staging storage: the generators append the full projection behind what is already staged
  auto staged_attempt = [&]() -> int {
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
    if (rc == NC_OK && c->n_proj > proj_before) c->stage_pending.push_back({proj_before, stage_start});
    return rc;
  };
  int rc = staged_attempt();
  if (rc == NC_ERR_CAPACITY && c->stage_n > 0) {
    // the full call did not fit BEHIND what earlier calls left staged (connect_core bounds staged + new by 2^32 - 1): filter
    // those first -- a failed call changes nothing -- and give this one the whole staging range
    const int frc = flush_shard(c);
    if (frc != NC_OK) return frc;
    rc = staged_attempt();
  }
  if (rc != NC_OK) return rc;
  return c->stage_n >= kShardFlush ? flush_shard(c) : NC_OK;
}

int nc_set_shard(nc_context* c, uint32_t first, uint32_t count) {
  if (!c) return NC_ERR_INVALID_ARG;
  if (c->finalized || c->n_conns || c->n_proj) return fail(c, NC_ERR_STATE, "nc_set_shard: only before the first nc_connect*");
  // one definition of the owned range for the device filter (32-bit t - first < count) and the direct sub-range path
  // (64-bit clamp): ids first .. first + count - 1 without wrapping
  if ((uint64_t)first + count > (1ull << 32)) return fail(c, NC_ERR_INVALID_ARG, "nc_set_shard: first + count exceeds 2^32");
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

