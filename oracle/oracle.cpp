/*
 * oracle.cpp -- plain single-threaded CPU ORACLE (TEST INFRASTRUCTURE ONLY; see oracle.h).
 *
 * Follows /root/reference/PAPER.md (arXiv 2306.09855) step by step, in the paper's order and
 * notation, plus the readings D1-D12 recorded in DESIGN.md for everything the paper leaves open
 * (RNG mapping, clamp/round order, tie order).  fp64 throughout; one thread; no blocking, fusion
 * or reordering; libm log/sqrt/sin/cos.  Build: g++ -std=c++17 -O2 -ffp-contract=off (so that
 * mean + sd*z is a rounded multiply followed by a rounded add, exactly as written).
 *
 * Shares nothing with the CUDA path: no header, constant table, helper or generator.
 */
#include "oracle.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>
#include <new>
#include <numeric>
#include <vector>

namespace {

/* ------------------------------------------------------------------ D2: Philox4x32-10 ----
 * Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3" (SC'11).
 * One round:  (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)),
 * key bump between rounds: k0 += 0x9E3779B9, k1 += 0xBB67AE85; ten rounds. */
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint64_t M0 = 0xD2511F53ull, M1 = 0xCD9E8D57ull;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) {
      k0 += 0x9E3779B9u;
      k1 += 0xBB67AE85u;
    }
    const uint64_t p0 = M0 * (uint64_t)c0;
    const uint64_t p1 = M1 * (uint64_t)c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    const uint32_t n1 = (uint32_t)p1;
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    const uint32_t n3 = (uint32_t)p0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* D2: key = (seed lo, seed hi); ctr = (idx lo, idx hi, projection_id, stream).
 * stream 0 = synapse stream (idx = i_newconns, or the pair index q for pairwise_bernoulli),
 * stream 1 = bernoulli trial stream (idx = q >> 2, word q & 3). */
void philox_stream(uint64_t seed, uint32_t projection_id, uint32_t stream, uint64_t idx,
                   uint32_t out[4]) {
  const uint32_t key[2] = {(uint32_t)(seed & 0xffffffffull), (uint32_t)(seed >> 32)};
  const uint32_t ctr[4] = {(uint32_t)(idx & 0xffffffffull), (uint32_t)(idx >> 32), projection_id,
                           stream};
  philox4x32_10(ctr, key, out);
}

/* D3: rand(N) of PAPER.md:95 ("random integer between 0 and N-1") = floor(word * N / 2^32). */
uint32_t bounded(uint32_t word, uint32_t n) { return (uint32_t)(((uint64_t)word * (uint64_t)n) >> 32); }

/* D4/Q14: accept pair q iff trial_word(q) < T, T = floor(p * 2^32) as a 64-bit integer. */
uint64_t bernoulli_threshold(double p) { return (uint64_t)std::floor(std::ldexp(p, 32)); }

double clampd(double v, double lo, double hi) { return v < lo ? lo : (v > hi ? hi : v); }

bool dist_ok(const oc_dist& d) {
  if (std::isnan(d.mean) || std::isnan(d.sd) || std::isnan(d.lo) || std::isnan(d.hi)) return false;
  if (std::isinf(d.mean) || std::isinf(d.sd)) return false;
  if (d.sd < 0.0) return false;
  if (d.lo > d.hi) return false;
  return true;
}

/* Q6: largest delay (in steps) a projection can produce.  |z| <= sqrt(48 ln 2) = 5.7681 by D5/D6
 * (u1 >= 2^-24); the planner uses the slightly larger 5.769. */
double max_delay_steps(const oc_dist& d, double inv_dt) {
  double top = d.mean + 5.769 * d.sd;
  if (top > d.hi) top = d.hi;
  if (top < d.lo) top = d.lo;
  return std::floor(top * inv_dt + 0.5);
}

/* Reading A5: a permutation of [0, M) keyed by four words -- cycle walking over a balanced Feistel network of
 * 6 + ceil(24 / h) rounds on 2h bits (narrow halves need more rounds: a two-round differential trail has probability 2^-h). */
uint32_t mix32(uint32_t v) {
  v ^= v >> 16;
  v *= 0x7feb352du;
  v ^= v >> 15;
  v *= 0x846ca68bu;
  v ^= v >> 16;
  return v;
}
uint32_t keyed_permutation(uint32_t M, uint32_t k, const uint32_t keys[4]) {
  if (M <= 1) return 0;
  uint32_t bits = 0;
  for (uint32_t v = M - 1; v; v >>= 1) ++bits;
  const uint32_t h = std::max<uint32_t>(1, (bits + 1) / 2);
  const uint32_t mask = (1u << h) - 1u; /* h <= 16 */
  uint32_t x = k;
  do {
    uint32_t L = x >> h, R = x & mask;
    const uint32_t rounds = 6 + (24 + h - 1) / h;
    for (uint32_t r = 0; r < rounds; ++r) {
      const uint32_t key_r = keys[r & 3] + r * 0x9E3779B9u;
      const uint32_t nR = L ^ (mix32(R ^ key_r) & mask);
      L = R;
      R = nR;
    }
    x = (L << h) | R;
  } while (x >= M);
  return x;
}

struct Projection {
  oc_range src, tgt;
  int rule;
  oc_rule_params params;
  oc_syn_spec syn;
  uint64_t seed;
  uint32_t id;
};

/* D4-D8 for one synapse.  `idx` is i_newconns (Eqs. 2-3), or q for bernoulli. */
void eval_synapse(const Projection& pr, double inv_dt, uint64_t idx, oc_synapse* out) {
  uint32_t w[4];
  philox_stream(pr.seed, pr.id, 0u, idx, w);

  const uint64_t n_src = pr.src.count, n_tgt = pr.tgt.count, K = pr.params.degree_or_total;
  uint64_t s = 0, t = 0;
  switch (pr.rule) {
    case OC_ONE_TO_ONE: /* Eqs. 4-5 */
      s = idx; t = idx; break;
    case OC_ALL_TO_ALL: /* Eqs. 6-7 */
    case OC_PAIRWISE_BERNOULLI: /* same source-major pair enumeration, reading D4/Q13 */
      s = idx / n_tgt; t = idx % n_tgt; break;
    case OC_FIXED_OUTDEGREE: /* Eqs. 8-9 */
      s = idx / K; t = bounded(w[1], (uint32_t)n_tgt); break;
    case OC_FIXED_INDEGREE: /* Eqs. 10-11 */
      s = bounded(w[0], (uint32_t)n_src); t = idx / K; break;
    case OC_FIXED_TOTAL_NUMBER: /* Eqs. 12-13 */
      s = bounded(w[0], (uint32_t)n_src); t = bounded(w[1], (uint32_t)n_tgt); break;
  }
  out->source = (uint32_t)(pr.src.first + s);
  out->target = (uint32_t)(pr.tgt.first + t);

  /* D5: 24-bit uniforms, u1 in (0,1], u2 in [0,1). */
  const double u1 = ((double)(w[2] >> 8) + 1.0) * (1.0 / 16777216.0);
  const double u2 = (double)(w[3] >> 8) * (1.0 / 16777216.0);
  /* D6: Box-Muller. */
  const double r = std::sqrt(-2.0 * std::log(u1));
  const double theta = 6.283185307179586 * u2;
  const double z0 = r * std::cos(theta);
  const double z1 = r * std::sin(theta);
  out->z0 = z0;
  out->z1 = z1;
  /* D7: weight ("randomly distributed according to a given probability distribution"). */
  const oc_dist& dw = pr.syn.weight;
  out->weight = (float)clampd(dw.mean + dw.sd * z0, dw.lo, dw.hi);
  /* D8: delay in ms -> integer steps: divide by the time step, round, at least 1. */
  const oc_dist& dd = pr.syn.delay_ms;
  const double d_ms = clampd(dd.mean + dd.sd * z1, dd.lo, dd.hi);
  const double x = d_ms * inv_dt;
  double steps = std::floor(x + 0.5); /* Q5: round half up */
  if (steps < 1.0) steps = 1.0;       /* "if the result is less than 1, the delay is set to 1" */
  if (steps > 65535.0) steps = 65535.0;
  out->delay = (uint16_t)(int64_t)steps;
  out->x = x;
  /* D8: "at a rounding boundary": the only synapses allowed to differ by one step on the GPU. */
  bool boundary = std::fabs(x - std::floor(x) - 0.5) < 1e-9;
  if (std::isfinite(dd.lo) && std::fabs(d_ms - dd.lo) <= 1e-12 * std::fabs(dd.lo) && d_ms != dd.lo) boundary = true;
  if (std::isfinite(dd.hi) && std::fabs(d_ms - dd.hi) <= 1e-12 * std::fabs(dd.hi) && d_ms != dd.hi) boundary = true;
  out->boundary = boundary ? 1 : 0;
  out->accepted = 1;
}

int validate(uint32_t n_nodes, oc_range src, oc_range tgt, int rule, const oc_rule_params* params,
             const oc_syn_spec* syn, double inv_dt, uint64_t* n_new_or_pairs) {
  if (!params || !syn) return OC_ERR_INVALID_ARG;
  if (src.count == 0 || tgt.count == 0) return OC_ERR_INVALID_ARG;
  if ((uint64_t)src.first + src.count > n_nodes) return OC_ERR_INVALID_ARG;
  if ((uint64_t)tgt.first + tgt.count > n_nodes) return OC_ERR_INVALID_ARG;
  if (!dist_ok(syn->weight) || !dist_ok(syn->delay_ms)) return OC_ERR_INVALID_ARG;
  const uint64_t K = params->degree_or_total;
  const uint64_t LIMIT = 0xffffffffull; /* u32 positions (hard limit 8 of DESIGN.md) */
  uint64_t n = 0;
  switch (rule) {
    case OC_ONE_TO_ONE:
      if (src.count != tgt.count) return OC_ERR_INVALID_ARG;
      n = src.count; break;
    case OC_ALL_TO_ALL:
      n = (uint64_t)src.count * tgt.count; break;
    case OC_FIXED_OUTDEGREE:
      if (K > LIMIT) return OC_ERR_CAPACITY;
      n = (uint64_t)src.count * K; break;
    case OC_FIXED_INDEGREE:
      if (K > LIMIT) return OC_ERR_CAPACITY;
      n = (uint64_t)tgt.count * K; break;
    case OC_FIXED_TOTAL_NUMBER:
      n = K; break;
    case OC_PAIRWISE_BERNOULLI:
      if (!(params->p >= 0.0 && params->p <= 1.0)) return OC_ERR_INVALID_ARG;
      n = (uint64_t)src.count * tgt.count; break; /* number of trials, not of synapses */
    default:
      return OC_ERR_INVALID_ARG;
  }
  if (rule != OC_PAIRWISE_BERNOULLI && n > LIMIT) return OC_ERR_CAPACITY;
  if (max_delay_steps(syn->delay_ms, inv_dt) > 65535.0) return OC_ERR_CAPACITY;
  *n_new_or_pairs = n;
  return OC_OK;
}

}  // namespace

struct oc_context {
  uint64_t B;
  double dt_ms, inv_dt;
  uint32_t n_nodes = 0;
  uint32_t n_projections = 0;
  std::vector<uint64_t> proj_start; /* bookkeeping: creation position of each projection's first connection */
  bool finalized = false;
  /* D9: creation order, flat (position pos lives in block pos / B, slot pos % B). */
  std::vector<uint32_t> src, tgt;
  std::vector<float> w;
  std::vector<uint16_t> d;
  std::vector<uint8_t> bnd;
  std::vector<uint8_t> port, group; /* receptor port index and synaptic group index of every connection */
  uint8_t cur_port = 0, cur_group = 0;
  uint32_t rule_flags = 0; /* OC_NO_AUTAPSES | OC_NO_MULTAPSES for the connect calls that follow (readings A1-A6) */
  bool sharded = false;    /* reading S1: keep only the connections whose target id lies in [shard_first, shard_first + shard_count) */
  uint32_t shard_first = 0, shard_count = 0;
  uint64_t n_blocks = 0;
  /* D10: sorted copies. */
  std::vector<uint32_t> perm, ssrc, stgt;
  std::vector<float> sw;
  std::vector<uint16_t> sd;
  std::vector<uint8_t> sbnd;
  /* D11 / D12 */
  std::vector<uint32_t> out_degree, in_degree, src_offsets, group_count, group_ptr, group_start;
  std::vector<uint16_t> group_delay;
  bool have_in = false, have_out = false;
};

extern "C" {

void oc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  philox4x32_10(ctr, key, out);
}
uint32_t oc_bounded(uint32_t word, uint32_t n) { return bounded(word, n); }
uint64_t oc_bernoulli_threshold(double p) { return bernoulli_threshold(p); }
uint32_t oc_bernoulli_trial_word(uint64_t seed, uint32_t projection_id, uint64_t q) {
  uint32_t w[4];
  philox_stream(seed, projection_id, 1u, q >> 2, w);
  return w[q & 3];
}

int oc_create(const oc_config* cfg, oc_context** out) {
  if (!cfg || !out) return OC_ERR_INVALID_ARG;
  if (!(cfg->dt_ms > 0.0) || std::isinf(cfg->dt_ms)) return OC_ERR_INVALID_ARG;
  oc_context* c = new (std::nothrow) oc_context();
  if (!c) return OC_ERR_OOM;
  c->B = cfg->block_size ? cfg->block_size : (1ull << 24); /* Q10 */
  c->dt_ms = cfg->dt_ms;
  c->inv_dt = 1.0 / cfg->dt_ms; /* Q5: computed once */
  *out = c;
  return OC_OK;
}

int oc_destroy(oc_context* ctx) {
  delete ctx;
  return OC_OK;
}

/* D1: nodes are identified by consecutive indices. */
int oc_create_population(oc_context* ctx, uint32_t n, uint32_t* first_id) {
  if (!ctx || !first_id || n == 0) return OC_ERR_INVALID_ARG;
  if (ctx->finalized) return OC_ERR_STATE;
  if ((uint64_t)ctx->n_nodes + n > 0xffffffffull) return OC_ERR_CAPACITY;
  *first_id = ctx->n_nodes;
  ctx->n_nodes += n;
  return OC_OK;
}

/* node_space: the size of the index space the two ranges must fit in (the node count, or -- for explicit node
 * arrays, PAPER.md:117 -- the array lengths, because the formulas then produce array indexes). */
static int connect_core(oc_context* ctx, uint64_t node_space, oc_range src, oc_range tgt, int rule,
                        const oc_rule_params* params, const oc_syn_spec* syn, uint64_t seed) {
  if (!ctx) return OC_ERR_INVALID_ARG;
  if (ctx->finalized) return OC_ERR_STATE;
  uint64_t n_iter = 0;
  int rc = validate((uint32_t)std::min<uint64_t>(node_space, 0xffffffffull), src, tgt, rule, params, syn, ctx->inv_dt, &n_iter);
  if (rc != OC_OK) return rc;

  Projection pr{src, tgt, rule, *params, *syn, seed, ctx->n_projections};
  const uint64_t n_before = ctx->src.size();
  try {
    if (rule != OC_PAIRWISE_BERNOULLI) {
      if (n_before + n_iter > 0xffffffffull) return OC_ERR_CAPACITY;
      /* Eq. 2: i_newconns = 0 .. N_newconns - 1, appended contiguously (D9). */
      for (uint64_t i = 0; i < n_iter; ++i) {
        oc_synapse sy;
        eval_synapse(pr, ctx->inv_dt, i, &sy);
        ctx->src.push_back(sy.source);
        ctx->tgt.push_back(sy.target);
        ctx->w.push_back(sy.weight);
        ctx->d.push_back(sy.delay);
        ctx->bnd.push_back(sy.boundary);
      }
    } else {
      /* D4/Q13: every ordered pair tried once, ascending q; accepted pairs are appended in that
       * order, and the synapse stream is indexed by q (not by the rank). */
      const uint64_t T = bernoulli_threshold(params->p);
      uint32_t tw[4] = {0, 0, 0, 0};
      for (uint64_t q = 0; q < n_iter; ++q) {
        if ((q & 3) == 0) philox_stream(seed, pr.id, 1u, q >> 2, tw);
        if ((uint64_t)tw[q & 3] < T) {
          if (ctx->src.size() >= 0xffffffffull) {
            ctx->src.resize(n_before); ctx->tgt.resize(n_before); ctx->w.resize(n_before);
            ctx->d.resize(n_before); ctx->bnd.resize(n_before);
            return OC_ERR_CAPACITY;
          }
          oc_synapse sy;
          eval_synapse(pr, ctx->inv_dt, q, &sy);
          ctx->src.push_back(sy.source);
          ctx->tgt.push_back(sy.target);
          ctx->w.push_back(sy.weight);
          ctx->d.push_back(sy.delay);
          ctx->bnd.push_back(sy.boundary);
        }
      }
    }
  } catch (const std::bad_alloc&) {
    ctx->src.resize(n_before); ctx->tgt.resize(n_before); ctx->w.resize(n_before);
    ctx->d.resize(n_before); ctx->bnd.resize(n_before);
    return OC_ERR_OOM;
  }
  /* Eq. 1: N_newblocks = floor((N_conns + N_newconns + B - 1) / B) - N_blocks. */
  const uint64_t n_conns = n_before, n_newconns = ctx->src.size() - n_before;
  const uint64_t n_newblocks = (n_conns + n_newconns + ctx->B - 1) / ctx->B - ctx->n_blocks;
  ctx->n_blocks += n_newblocks;
  ctx->n_projections += 1;
  ctx->proj_start.push_back(n_before);
  ctx->have_in = ctx->have_out = false;
  ctx->port.resize(ctx->src.size(), ctx->cur_port);   /* the new connections carry the attributes in force */
  ctx->group.resize(ctx->src.size(), ctx->cur_group);
  return OC_OK;
}


/* Readings A1-A6: a connect call with autapses and / or multapses prohibited.  src / tgt are index ranges into the node
 * arrays when those are given (first = 0), node ranges otherwise. */
static int connect_flagged(oc_context* ctx, const uint32_t* src_nodes, oc_range src, const uint32_t* tgt_nodes, oc_range tgt,
                           int rule, const oc_rule_params* params, const oc_syn_spec* syn, uint64_t seed, uint32_t flags) {
  if (ctx->finalized) return OC_ERR_STATE;
  const bool no_aut = (flags & OC_NO_AUTAPSES) != 0, no_mult = (flags & OC_NO_MULTAPSES) != 0;
  uint64_t n_iter = 0;
  const uint64_t space = std::max<uint64_t>(ctx->n_nodes, std::max<uint64_t>(src_nodes ? src.count : 0, tgt_nodes ? tgt.count : 0));
  int rc = validate((uint32_t)std::min<uint64_t>(space, 0xffffffffull), src, tgt, rule, params, syn, ctx->inv_dt, &n_iter);
  if (rc != OC_OK) return rc;
  auto sid = [&](uint64_t sl) -> uint32_t { return src_nodes ? src_nodes[sl] : (uint32_t)(src.first + sl); };
  auto tid = [&](uint64_t tl) -> uint32_t { return tgt_nodes ? tgt_nodes[tl] : (uint32_t)(tgt.first + tl); };
  /* A1: no repeated ids in explicit arrays */
  for (int side = 0; side < 2; ++side) {
    const uint32_t* a = side ? tgt_nodes : src_nodes;
    if (!a) continue;
    std::vector<uint32_t> v(a, a + (side ? tgt.count : src.count));
    std::sort(v.begin(), v.end());
    if (std::adjacent_find(v.begin(), v.end()) != v.end()) return OC_ERR_INVALID_ARG;
  }
  /* index of a node id among the sources / targets, or -1 */
  auto find_in = [&](bool in_src, uint32_t id) -> int64_t {
    const uint32_t* a = in_src ? src_nodes : tgt_nodes;
    const oc_range r = in_src ? src : tgt;
    if (!a) return (id >= r.first && (uint64_t)id < (uint64_t)r.first + r.count) ? (int64_t)(id - r.first) : -1;
    for (uint32_t k = 0; k < r.count; ++k)
      if (a[k] == id) return k;
    return -1;
  };
  const uint64_t K = params->degree_or_total;
  if (rule == OC_FIXED_TOTAL_NUMBER && no_mult) return OC_ERR_INVALID_ARG; /* A6 */
  /* feasibility */
  if (rule == OC_FIXED_INDEGREE || rule == OC_FIXED_OUTDEGREE) {
    const bool indeg = rule == OC_FIXED_INDEGREE;
    const uint64_t n_fixed = indeg ? tgt.count : src.count, n_part = indeg ? src.count : tgt.count;
    for (uint64_t f = 0; f < n_fixed; ++f) {
      const uint32_t fid = indeg ? tid(f) : sid(f);
      const uint64_t e = (no_aut && find_in(indeg, fid) >= 0) ? 1 : 0;
      const uint64_t M = n_part - e;
      if (no_mult ? K > M : (K > 0 && M == 0)) return OC_ERR_INVALID_ARG;
    }
  }
  if (rule == OC_FIXED_TOTAL_NUMBER && no_aut && K > 0 && src.count == 1 && tgt.count == 1 && sid(0) == tid(0))
    return OC_ERR_INVALID_ARG;

  Projection pr{src, tgt, rule, *params, *syn, seed, ctx->n_projections};
  const uint64_t n_before = ctx->src.size();
  auto rollback = [&]() {
    ctx->src.resize(n_before); ctx->tgt.resize(n_before); ctx->w.resize(n_before); ctx->d.resize(n_before); ctx->bnd.resize(n_before);
  };
  auto append = [&](uint64_t idx, uint32_t s_id, uint32_t t_id) { /* weight and delay: words 2, 3 of Philox(idx, stream 0) */
    oc_synapse sy;
    eval_synapse(pr, ctx->inv_dt, idx, &sy);
    ctx->src.push_back(s_id);
    ctx->tgt.push_back(t_id);
    ctx->w.push_back(sy.weight);
    ctx->d.push_back(sy.delay);
    ctx->bnd.push_back(sy.boundary);
  };
  try {
    if (rule == OC_ONE_TO_ONE || rule == OC_ALL_TO_ALL || rule == OC_PAIRWISE_BERNOULLI) { /* A2 */
      const uint64_t T = rule == OC_PAIRWISE_BERNOULLI ? bernoulli_threshold(params->p) : 0;
      uint32_t tw[4] = {0, 0, 0, 0};
      for (uint64_t q = 0; q < n_iter; ++q) {
        if (rule == OC_PAIRWISE_BERNOULLI) {
          if ((q & 3) == 0) philox_stream(seed, pr.id, 1u, q >> 2, tw);
          if (!((uint64_t)tw[q & 3] < T)) continue;
        }
        const uint64_t sl = rule == OC_ONE_TO_ONE ? q : q / tgt.count, tl = rule == OC_ONE_TO_ONE ? q : q % tgt.count;
        if (no_aut && sid(sl) == tid(tl)) continue;
        if (ctx->src.size() >= 0xffffffffull) {
          rollback();
          return OC_ERR_CAPACITY;
        }
        append(q, sid(sl), tid(tl));
      }
    } else {
      if (n_before + n_iter > 0xffffffffull) return OC_ERR_CAPACITY;
      const bool indeg = rule == OC_FIXED_INDEGREE, outdeg = rule == OC_FIXED_OUTDEGREE;
      for (uint64_t i = 0; i < n_iter; ++i) {
        uint32_t w[4];
        if (rule == OC_FIXED_TOTAL_NUMBER) { /* A4 */
          uint64_t sl = 0, tl = 0;
          for (uint32_t a = 0;; ++a) {
            philox_stream(seed, pr.id, a == 0 ? 0u : 1u + a, i, w);
            sl = bounded(w[0], src.count);
            tl = bounded(w[1], tgt.count);
            if (sid(sl) != tid(tl)) break;
            if (a == 63) { /* never reached in practice: take the next target, cyclically */
              tl = (tl + 1) % tgt.count;
              if (sid(sl) == tid(tl)) sl = (sl + 1) % src.count;
              break;
            }
          }
          append(i, sid(sl), tid(tl));
          continue;
        }
        const uint64_t f = i / K, k = i % K; /* fixed node number and which of its K partners */
        const uint32_t fid = indeg ? tid(f) : sid(f);
        const uint32_t n_part = indeg ? src.count : tgt.count;
        uint64_t x = 0;
        if (!no_mult) { /* A3 */
          for (uint32_t a = 0;; ++a) {
            philox_stream(seed, pr.id, a == 0 ? 0u : 1u + a, i, w);
            x = bounded(indeg ? w[0] : w[1], n_part);
            if ((indeg ? sid(x) : tid(x)) != fid) break;
            if (a == 63) {
              x = (x + 1) % n_part;
              break;
            }
          }
        } else { /* A5 */
          const int64_t z = no_aut ? find_in(indeg, fid) : -1;
          const uint32_t M = n_part - (z >= 0 ? 1u : 0u);
          philox_stream(seed, pr.id, 2u, f, w);
          x = keyed_permutation(M, (uint32_t)k, w);
          if (z >= 0 && x >= (uint64_t)z) x += 1;
        }
        (void)outdeg;
        if (indeg) append(i, sid(x), fid);
        else append(i, fid, tid(x));
      }
    }
  } catch (const std::bad_alloc&) {
    rollback();
    return OC_ERR_OOM;
  }
  const uint64_t n_newconns = ctx->src.size() - n_before;
  const uint64_t n_newblocks = (n_before + n_newconns + ctx->B - 1) / ctx->B - ctx->n_blocks; /* Eq. 1 */
  ctx->n_blocks += n_newblocks;
  ctx->n_projections += 1;
  ctx->proj_start.push_back(n_before);
  ctx->have_in = ctx->have_out = false;
  ctx->port.resize(ctx->src.size(), ctx->cur_port);
  ctx->group.resize(ctx->src.size(), ctx->cur_group);
  return OC_OK;
}

int oc_set_rule_flags(oc_context* ctx, uint32_t flags) {
  if (!ctx || (flags & ~3u)) return OC_ERR_INVALID_ARG;
  if (ctx->finalized) return OC_ERR_STATE;
  ctx->rule_flags = flags;
  return OC_OK;
}
uint32_t oc_keyed_permutation(uint32_t M, uint32_t k, const uint32_t keys[4]) { return keyed_permutation(M, k, keys); }

static int connect_impl(oc_context* ctx, oc_range src, oc_range tgt, int rule, const oc_rule_params* params,
                        const oc_syn_spec* syn, uint64_t seed) {
  if (!ctx) return OC_ERR_INVALID_ARG;
  if (ctx->rule_flags) return connect_flagged(ctx, nullptr, src, nullptr, tgt, rule, params, syn, seed, ctx->rule_flags);
  return connect_core(ctx, ctx->n_nodes, src, tgt, rule, params, syn, seed);
}

/* "If the indexes of source or target nodes are not consecutive but are explicitly given by an array,
 * the above formulas are used to derive the indexes of the array elements from which to extract the node indexes."
 * So: run the rule over the index ranges 0..n_src-1 / 0..n_tgt-1 (s0 = t0 = 0), then look every result up. */
static int connect_nodes_impl(oc_context* ctx, const uint32_t* src_nodes, uint32_t n_src, oc_range src,
                              const uint32_t* tgt_nodes, uint32_t n_tgt, oc_range tgt, int rule, const oc_rule_params* params,
                              const oc_syn_spec* syn, uint64_t seed) {
  if (!ctx) return OC_ERR_INVALID_ARG;
  if (ctx->finalized) return OC_ERR_STATE;
  for (uint32_t k = 0; src_nodes && k < n_src; ++k)
    if (src_nodes[k] >= ctx->n_nodes) return OC_ERR_INVALID_ARG;
  for (uint32_t k = 0; tgt_nodes && k < n_tgt; ++k)
    if (tgt_nodes[k] >= ctx->n_nodes) return OC_ERR_INVALID_ARG;
  if (src_nodes) src = oc_range{0u, n_src};
  if (tgt_nodes) tgt = oc_range{0u, n_tgt};
  if ((!src_nodes && (uint64_t)src.first + src.count > ctx->n_nodes) ||
      (!tgt_nodes && (uint64_t)tgt.first + tgt.count > ctx->n_nodes))
    return OC_ERR_INVALID_ARG;
  if (ctx->rule_flags) return connect_flagged(ctx, src_nodes, src, tgt_nodes, tgt, rule, params, syn, seed, ctx->rule_flags);
  const uint64_t space = std::max<uint64_t>(ctx->n_nodes, std::max<uint64_t>(src_nodes ? n_src : 0, tgt_nodes ? n_tgt : 0));
  const size_t before = ctx->src.size();
  int rc = connect_core(ctx, space, src, tgt, rule, params, syn, seed);
  if (rc != OC_OK) return rc;
  for (size_t j = before; j < ctx->src.size(); ++j) {
    if (src_nodes) ctx->src[j] = src_nodes[ctx->src[j]];
    if (tgt_nodes) ctx->tgt[j] = tgt_nodes[ctx->tgt[j]];
  }
  return OC_OK;
}

/* "Weights and delays can have identical values for all connections, or be specified for each
 * connection by an array having a size equal to the number of connections, or be randomly distributed".  The array
 * form: entry i belongs to connection i_newconns = i (Eq. 2); a NULL array leaves that parameter to `syn`.  The
 * rule, its random draws and the other parameter are exactly those of oc_connect_nodes.  A given weight is stored
 * as it is; a given delay in ms goes through reading D8 (times 1/dt, round half up, at least one step). */
static int connect_values_impl(oc_context* ctx, const uint32_t* src_nodes, uint32_t n_src, oc_range src,
                               const uint32_t* tgt_nodes, uint32_t n_tgt, oc_range tgt, int rule, const oc_rule_params* params,
                               const oc_syn_spec* syn, uint64_t seed, const float* weights, const double* delays_ms,
                               uint64_t n_values) {
  if (!ctx) return OC_ERR_INVALID_ARG;
  if (ctx->finalized) return OC_ERR_STATE;
  if (!weights && !delays_ms) return OC_ERR_INVALID_ARG;
  if (rule == OC_PAIRWISE_BERNOULLI) return OC_ERR_INVALID_ARG; /* its number of connections is not known beforehand */
  if ((ctx->rule_flags & OC_NO_AUTAPSES) && (rule == OC_ONE_TO_ONE || rule == OC_ALL_TO_ALL))
    return OC_ERR_INVALID_ARG; /* reading A2: nor is it when pairs with equal ids are left out */
  for (uint64_t i = 0; weights && i < n_values; ++i)
    if (std::isnan(weights[i])) return OC_ERR_INVALID_ARG;
  for (uint64_t i = 0; delays_ms && i < n_values; ++i) {
    if (!std::isfinite(delays_ms[i])) return OC_ERR_INVALID_ARG;
    if (std::floor(delays_ms[i] * ctx->inv_dt + 0.5) > 65535.0) return OC_ERR_CAPACITY;
  }
  const size_t before = ctx->src.size();
  const uint64_t blocks_before = ctx->n_blocks;
  int rc = connect_nodes_impl(ctx, src_nodes, n_src, src, tgt_nodes, n_tgt, tgt, rule, params, syn, seed);
  if (rc != OC_OK) return rc;
  if (ctx->src.size() - before != n_values) { /* "an array having a size equal to the number of connections" */
    ctx->src.resize(before); ctx->tgt.resize(before); ctx->w.resize(before); ctx->d.resize(before); ctx->bnd.resize(before);
    ctx->port.resize(before); ctx->group.resize(before);
    ctx->n_blocks = blocks_before;
    ctx->n_projections -= 1;
    ctx->proj_start.pop_back();
    return OC_ERR_INVALID_ARG;
  }
  for (uint64_t i = 0; i < n_values; ++i) {
    if (weights) ctx->w[before + i] = weights[i];
    if (delays_ms) {
      const double x = delays_ms[i] * ctx->inv_dt;
      double steps = std::floor(x + 0.5);
      if (steps < 1.0) steps = 1.0;
      ctx->d[before + i] = (uint16_t)(int64_t)steps;
      ctx->bnd[before + i] = std::fabs(x - std::floor(x) - 0.5) < 1e-9 ? 1 : 0;
    }
  }
  return OC_OK;
}


/* Reading S1 ("future work is required to extend the algorithm to employing multiple GPUs"):
 * a context that holds ONE SHARD of a network keeps, of every connect call, exactly the connections whose target id lies
 * in [first, first + count) -- the nodes this shard owns -- in the order the full call creates them, with the full call's
 * random numbers (Philox indices are those of the full call) and projection ids.  Everything after that (Eq. 1 blocks,
 * sort, index) runs on what was kept.  Here: generate the full call, then erase what is not owned. */
static void apply_shard(oc_context* ctx, size_t before) {
  if (!ctx->sharded) return;
  size_t o = before;
  for (size_t j = before; j < ctx->src.size(); ++j) {
    const uint32_t t = ctx->tgt[j];
    if (t >= ctx->shard_first && (uint64_t)t < (uint64_t)ctx->shard_first + ctx->shard_count) {
      ctx->src[o] = ctx->src[j]; ctx->tgt[o] = ctx->tgt[j]; ctx->w[o] = ctx->w[j]; ctx->d[o] = ctx->d[j];
      ctx->bnd[o] = ctx->bnd[j]; ctx->port[o] = ctx->port[j]; ctx->group[o] = ctx->group[j];
      ++o;
    }
  }
  ctx->src.resize(o); ctx->tgt.resize(o); ctx->w.resize(o); ctx->d.resize(o); ctx->bnd.resize(o);
  ctx->port.resize(o); ctx->group.resize(o);
  ctx->n_blocks = (o + ctx->B - 1) / ctx->B; /* Eq. 1 over what this shard holds */
}

int oc_set_shard(oc_context* ctx, uint32_t first, uint32_t count) {
  if (!ctx) return OC_ERR_INVALID_ARG;
  if (ctx->finalized || !ctx->src.empty() || ctx->n_projections) return OC_ERR_STATE; /* before the first connect call */
  ctx->sharded = true;
  ctx->shard_first = first;
  ctx->shard_count = count;
  return OC_OK;
}

int oc_connect(oc_context* ctx, oc_range src, oc_range tgt, int rule, const oc_rule_params* params,
               const oc_syn_spec* syn, uint64_t seed) {
  if (!ctx) return OC_ERR_INVALID_ARG;
  const size_t before = ctx->src.size();
  const int rc = connect_impl(ctx, src, tgt, rule, params, syn, seed);
  if (rc == OC_OK) apply_shard(ctx, before);
  return rc;
}
int oc_connect_nodes(oc_context* ctx, const uint32_t* src_nodes, uint32_t n_src, oc_range src,
                     const uint32_t* tgt_nodes, uint32_t n_tgt, oc_range tgt, int rule, const oc_rule_params* params,
                     const oc_syn_spec* syn, uint64_t seed) {
  if (!ctx) return OC_ERR_INVALID_ARG;
  const size_t before = ctx->src.size();
  const int rc = connect_nodes_impl(ctx, src_nodes, n_src, src, tgt_nodes, n_tgt, tgt, rule, params, syn, seed);
  if (rc == OC_OK) apply_shard(ctx, before);
  return rc;
}
int oc_connect_values(oc_context* ctx, const uint32_t* src_nodes, uint32_t n_src, oc_range src,
                      const uint32_t* tgt_nodes, uint32_t n_tgt, oc_range tgt, int rule, const oc_rule_params* params,
                      const oc_syn_spec* syn, uint64_t seed, const float* weights, const double* delays_ms,
                      uint64_t n_values) {
  if (!ctx) return OC_ERR_INVALID_ARG;
  const size_t before = ctx->src.size();
  const int rc = connect_values_impl(ctx, src_nodes, n_src, src, tgt_nodes, n_tgt, tgt, rule, params, syn, seed, weights,
                                     delays_ms, n_values);
  if (rc == OC_OK) apply_shard(ctx, before);
  return rc;
}

/* "The basic structure of a NEST GPU connection includes the source node index, the target node index, the
 * receptor port index, the weight, the delay, and the synaptic group index.  The synaptic group index takes non-zero
 * values only for non-static synapses".  Both are set for the connect calls that follow (0, 0 at the start) and
 * stored with every connection; nothing here interprets them. */
int oc_set_connection_attributes(oc_context* ctx, uint8_t port, uint8_t syn_group) {
  if (!ctx) return OC_ERR_INVALID_ARG;
  if (ctx->finalized) return OC_ERR_STATE;
  ctx->cur_port = port;
  ctx->cur_group = syn_group;
  return OC_OK;
}

/* entries first .. first+count-1 of the creation-order (sorted = 0) or organised (sorted = 1: entry j is the
 * connection created at perm[j]) view; either output may be NULL */
int oc_read_connection_attributes(oc_context* ctx, int sorted, uint64_t first, uint64_t count, uint8_t* port,
                                  uint8_t* syn_group) {
  if (!ctx) return OC_ERR_INVALID_ARG;
  if (sorted && !ctx->finalized) return OC_ERR_STATE;
  if (first + count > ctx->src.size()) return OC_ERR_INVALID_ARG;
  for (uint64_t j = 0; j < count; ++j) {
    const uint64_t pos = sorted ? ctx->perm[first + j] : first + j;
    if (port) port[j] = ctx->port[pos];
    if (syn_group) syn_group[j] = ctx->group[pos];
  }
  return OC_OK;
}

int oc_num_connections(oc_context* ctx, uint64_t* n) {
  if (!ctx || !n) return OC_ERR_INVALID_ARG;
  *n = ctx->src.size();
  return OC_OK;
}
int oc_num_nodes(oc_context* ctx, uint32_t* n) {
  if (!ctx || !n) return OC_ERR_INVALID_ARG;
  *n = ctx->n_nodes;
  return OC_OK;
}
int oc_num_blocks(oc_context* ctx, uint64_t* n_blocks) {
  if (!ctx || !n_blocks) return OC_ERR_INVALID_ARG;
  *n_blocks = ctx->n_blocks;
  return OC_OK;
}
/* bookkeeping for the tests (no arithmetic of the method): creation position at which each projection starts */
int oc_get_projection_starts(oc_context* ctx, const uint64_t** starts, uint32_t* n_projections) {
  if (!ctx || !starts || !n_projections) return OC_ERR_INVALID_ARG;
  *starts = ctx->proj_start.data();
  *n_projections = (uint32_t)ctx->proj_start.size();
  return OC_OK;
}
int oc_block_slot(oc_context* ctx, uint64_t pos, uint64_t* block, uint64_t* slot) {
  if (!ctx || !block || !slot) return OC_ERR_INVALID_ARG;
  *block = pos / ctx->B;
  *slot = pos % ctx->B;
  return OC_OK;
}

/* D10 + D11: organise for spike delivery. */
int oc_finalize(oc_context* ctx) {
  if (!ctx) return OC_ERR_INVALID_ARG;
  if (ctx->finalized) return OC_ERR_STATE;
  const uint64_t n = ctx->src.size();
  const uint32_t N = ctx->n_nodes;
  try {
    /* D10: stable sort, source first key, delay second; ties keep creation order. */
    ctx->perm.resize(n);
    std::iota(ctx->perm.begin(), ctx->perm.end(), 0u);
    const uint32_t* src = ctx->src.data();
    const uint16_t* d = ctx->d.data();
    std::stable_sort(ctx->perm.begin(), ctx->perm.end(), [src, d](uint32_t a, uint32_t b) {
      const uint64_t ka = ((uint64_t)src[a] << 16) | d[a];
      const uint64_t kb = ((uint64_t)src[b] << 16) | d[b];
      return ka < kb;
    });
    ctx->ssrc.resize(n); ctx->stgt.resize(n); ctx->sw.resize(n); ctx->sd.resize(n); ctx->sbnd.resize(n);
    for (uint64_t j = 0; j < n; ++j) {
      const uint32_t p = ctx->perm[j];
      ctx->ssrc[j] = ctx->src[p];
      ctx->stgt[j] = ctx->tgt[p];
      ctx->sw[j] = ctx->w[p];
      ctx->sd[j] = ctx->d[p];
      ctx->sbnd[j] = ctx->bnd[p];
    }
    /* D11: out-degree over ALL nodes (Q9), exclusive scan -> src_offsets. */
    ctx->out_degree.assign(N, 0u);
    for (uint64_t j = 0; j < n; ++j) ctx->out_degree[ctx->ssrc[j]] += 1;
    ctx->src_offsets.assign((size_t)N + 1, 0u);
    for (uint32_t s = 0; s < N; ++s) ctx->src_offsets[s + 1] = ctx->src_offsets[s] + ctx->out_degree[s];
    /* Group heads: source or delay differs from the previous connection. G_i. */
    ctx->group_count.assign(N, 0u);
    std::vector<uint8_t> head(n, 0);
    for (uint64_t j = 0; j < n; ++j) {
      const bool is_head = (j == 0) || ctx->ssrc[j] != ctx->ssrc[j - 1] || ctx->sd[j] != ctx->sd[j - 1];
      head[j] = is_head;
      if (is_head) ctx->group_count[ctx->ssrc[j]] += 1;
    }
    /* Eq. 14: p_i = sum_{j<i} G_j, p_0 = 0; entry N = total (Q8). */
    ctx->group_ptr.assign((size_t)N + 1, 0u);
    for (uint32_t s = 0; s < N; ++s) ctx->group_ptr[s + 1] = ctx->group_ptr[s] + ctx->group_count[s];
    const uint32_t total_groups = ctx->group_ptr[N];
    /* per source, the global indexes of the first connection of each group,
     * all sub-arrays concatenated; sub-array of source i starts at p_i. */
    ctx->group_start.assign(total_groups, 0u);
    ctx->group_delay.assign(total_groups, 0);
    std::vector<uint32_t> fill(N, 0u);
    for (uint64_t j = 0; j < n; ++j) {
      if (!head[j]) continue;
      const uint32_t s = ctx->ssrc[j];
      const uint32_t g = ctx->group_ptr[s] + fill[s]++;
      ctx->group_start[g] = (uint32_t)j;
      ctx->group_delay[g] = ctx->sd[j];
    }
  } catch (const std::bad_alloc&) {
    return OC_ERR_OOM;
  }
  ctx->finalized = true;
  ctx->have_out = true;
  return OC_OK;
}

int oc_get_connections(oc_context* ctx, int sorted, oc_connections_view* out) {
  if (!ctx || !out) return OC_ERR_INVALID_ARG;
  if (sorted && !ctx->finalized) return OC_ERR_STATE;
  std::memset(out, 0, sizeof(*out));
  out->n = ctx->src.size();
  if (sorted) {
    out->source = ctx->ssrc.data(); out->target = ctx->stgt.data(); out->weight = ctx->sw.data();
    out->delay = ctx->sd.data(); out->perm = ctx->perm.data(); out->boundary = ctx->sbnd.data();
  } else {
    out->source = ctx->src.data(); out->target = ctx->tgt.data(); out->weight = ctx->w.data();
    out->delay = ctx->d.data(); out->perm = nullptr; out->boundary = ctx->bnd.data();
  }
  return OC_OK;
}

int oc_get_index(oc_context* ctx, oc_index_view* out) {
  if (!ctx || !out) return OC_ERR_INVALID_ARG;
  if (!ctx->finalized) return OC_ERR_STATE;
  out->src_offsets = ctx->src_offsets.data();
  out->group_count = ctx->group_count.data();
  out->group_ptr = ctx->group_ptr.data();
  out->group_start = ctx->group_start.data();
  out->group_delay = ctx->group_delay.data();
  out->n_nodes = ctx->n_nodes;
  out->total_groups = (uint32_t)ctx->group_start.size();
  return OC_OK;
}

/* D12: per-node degree by plain counting over the creation-order arrays. */
int oc_degree_histogram(oc_context* ctx, int kind, const uint32_t** per_node, uint32_t* max_degree) {
  if (!ctx || (kind != 0 && kind != 1)) return OC_ERR_INVALID_ARG;
  std::vector<uint32_t>& deg = kind == 0 ? ctx->in_degree : ctx->out_degree;
  const std::vector<uint32_t>& col = kind == 0 ? ctx->tgt : ctx->src;
  deg.assign(ctx->n_nodes, 0u);
  for (uint64_t i = 0; i < col.size(); ++i) deg[col[i]] += 1;
  uint32_t mx = 0;
  for (uint32_t v : deg) mx = std::max(mx, v);
  if (per_node) *per_node = deg.data();
  if (max_degree) *max_degree = mx;
  return OC_OK;
}

int oc_eval_synapse(oc_range src, oc_range tgt, int rule, const oc_rule_params* params,
                    const oc_syn_spec* syn, uint64_t seed, uint32_t projection_id, double dt_ms,
                    uint64_t idx, oc_synapse* out) {
  if (!params || !syn || !out || !(dt_ms > 0.0)) return OC_ERR_INVALID_ARG;
  if (src.count == 0 || tgt.count == 0) return OC_ERR_INVALID_ARG;
  Projection pr{src, tgt, rule, *params, *syn, seed, projection_id};
  eval_synapse(pr, 1.0 / dt_ms, idx, out);
  if (rule == OC_PAIRWISE_BERNOULLI) {
    const uint64_t T = bernoulli_threshold(params->p);
    out->accepted = (uint64_t)oc_bernoulli_trial_word(seed, projection_id, idx) < T ? 1 : 0;
  }
  return OC_OK;
}

/* oc_eval_synapse over an array of indexes (the same function, called in a loop): sampled parity at sizes the
 * full oracle cannot hold.  Outputs are HOST arrays of n entries; accepted may be NULL. */
int oc_eval_synapse_batch(oc_range src, oc_range tgt, int rule, const oc_rule_params* params,
                          const oc_syn_spec* syn, uint64_t seed, uint32_t projection_id, double dt_ms,
                          const uint64_t* idx, uint64_t n, uint32_t* source, uint32_t* target, float* weight,
                          uint16_t* delay, uint8_t* boundary, uint8_t* accepted) {
  if (!idx || !source || !target || !weight || !delay || !boundary) return OC_ERR_INVALID_ARG;
  for (uint64_t k = 0; k < n; ++k) {
    oc_synapse sy;
    const int rc = oc_eval_synapse(src, tgt, rule, params, syn, seed, projection_id, dt_ms, idx[k], &sy);
    if (rc != OC_OK) return rc;
    source[k] = sy.source; target[k] = sy.target; weight[k] = sy.weight; delay[k] = sy.delay;
    boundary[k] = sy.boundary;
    if (accepted) accepted[k] = sy.accepted;
  }
  return OC_OK;
}

}  // extern "C"
