/*
 * oracle.h -- C interface of the CPU ORACLE for the network-construction hot path of
 * arXiv 2306.09855 (Golosio, Villamar, Tiddia et al., "Runtime Construction of Large-Scale
 * Spiking Neuronal Network Models on GPU Devices").
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may load it.  It is a plain, slow,
 * single-threaded fp64 restatement of what the path computes, written from the paper
 * (/root/reference/PAPER.md, cited below as PAPER.md:<line>) and from the readings D1-D12 /
 * Q1-Q20 listed in DESIGN.md.  It shares no code, header, table or helper with the CUDA path
 * under paper_2306_09855_b200/csrc: the struct definitions below are its own.
 *
 * All pointers are HOST pointers.  Every function returns 0 (OC_OK) or a negative error code.
 *
 * Parity status: every function here is pinned by tests/test_oracle_*.py (-m "not gpu") against
 * known-answer vectors, closed forms, invariants, library routines and brute force; the one
 * thing that stays "parity unpinned" is agreement with the PAPER'S OWN implementation, whose
 * RNG (cuRAND) mapping is unspecified and which prints no output values.
 */
#ifndef ORACLE_H_
#define ORACLE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  OC_OK = 0,
  OC_ERR_INVALID_ARG = -1,
  OC_ERR_STATE = -2,
  OC_ERR_CAPACITY = -3,
  OC_ERR_OOM = -4
};

/* Connection rules of PAPER.md:73-115 (Eqs. 4-13) plus pairwise_bernoulli. */
enum {
  OC_ONE_TO_ONE = 0,
  OC_ALL_TO_ALL = 1,
  OC_FIXED_INDEGREE = 2,
  OC_FIXED_OUTDEGREE = 3,
  OC_FIXED_TOTAL_NUMBER = 4,
  OC_PAIRWISE_BERNOULLI = 5
};

typedef struct oc_context oc_context;

typedef struct {
  uint64_t block_size; /* B, connections per block; 0 -> 1<<24 */
  double dt_ms;        /* simulation time resolution in ms */
} oc_config;

typedef struct {
  uint64_t degree_or_total; /* K (fixed_in/outdegree) or N (fixed_total_number) */
  double p;                 /* pairwise_bernoulli connection probability */
} oc_rule_params;

/* normal(mean, sd) clamped to [lo, hi]; sd = 0 -> constant; lo/hi may be -inf/+inf */
typedef struct {
  double mean, sd, lo, hi;
} oc_dist;

typedef struct {
  oc_dist weight;
  oc_dist delay_ms;
} oc_syn_spec;

typedef struct {
  uint32_t first, count;
} oc_range;

typedef struct {
  const uint32_t* source;
  const uint32_t* target;
  const float* weight;
  const uint16_t* delay;   /* integer time steps, >= 1 */
  const uint32_t* perm;    /* sorted view only: creation position of sorted entry j; else NULL */
  const uint8_t* boundary; /* 1 where the delay sits at a rounding/clip boundary (reading D8) */
  uint64_t n;
} oc_connections_view;

typedef struct {
  const uint32_t* src_offsets; /* [n_nodes+1] exclusive scan of out_degree */
  const uint32_t* group_count; /* [n_nodes]   G_i of PAPER.md:121 */
  const uint32_t* group_ptr;   /* [n_nodes+1] p_i of Eq. 14 */
  const uint32_t* group_start; /* [total_groups] sorted position of each group's first connection */
  const uint16_t* group_delay; /* [total_groups] delay (steps) of each group */
  uint32_t n_nodes;
  uint32_t total_groups;
} oc_index_view;

/* ---- the path (same call sequence as the nc_ ABI of include/nc.h) ---- */
int oc_create(const oc_config* cfg, oc_context** out);
int oc_destroy(oc_context* ctx);
int oc_create_population(oc_context* ctx, uint32_t n, uint32_t* first_id);
int oc_connect(oc_context* ctx, oc_range src, oc_range tgt, int rule, const oc_rule_params* params,
               const oc_syn_spec* syn, uint64_t seed);
/* explicit node arrays: HOST arrays of n_src / n_tgt node ids; NULL = use the range of that side */
int oc_connect_nodes(oc_context* ctx, const uint32_t* src_nodes, uint32_t n_src, oc_range src,
                     const uint32_t* tgt_nodes, uint32_t n_tgt, oc_range tgt, int rule, const oc_rule_params* params,
                     const oc_syn_spec* syn, uint64_t seed);
/* per-connection value arrays: HOST arrays of n_values = N_newconns entries, either may be NULL (that
 * parameter then follows syn); entry i belongs to connection i_newconns = i.  pairwise_bernoulli is rejected. */
int oc_connect_values(oc_context* ctx, const uint32_t* src_nodes, uint32_t n_src, oc_range src,
                      const uint32_t* tgt_nodes, uint32_t n_tgt, oc_range tgt, int rule, const oc_rule_params* params,
                      const oc_syn_spec* syn, uint64_t seed, const float* weights, const double* delays_ms,
                      uint64_t n_values);
/* receptor port and synaptic group of the connections created by the connect calls that follow;
 * oc_read_connection_attributes returns them per connection for either view (HOST arrays, either may be NULL) */
int oc_set_connection_attributes(oc_context* ctx, uint8_t port, uint8_t syn_group);
int oc_read_connection_attributes(oc_context* ctx, int sorted, uint64_t first, uint64_t count, uint8_t* port,
                                  uint8_t* syn_group);
/* Prohibiting autapses and multapses ("Autapses and multapses are currently always allowed in NEST GPU;
 * therefore another useful addition would be the possibility to prohibit them (for example, using a flag as in the CPU
 * version of NEST)"; PAPER.md:47, 148 for the allowed default).  The flags hold for the connect calls that follow
 * (0 at the start).  Readings A1-A6 of DESIGN.md section 8c:
 *  A1 an autapse is a connection whose source node id equals its target node id; a multapse is a second connection of
 *     the SAME connect call with the same (source id, target id).  With either flag set, explicit node arrays must not
 *     repeat an id (OC_ERR_INVALID_ARG).
 *  A2 one_to_one, all_to_all, pairwise_bernoulli: every pair occurs at most once, so OC_NO_MULTAPSES changes nothing;
 *     under OC_NO_AUTAPSES the pairs with equal ids are left out, the others keep their pair index q for the synapse
 *     stream (same weight and delay as without the flag) and take consecutive creation positions in ascending q.
 *  A3 fixed_indegree / fixed_outdegree under OC_NO_AUTAPSES alone: connection i redraws its random partner until its id
 *     differs from the fixed node's: attempt 0 is the draw of the unflagged rule (stream 0), attempt a >= 1 takes the
 *     same word of Philox(idx = i, stream = 1 + a); after 64 attempts the next partner index (cyclically) is taken.
 *  A4 fixed_total_number under OC_NO_AUTAPSES: the same with both coordinates redrawn (words 0 and 1).
 *  A5 fixed_indegree / fixed_outdegree under OC_NO_MULTAPSES: the K partners of fixed node number f are the first K values
 *     of a keyed permutation of the M allowed partner indexes, partner(f, k) = skip(perm_M(k; keys(f))), where
 *     M = N_partners - e, e = 1 iff OC_NO_AUTAPSES is also set and f's id is among the partners (at index z), and
 *     skip(x) = x + (e and x >= z).  keys(f) = the four words of Philox(idx = f, stream = 2).  K > M is
 *     OC_ERR_INVALID_ARG.  perm_M: oc_keyed_permutation below.
 *  A6 fixed_total_number under OC_NO_MULTAPSES is not offered (OC_ERR_INVALID_ARG).
 * Weight and delay of connection i always come from words 2 and 3 of Philox(idx = i, stream 0) (D5-D8). */
enum { OC_NO_AUTAPSES = 1, OC_NO_MULTAPSES = 2 };
/* Reading S1: this context holds ONE SHARD of the network: of every connect call it keeps
 * exactly the connections whose target id lies in [first, first + count), in the order the full call creates them and with
 * the full call's random numbers and projection ids.  To be called before the first connect call. */
int oc_set_shard(oc_context* ctx, uint32_t first, uint32_t count);
int oc_set_rule_flags(oc_context* ctx, uint32_t flags);
/* perm_M(k; keys), k < M: a permutation of [0, M) by cycle walking over a balanced Feistel network on 2h bits,
 * h = max(1, ceil(bits(M - 1) / 2)): x = k; repeat { (L, R) = (x >> h, x & (2^h - 1)); 6 + ceil(24 / h) rounds
 * r = 0, 1, ...: (L, R) <- (R, L ^ (mix32(R ^ key_r) & (2^h - 1))), key_r = keys[r & 3] + r * 0x9E3779B9; x = L << h | R }
 * until x < M.  (Narrow halves get more rounds: a two-round differential trail of the network has probability 2^-h, and
 * tests/test_oracle_flags.py sees the resulting excess of neighbouring pairs with six rounds on a 4-bit domain.)
 * mix32(v): v ^= v >> 16; v *= 0x7feb352d; v ^= v >> 15; v *= 0x846ca68b; v ^= v >> 16. */
uint32_t oc_keyed_permutation(uint32_t M, uint32_t k, const uint32_t keys[4]);
int oc_finalize(oc_context* ctx);
int oc_num_connections(oc_context* ctx, uint64_t* n);
int oc_num_nodes(oc_context* ctx, uint32_t* n);
int oc_num_blocks(oc_context* ctx, uint64_t* n_blocks);          /* Eq. 1 */
/* test bookkeeping: creation position of the first connection of each successful connect call (n entries) */
int oc_get_projection_starts(oc_context* ctx, const uint64_t** starts, uint32_t* n_projections);
int oc_block_slot(oc_context* ctx, uint64_t pos, uint64_t* block, uint64_t* slot); /* reading D9 */
int oc_get_connections(oc_context* ctx, int sorted, oc_connections_view* out);
int oc_get_index(oc_context* ctx, oc_index_view* out);
int oc_degree_histogram(oc_context* ctx, int kind /*0=in,1=out*/, const uint32_t** per_node,
                        uint32_t* max_degree);

/* ---- single steps, exposed so the tests can pin them one by one ---- */
/* Philox4x32-10 (Salmon et al., SC'11): reading D2. */
void oc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* rand(N) of PAPER.md:95 as multiply-high: reading D3. */
uint32_t oc_bounded(uint32_t word, uint32_t n);
/* Bernoulli acceptance threshold T = floor(p * 2^32) as u64: reading D4/Q14. */
uint64_t oc_bernoulli_threshold(double p);
/* Trial word of pair q on the trial stream (stream 1): reading D2/D4. */
uint32_t oc_bernoulli_trial_word(uint64_t seed, uint32_t projection_id, uint64_t q);

/* One synapse as a pure function of (seed, projection_id, idx).  idx is i_newconns for every
 * rule except pairwise_bernoulli, where it is the pair index q (and *accepted says whether the
 * pair exists at all).  Used for sampled parity at sizes the full oracle cannot hold. */
typedef struct {
  uint32_t source, target;
  float weight;
  uint16_t delay;
  uint8_t boundary;
  uint8_t accepted;
  double z0, z1; /* Box-Muller pair, reading D6 */
  double x;      /* clamp(mean_d + sd_d z1) * inv_dt, the value that is rounded (reading D8) */
} oc_synapse;
int oc_eval_synapse(oc_range src, oc_range tgt, int rule, const oc_rule_params* params,
                    const oc_syn_spec* syn, uint64_t seed, uint32_t projection_id, double dt_ms,
                    uint64_t idx, oc_synapse* out);

/* the same function over an array of indexes; outputs are HOST arrays of n entries, accepted may be NULL */
int oc_eval_synapse_batch(oc_range src, oc_range tgt, int rule, const oc_rule_params* params,
                          const oc_syn_spec* syn, uint64_t seed, uint32_t projection_id, double dt_ms,
                          const uint64_t* idx, uint64_t n, uint32_t* source, uint32_t* target, float* weight,
                          uint16_t* delay, uint8_t* boundary, uint8_t* accepted);

#ifdef __cplusplus
}
#endif
#endif /* ORACLE_H_ */
