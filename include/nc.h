/*
 * nc.h -- C ABI of the B200-native network-construction library (libnc.so).
 *
 * The library builds the connectivity of a spiking network directly in GPU memory from high-level
 * connection rules and organises it for spike delivery: the hot path of arXiv 2306.09855 (Golosio,
 * Villamar, Tiddia et al., "Runtime Construction of Large-Scale Spiking Neuronal Network Models on
 * GPU Devices").  Citations "PAPER.md:<line>" refer to /root/reference/PAPER.md; "D<n>"/"Q<n>" to the
 * readings listed in DESIGN.md.
 *
 * Call sequence (node creation -> node connection -> calibration):
 *     nc_create -> nc_create_population* -> nc_connect* -> nc_finalize -> nc_get_* / nc_read_* -> nc_destroy
 *
 * Conventions
 *  - Every function returns NC_OK (0) or a negative nc_status; no exception crosses the ABI.
 *    nc_last_error() gives a human-readable message for the last failure on that context.
 *  - One context = one GPU and one CUDA stream.  All kernels are enqueued on that stream; results are
 *    valid for work enqueued later on the same stream, or after nc_synchronize().  Functions that
 *    return host values (nc_num_connections, nc_read_*, nc_degree_histogram's max) synchronise.
 *  - The library owns every device buffer.  It obtains them through nc_config.mem (PyTorch's caching
 *    allocator in the Python binding; cudaMalloc/cudaFree when mem.alloc is NULL) and releases them in
 *    nc_destroy.  Pointers returned by nc_get_* are BORROWED device pointers, valid until nc_destroy;
 *    the caller never frees them.  nc_read_* take HOST pointers owned by the caller.
 *  - There is no CPU fallback: if no CUDA device is usable nc_create fails with NC_ERR_CUDA.
 *  - A failed nc_connect leaves the context unchanged and does not consume a projection id.
 *  - Limits: total connections <= 2^32 - 1, nodes <= 2^32 - 1, delay <= 65535 steps.
 */
#ifndef NC_H_
#define NC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  NC_OK = 0,
  NC_ERR_INVALID_ARG = -1, /* range outside created nodes, count 0, N_src != N_tgt for one_to_one
                              (PAPER.md:79), p outside [0,1], sd < 0, lo > hi, dt <= 0, NULL pointer */
  NC_ERR_STATE = -2,       /* connect/create after finalize, sorted view or index before finalize */
  NC_ERR_CAPACITY = -3,    /* > 2^32-1 connections or nodes, or a delay that can exceed 65535 steps */
  NC_ERR_OOM = -4,         /* the allocator returned NULL */
  NC_ERR_CUDA = -5         /* a CUDA call failed or no device is present */
} nc_status;

/* Connection rules: Eqs. 4-13, names as in Senk et al. 2022.
 * Autapses and multapses are allowed unless nc_set_rule_flags prohibits them. */
typedef enum {
  NC_ONE_TO_ONE = 0,         /* Eqs. 4-5:   s = s0 + i,            t = t0 + i            N = N_src = N_tgt */
  NC_ALL_TO_ALL = 1,         /* Eqs. 6-7:   s = s0 + i / N_tgt,    t = t0 + i % N_tgt    N = N_src N_tgt  */
  NC_FIXED_INDEGREE = 2,     /* Eqs. 10-11: s = s0 + rand(N_src),  t = t0 + i / K        N = N_tgt K      */
  NC_FIXED_OUTDEGREE = 3,    /* Eqs. 8-9:   s = s0 + i / K,        t = t0 + rand(N_tgt)  N = N_src K      */
  NC_FIXED_TOTAL_NUMBER = 4, /* Eqs. 12-13: s = s0 + rand(N_src),  t = t0 + rand(N_tgt)  N given          */
  NC_PAIRWISE_BERNOULLI = 5  /* not in the paper's code; every ordered pair (s,t) of the two
                                ranges is tried once with probability p, pairs kept in ascending
                                q = (s-s0) N_tgt + (t-t0) (readings D4, Q13, Q14) */
} nc_rule;

typedef struct nc_context nc_context; /* opaque */

/* Device-memory provider.  alloc returns a DEVICE pointer aligned to >= 256 bytes or NULL; free releases
 * it.  Both are called on the thread that calls into the library, never from a CUDA callback. */
typedef struct {
  void* (*alloc)(void* user, size_t bytes);
  void (*free)(void* user, void* ptr);
  void* user;
} nc_allocator;

enum {
  NC_FLAG_TIMING = 1u << 0,     /* record CUDA events around every phase (nc_get_timings) */
  NC_FLAG_EXACT_FP64 = 1u << 1, /* debug: draw every delay on the fp64 path (no fp32 fast path) */
  NC_FLAG_SORT_PAIRS = 1u << 2, /* sort (key, position) pairs with single-pass digit sweeps (decoupled look-back)
                                   and gather target/weight by the permutation afterwards, instead of carrying
                                   the whole connection through the digit passes; keys wider than 32 bits always
                                   take this path */
  NC_FLAG_SORT_ONESWEEP = 1u << 3, /* carry the whole connection, but chain the tiles of a digit pass inside the
                                   pass (decoupled look-back) instead of the default count / scan / scatter
                                   kernels per pass */
  NC_FLAG_ORGANISE_COPASS = 1u << 4, /* organise the connections INSIDE their storage blocks with the COPASS block-sort
                                   of PAPER.md:426-642 (Appendix A): auxiliary memory of a few blocks instead of two
                                   more copies of all connections.  The organised view then keeps the block structure
                                   (see nc_connections_view) and the creation-order view is gone after nc_finalize.
                                   Needs a (source, delay) key of <= 32 bits and <= 4096 blocks (NC_ERR_CAPACITY).
                                   See include/nc_copass.h. */
  NC_FLAG_COPASS_SHIFT = 1u << 5,  /* with NC_FLAG_ORGANISE_COPASS: follow Fig. 6 C-E to the letter (one partition per
                                   output block on what the previous extraction left, right partitions shifted
                                   right) instead of the default extraction by hole filling (include/nc_copass.h) */
  NC_FLAG_SORT_BULK = 1u << 6,     /* default organisation path, but every digit pass runs as a persistent kernel fed by
                                   the bulk-async copy engine (cp.async.bulk loads of whole tiles tracked by mbarriers,
                                   one bulk store per digit run) instead of one CTA per tile with ordinary loads and
                                   stores.  Same result bit for bit; measured on par, kept selectable.
                                   The first pass takes this form only when block_size is a multiple of 4096. */
  NC_FLAG_SORT_BUCKETS = 1u << 7   /* bucket-first organisation (keys of at most 32 bits): one stable pass scatters the
                                   connections into at most 256 buckets of consecutive source ids, then every bucket is
                                   sorted on its own by the remaining key bits with its intermediate records in a slot
                                   meant to stay in the L2 cache (66 instead of 102 bytes of device-memory traffic per
                                   connection for configs[2] if it does).  Same result bit for bit.  nc_finalize waits
                                   for the device once (the 256 bucket sizes); with other than two in-bucket passes it
                                   spreads the buckets over up to three CUDA streams of its own, joined again before it
                                   returns.  Measured SLOWER than the default on a B200 (the pass is bound by the SM, not
                                   by HBM); kept selectable as the evidence. */
};

typedef struct {
  uint64_t block_size; /* B: connections per storage block.  0 -> 2^24.  Any B >= 1 works;
                          the paper's default 10^7 too (Q10). */
  double dt_ms;        /* simulation time resolution in ms; delays are stored in units of it */
  nc_allocator mem;    /* device memory provider; mem.alloc == NULL -> cudaMalloc / cudaFree */
  void* cuda_stream;   /* cudaStream_t all work is enqueued on (NULL = the legacy default stream) */
  int32_t device;      /* CUDA device ordinal; -1 = the calling thread's current device */
  uint32_t flags;      /* NC_FLAG_* */
} nc_config;

typedef struct {
  uint64_t degree_or_total; /* K for fixed_indegree / fixed_outdegree, N for fixed_total_number */
  double p;                 /* connection probability for pairwise_bernoulli, in [0, 1] */
} nc_rule_params;

/* Normal(mean, sd) clamped to [lo, hi] (never redrawn, Q4).  sd = 0 -> the constant `mean`
 * ("identical values for all connections").  lo / hi may be -INFINITY / +INFINITY. */
typedef struct {
  double mean, sd, lo, hi;
} nc_dist;

/* Per-connection parameters: weight, and delay in ms which is converted to integer time
 * steps by dividing by dt, rounding half up and clamping to [1, 65535] (readings D8, Q5, Q6). */
typedef struct {
  nc_dist weight;
  nc_dist delay_ms;
} nc_syn_spec;

typedef struct {
  uint32_t first, count; /* nodes first .. first+count-1 (consecutive indexes) */
} nc_range;

/* Connections, either in creation order (sorted = 0) or organised for delivery (sorted = 1).
 *  sorted = 1: source/target/weight/delay/perm are flat device arrays of n entries ordered by
 *              (source, delay, creation position) (D10); perm[j] = creation position.
 *  sorted = 0: the connections live in n_blocks storage blocks of block_size entries.
 *              blocks is a HOST array of n_blocks device base pointers; inside a block the four arrays
 *              start at byte offsets off_source/off_target/off_weight/off_delay.  Creation position pos
 *              is entry pos % block_size of block pos / block_size (D9).  The flat pointers are NULL
 *              unless n_blocks == 1, in which case they point into that single block.  The block pointers stay valid
 *              until nc_destroy; the HOST array `blocks` itself is valid until the next nc_connect* call (which may
 *              append to it and move it) -- ask for the view again after connecting.
 *  sorted = 1 under NC_FLAG_ORGANISE_COPASS: the organised connections stay in the storage blocks: sorted position j
 *              is entry j % block_size of block j / block_size, the view is filled as for sorted = 0 plus
 *              off_perm (creation positions), and sorted = 0 is NC_ERR_STATE after nc_finalize (the blocks were
 *              sorted in place). */
typedef struct {
  const uint32_t* source;
  const uint32_t* target;
  const float* weight;
  const uint16_t* delay;
  const uint32_t* perm;
  uint64_t n;
  uint64_t block_size;
  uint64_t n_blocks;
  void* const* blocks;
  uint64_t off_source, off_target, off_weight, off_delay;
  uint64_t off_perm; /* only under NC_FLAG_ORGANISE_COPASS with sorted = 1, else 0 */
} nc_connections_view;

/* Index over the sorted connections (D11).  All device pointers.
 *  src_offsets[s] .. src_offsets[s+1]: sorted positions of the connections of source s   [n_nodes+1]
 *  group_count[s]  = G_s, number of distinct delays of source s            [n_nodes]
 *  group_ptr[s]    = p_s = sum_{j<s} G_j (Eq. 14), group_ptr[n_nodes] = total_groups      [n_nodes+1]
 *  group_start[g]  = sorted position of the first connection of group g    [total_groups]
 *  group_delay[g]  = delay in steps shared by the connections of group g                  [total_groups] */
typedef struct {
  const uint32_t* src_offsets;
  const uint32_t* group_count;
  const uint32_t* group_ptr;
  const uint32_t* group_start;
  const uint16_t* group_delay;
  uint32_t n_nodes;
  uint32_t total_groups;
} nc_index_view;

typedef enum {
  NC_PHASE_GENERATE = 0, /* rule expansion + draws + append (nc_connect) */
  NC_PHASE_HISTOGRAM = 1, /* sort: digit histograms over the packed (source, delay) key */
  NC_PHASE_SORT = 2,     /* sort: digit passes (scatter kernels) */
  NC_PHASE_PERMUTE = 3,  /* materialise sorted source/target/weight/delay */
  NC_PHASE_INDEX = 4,    /* head flags, scans, group compaction */
  NC_PHASE_DEGREE = 5,   /* nc_degree_histogram */
  NC_PHASE_COPASS = 6,   /* COPASS organisation: partitions and the moves of Fig. 6 D-E */
  NC_PHASE_COUNT = 7
} nc_phase;

typedef struct {
  double ms[NC_PHASE_COUNT];          /* device time per phase, summed over the context's life */
  uint32_t launches[NC_PHASE_COUNT];  /* kernels launched per phase */
  double sort_pass_ms;                /* device time of the digit-pass kernels alone */
  uint32_t sort_passes;               /* how many digit-pass kernels ran */
} nc_timings;

typedef struct {
  uint64_t kernel_launches;   /* kernels this context launched so far */
  uint64_t bytes_in_use;      /* device bytes currently held */
  uint64_t bytes_peak;        /* high-water mark of bytes_in_use */
  uint64_t n_blocks;          /* storage blocks allocated (Eq. 1) */
  uint32_t n_projections;     /* successful nc_connect calls */
  uint32_t key_bits;          /* width of the packed (source, delay) sort key, set by nc_finalize */
  uint32_t sort_passes;       /* digit passes nc_finalize used */
  uint32_t delay_bits;        /* bits of the key that hold the delay */
} nc_stats;

/* ---- lifecycle ---- */
int nc_create(const nc_config* cfg, nc_context** out);
int nc_destroy(nc_context* ctx); /* NC_ERR_STATE, nothing destroyed, while nc_delivery objects of the context exist (nc_delivery.h) */
const char* nc_last_error(nc_context* ctx);
int nc_synchronize(nc_context* ctx);

/* ---- node creation (D1): ids are contiguous, *first_id = nodes created so far ---- */
int nc_create_population(nc_context* ctx, uint32_t n, uint32_t* first_id);

/* ---- node connection.  Appends N_newconns connections at creation positions
 * N_conns .. N_conns+N_newconns-1, allocating floor((N_conns+N_newconns+B-1)/B) - N_blocks new blocks (Eq. 1).
 * Connection i draws its randomness from Philox4x32-10 keyed by (seed, projection_id, i) (D2), where
 * projection_id = number of earlier successful nc_connect calls, so the result does not depend on thread
 * order.  Asynchronous except for pairwise_bernoulli, which waits for its exact count. ---- */
int nc_connect(nc_context* ctx, nc_range src, nc_range tgt, nc_rule rule, const nc_rule_params* params,
               const nc_syn_spec* syn, uint64_t seed);

/* Prohibiting autapses and multapses ("Autapses and multapses are currently always allowed in NEST GPU;
 * therefore another useful addition would be the possibility to prohibit them (for example, using a flag as in the CPU
 * version of NEST)"; PAPER.md:47, 148 for the allowed default).  The flags hold for the nc_connect* calls that follow
 * (0 at nc_create).  Readings:
 *  A1 an autapse is a connection whose source node id equals its target node id; a multapse is a second connection of the
 *     SAME connect call with the same (source id, target id).  With either flag set, explicit node arrays must not repeat
 *     an id (NC_ERR_INVALID_ARG).
 *  A2 one_to_one, all_to_all, pairwise_bernoulli: every pair occurs at most once, so NC_NO_MULTAPSES changes nothing;
 *     under NC_NO_AUTAPSES the pairs with equal ids are left out, the others keep their pair index q for the synapse stream
 *     (same weight and delay as without the flag) and take consecutive creation positions in ascending q; the call then
 *     waits for its exact count like pairwise_bernoulli, and nc_connect_values refuses these two rules.
 *  A3 fixed_indegree / fixed_outdegree under NC_NO_AUTAPSES alone: connection i redraws its random partner until its id
 *     differs from the fixed node's: attempt 0 is the draw of the unflagged rule (stream 0), attempt a >= 1 takes the same
 *     word of Philox(idx = i, stream = 1 + a); after 64 attempts the next partner index (cyclically) is taken.  Only the
 *     connections that were autapses change.
 *  A4 fixed_total_number under NC_NO_AUTAPSES: the same with both coordinates redrawn (words 0 and 1).
 *  A5 fixed_indegree / fixed_outdegree under NC_NO_MULTAPSES: the K partners of fixed node number f are the first K values
 *     of a keyed permutation of the M allowed partner indexes, partner(f, k) = skip(perm_M(k; keys(f))), M = N_partners - e,
 *     e = 1 iff NC_NO_AUTAPSES is also set and f's id is among the partners (at index z), skip(x) = x + (e and x >= z),
 *     keys(f) = the four words of Philox(idx = f, stream 2).  perm_M: cycle walking over a balanced Feistel network on 2h
 *     bits, h = max(1, ceil(bits(M - 1) / 2)), 6 + ceil(24 / h) rounds (L, R) <- (R, L ^ (mix32(R ^ key_r) & (2^h - 1))),
 *     key_r = keys[r & 3] + r * 0x9E3779B9, mix32(v): v ^= v >> 16; v *= 0x7feb352d; v ^= v >> 15; v *= 0x846ca68b;
 *     v ^= v >> 16.  K > M for some fixed node is NC_ERR_INVALID_ARG.
 *  A6 fixed_total_number under NC_NO_MULTAPSES is not offered (NC_ERR_INVALID_ARG).
 * Weight and delay of connection i always come from words 2 and 3 of Philox(idx = i, stream 0) (D5-D8). ---- */
enum { NC_NO_AUTAPSES = 1u, NC_NO_MULTAPSES = 2u };
int nc_set_rule_flags(nc_context* ctx, uint32_t flags);

/* One shard of a network per context ("future work is required to extend the algorithm to employing multiple
 * GPUs"; reading S1): after nc_set_shard(first, count) every nc_connect* call keeps exactly the connections whose TARGET id
 * lies in first .. first + count - 1 -- the nodes this shard owns -- in the order the full call creates them, with the full
 * call's random numbers (Philox indices are those of the full call) and projection ids; Eq. 1, the sort and the index then
 * run over what was kept, so perm refers to the shard's own creation positions.  One process per GPU builds one shard;
 * the shards of a partition of the nodes together hold every connection of the unsharded network exactly once, each in the
 * unsharded order (creation order and organised order), without any exchange between ranks: a rank draws the random
 * numbers of the connections it does not own as well and skips them (owner-computes with redundant generation; only
 * one_to_one, fixed_indegree and all_to_all over a target range generate just the owned connections -- an index sub-range,
 * or for all_to_all the owned target columns of every source -- without flags or value arrays).  Any other call is staged in
 * full on the device first, 14 B per connection of the FULL call, in staging blocks that are reused from call to call and
 * released by nc_finalize; staged calls are filtered in batches (after 2^28 staged connections, before a call that would
 * not fit behind them, and by every query), which waits for the owned count.  Generation time, filter time and staging
 * memory of such calls therefore do not shrink with the number of shards.  To be called before the first nc_connect*;
 * first + count <= 2^32 (NC_ERR_INVALID_ARG); node ids outside the created nodes own nothing. ---- */
int nc_set_shard(nc_context* ctx, uint32_t first, uint32_t count);

/* The same with explicit node arrays ("If the indexes of source or target nodes are not consecutive but
 * are explicitly given by an array, the above formulas are used to derive the indexes of the array elements from
 * which to extract the node indexes").  src_nodes / tgt_nodes are HOST arrays of n_src / n_tgt node ids (copied
 * during the call -- the call waits for the upload, pageable or page-locked, so the arrays may be reused on return;
 * ids may repeat and need not be sorted; every id must be a created node, else NC_ERR_INVALID_ARG);
 * a NULL array means "use the range argument of that side".  Rule formulas and random draws are those of nc_connect
 * with N_sources = n_src, N_targets = n_tgt and s0 = t0 = 0; the result indexes the arrays. ---- */
int nc_connect_nodes(nc_context* ctx, const uint32_t* src_nodes, uint32_t n_src, nc_range src,
                     const uint32_t* tgt_nodes, uint32_t n_tgt, nc_range tgt, nc_rule rule,
                     const nc_rule_params* params, const nc_syn_spec* syn, uint64_t seed);

/* The same with per-connection values (weights and delays can "be specified for each connection by an
 * array having a size equal to the number of connections").  weights[n_values] (fp32, stored as they are) and
 * delays_ms[n_values] (fp64, in ms; converted like a drawn delay: times 1/dt, rounded half up, at least one step --
 * readings D8, Q5) are HOST arrays, copied during the call; entry i belongs to connection i_newconns = i of the rule
 * (Eq. 2).  Either may be NULL: that parameter then follows `syn`, as does nothing else -- sources, targets and the
 * other parameter are exactly those nc_connect_nodes gives for the same arguments.  n_values must equal N_newconns of
 * the rule, the delays must be finite and the weights not NaN (NC_ERR_INVALID_ARG), no delay may exceed 65535 steps
 * (NC_ERR_CAPACITY); pairwise_bernoulli, whose count is not known beforehand, is rejected (NC_ERR_INVALID_ARG).
 * src_nodes / tgt_nodes as in nc_connect_nodes (NULL = the range). ---- */
int nc_connect_values(nc_context* ctx, const uint32_t* src_nodes, uint32_t n_src, nc_range src,
                      const uint32_t* tgt_nodes, uint32_t n_tgt, nc_range tgt, nc_rule rule,
                      const nc_rule_params* params, const nc_syn_spec* syn, uint64_t seed, const float* weights,
                      const double* delays_ms, uint64_t n_values);

/* Receptor port and synaptic group (a connection "includes the source node index, the target node index,
 * the receptor port index, the weight, the delay, and the synaptic group index.  The synaptic group index takes
 * non-zero values only for non-static synapses").  The pair set here (0, 0 at the start) belongs to every connection
 * the following nc_connect* calls create.  Both are constants of a projection, so the library keeps them per
 * projection instead of per connection; nc_read_connection_attributes resolves entries first .. first+count-1 of
 * either view through their creation positions and copies them to HOST arrays (either may be NULL; synchronises).
 * The library stores and returns them; synapses are static, and spike delivery (nc_delivery.h) adds a connection's weight
 * to input [port * n_nodes + target], one fp32 accumulator per (receptor port, node), 1 + the largest port in use ports. ---- */
int nc_set_connection_attributes(nc_context* ctx, uint8_t port, uint8_t syn_group);
int nc_read_connection_attributes(nc_context* ctx, int sorted, uint64_t first, uint64_t count, uint8_t* port,
                                  uint8_t* syn_group);

/* ---- calibration: stable sort by (source, delay), then the group index ---- */
int nc_finalize(nc_context* ctx);

/* ---- queries ---- */
int nc_num_connections(nc_context* ctx, uint64_t* n);
int nc_num_nodes(nc_context* ctx, uint32_t* n);
int nc_get_connections(nc_context* ctx, int sorted, nc_connections_view* out);
int nc_get_index(nc_context* ctx, nc_index_view* out);
/* kind 0 = in-degree (counted over targets), 1 = out-degree (counted over sources); *per_node_degree is a
 * borrowed device array of n_nodes entries; *max_degree is written to host (synchronises).  Either may be NULL. */
int nc_degree_histogram(nc_context* ctx, int kind, const uint32_t** per_node_degree, uint32_t* max_degree);
int nc_get_stats(nc_context* ctx, nc_stats* out);
/* Needs NC_FLAG_TIMING; synchronises the stream. */
int nc_get_timings(nc_context* ctx, nc_timings* out);

/* ---- host-buffer reads (device -> host copies; every destination is a HOST pointer and may be NULL) ----
 * nc_read_connections copies entries first .. first+count-1 of the chosen view (gathering across storage
 * blocks for the creation-order view).  perm is only written for sorted = 1. */
int nc_read_connections(nc_context* ctx, int sorted, uint64_t first, uint64_t count, uint32_t* source,
                        uint32_t* target, float* weight, uint16_t* delay, uint32_t* perm);
int nc_read_index(nc_context* ctx, uint32_t* src_offsets, uint32_t* group_count, uint32_t* group_ptr,
                  uint32_t* group_start, uint16_t* group_delay);
int nc_read_degree_histogram(nc_context* ctx, int kind, uint32_t* per_node_degree, uint32_t* max_degree);

/* ---- device self-tests used by the GPU test-suite (each runs a small kernel on the context's stream) ----
 * nc_selftest_philox: out[4*k..4*k+3] = Philox4x32-10(ctr[4*k..], key[2*k..]) computed on the device (D2).
 * nc_selftest_fastpath: exhaustive check of the fp32 Box-Muller fast path against fp64 on the device over all
 *   2^24 values of u1 and of u2 (D5, D6).  out[0] = max |r32 - r64| / (bound on it that the delay guard band
 *   assumes), out[1], out[2] = the same ratio for sin and cos, out[3] = max |r32 - r64| (the fp32 weight is off by
 *   at most sd_w (out[3] + r |cos32 - cos|)).  The guard band is sound iff out[0..2] < 1; the GPU tests require
 *   < 0.25 and out[3] < 4e-6.
 * nc_selftest_guard: with NC_GUARD=1 in the environment at nc_create, every device buffer of the library lies between two
 *   256-byte guard zones that are compared when the buffer is released (a stand-in where compute-sanitizer cannot be
 *   run: writes up to 256 bytes outside a buffer are counted, reported on stderr, and make nc_destroy return
 *   NC_ERR_STATE).  The self-test writes one byte behind a scratch buffer (offset = 1) or before it (offset = -1) or
 *   nowhere (0) and returns in *violations how many guard zones were found overwritten when it was released.
 *   NC_ERR_STATE when guards are off. */
int nc_selftest_philox(nc_context* ctx, uint32_t n, const uint32_t* ctr, const uint32_t* key, uint32_t* out);
int nc_selftest_fastpath(nc_context* ctx, double out[4]);
int nc_selftest_guard(nc_context* ctx, int offset, uint64_t* violations);

#ifdef __cplusplus
}
#endif
#endif /* NC_H_ */
