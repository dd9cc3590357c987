/*
 * nc_copass.h -- C ABI of the COPASS block-sort (libnc.so): the paper's way of organising connections that are held
 * in fixed-size blocks with auxiliary memory of the order of ONE block (Appendix A; Fig. 6).
 *
 * Two ways in:
 *  1. nc_config.flags |= NC_FLAG_ORGANISE_COPASS (nc.h): nc_finalize then sorts the connections by (source, delay)
 *     inside their storage blocks.  Steps of Fig. 6: (B) every block is sorted by the underlying sort
 *     (the stable radix passes of the default path, one block at a time); per output block b: (C) COPASS partition of
 *     the k sorted logical subarrays -- a common threshold t and left partition sizes m_i with sum m_i = N_b
 *     (Sec. A2-A4); (D) the left partitions are copied to the auxiliary array; (E) the right partitions are shifted
 *     right so that block b becomes free; (F) the auxiliary array is sorted into block b.  The result is the same
 *     stable order as the default path (readings C3, C4, C6 of DESIGN.md), left in the blocks: see
 *     nc_connections_view in nc.h.  By default step (E) is replaced: all partitions are taken at once on the sorted
 *     blocks (extraction b needs the first (b+1) N elements, which does not depend on extraction b-1), the subarrays
 *     are kept as lists of extents ("the subarrays do not need to be stored in contiguous locations"),
 *     each output block is gathered into a spare block and sorted there, and one block is then emptied into the holes
 *     the left partitions left behind and becomes the next spare -- about 2 N records move per extraction instead of
 *     everything to the right of block b.  NC_FLAG_COPASS_SHIFT keeps (C)-(E) to the letter (one partition per output
 *     block on what the previous extraction left; right partitions shifted right, assembled block by block in a spare
 *     block so that no move overlaps its source).  Auxiliary device memory: one spare block (two with the shift: the
 *     auxiliary array of Eq. A3 as well) plus the scratch of the underlying sort for one block -- "the largest
 *     between the auxiliary storage requirement of the underlying sorting algorithm for an array of size m_max and
 *     the auxiliary array" -- instead of 50 bytes per connection.  nc_get_copass_stats reports what the
 *     partitions did.  The organisation rewrites the blocks: should nc_finalize fail under this flag after it has
 *     started (NC_ERR_OOM, NC_ERR_CUDA), the connections are lost and every later call but nc_destroy returns
 *     NC_ERR_STATE; argument and capacity errors are detected before anything is touched.
 *  2. nc_copass_partition: the partition step alone on caller-supplied keys (used by the tests to compare it with
 *     the oracle on inputs the connection keys never produce: long runs of ties, empty subarrays, k up to 4096).
 *
 * Conventions as in nc.h: int status returns (NC_OK or a negative nc_status), no exceptions; pointers are HOST
 * pointers unless named d_*; the calls synchronise the context's stream.
 */
#ifndef NC_COPASS_H_
#define NC_COPASS_H_

#include "nc.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  uint32_t t;          /* common threshold: S_ij <= t for j < m_i, S_ij >= t for j >= m_i (Eqs. A6, A7) */
  uint32_t iterations; /* iteration indices s that computed mu / mu-bar (Eqs. A21-A28) */
  int32_t last_step;   /* 1 = Sec. A3 (condition A36), 2 = Sec. A4 (condition A29) */
} nc_copass_info;

/* COPASS partition.  keys[n_keys]: 32-bit keys; subarray i is keys[start[i] .. start[i]+len[i]),
 * ascending (Eq. A5; not checked), i < k <= 4096.  0 < m < sum len, else NC_ERR_INVALID_ARG.
 * m_out[k] receives the left partition sizes (Eq. A8: their sum is m).  Ties are resolved as in readings C2-C4:
 * widest interval -> lowest i; candidates of Eq. A37 ordered as pairs (value, i); d_i of Eq. A46 lowest i first.
 * The keys are copied to the device, the partition runs there in one kernel (copass_partition_kernel), and the
 * results are copied back. */
int nc_copass_partition(nc_context* ctx, const uint32_t* keys, uint64_t n_keys, const uint32_t* start,
                        const uint32_t* len, uint32_t k, uint32_t m, uint32_t* m_out, nc_copass_info* info);

typedef struct {
  uint32_t partitions;  /* COPASS partitions run by nc_finalize (one per output block but the last) */
  uint32_t iterations;  /* summed over them */
  uint32_t last_step_1; /* how many ended in Sec. A3 */
  uint32_t last_step_2; /* how many ended in Sec. A4 */
  uint64_t n_blocks;    /* k */
  uint64_t aux_bytes;   /* auxiliary device memory the organisation step held at its peak */
  uint64_t records_moved; /* records copied by the moves of Fig. 6 D-E (or by gathering and hole filling) */
} nc_copass_stats;

/* NC_ERR_STATE unless the context was finalized under NC_FLAG_ORGANISE_COPASS. */
int nc_get_copass_stats(nc_context* ctx, nc_copass_stats* out);

#ifdef __cplusplus
}
#endif
#endif /* NC_COPASS_H_ */
