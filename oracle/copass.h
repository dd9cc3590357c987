/*
 * copass.h -- CPU oracle of the COPASS block-sort (Appendix A).
 * TEST INFRASTRUCTURE, like oracle.h: plain single-threaded C++, shares no code with the CUDA path; only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline leg may use it.
 *
 * Two functions, each following the appendix step by step in its own order and notation:
 *   oc_copass_partition   Sec. A2 (iteration, Eqs. A11-A35), Sec. A3 (last step, case 1, Eqs. A36-A43) and
 *                         Sec. A4 (last step, case 2, Eqs. A44-A49);
 *   oc_copass_block_sort  Sec. A1 and Fig. 6 (sort every block; per output block: partition, left partitions to
 *                         the auxiliary array, right partitions shifted right, auxiliary array sorted into the
 *                         block).
 * "Real numbers" of Eqs. A1-A4 are int64 here (the connection keys are integers); thresholds are int64 too.
 *
 * Readings of garbled or open passages (DESIGN.md section 8d lists them as C1-C6):
 *  C1  Eqs. A1, A2, A4 let j run to N_i; the subarrays have N_i elements, j = 0 .. N_i - 1.  "m < sum S_{i,j}"
 *       is m < sum_i N_i; m is positive.
 *  C2  Eq. A21: among equal maxima of m-bar - m-underbar the lowest i is taken.
 *  C3  Eq. A37: with m-bar_i = m-underbar_i + 1 the one element of subarray i strictly between the thresholds has
 *      0-based index m-underbar_i; the candidates are ordered as the PAIRS (value, i) the equation writes down, so
 *      equal values are taken lowest i first.  The threshold reported for this case is the largest value put left.
 *  C4  Eq. A47 contradicts the sentence before it: 0 <= d_i <= mu-bar_i - mu_i is meant.  The
 *      paper leaves the choice of the d_i open; here d_i = min(mu-bar_i - mu_i, d - sum_{j<i} d_j) (lowest i first).
 *  C5  Fig. 6 (E)-(F): the auxiliary array is "copied to the first block" and then "sorted"; read as: the block
 *      ends up holding the sorted auxiliary array.  The last block needs no partition (m would equal the number of
 *      elements left, which Eq. A4's m < sum N_i excludes): everything left is its left partition.
 *  C6  The underlying sort is taken stable.  With C3 and C4 and the logical subarrays kept in block
 *      order, the whole block-sort is then a STABLE sort of A: equal keys keep their original order, which is what
 *      reading D10 (oracle.h) asks of the organised connections.
 *
 * Parity status: pinned by tests/test_oracle_copass.py -- the conditions A6-A8 checked by brute force, the left
 * partitions against the first m elements of a stable merge written with numpy, two hand-computed iterations
 * (tests/golden/copass_partition.txt), Eq. A3 for the auxiliary array, and the block-sort against numpy's stable
 * argsort of the whole array (the plain definition of what it reaches).
 */
#ifndef ORACLE_COPASS_H_
#define ORACLE_COPASS_H_
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  int64_t t;           /* common threshold: S_ij <= t for j < m_i, S_ij >= t for j >= m_i (A6, A7) */
  uint32_t iterations; /* how many iteration indices s computed mu / mu-bar (Eqs. A21-A28) */
  int32_t last_step;   /* 1 = Sec. A3 (condition A36), 2 = Sec. A4 (condition A29) */
} oc_copass_info;

/* Subarray i is keys[start[i] .. start[i] + len[i]), ascending.  0 < m < sum len, else OC_ERR_INVALID_ARG (-1).
 * m_out[k] receives the left partition sizes (A8: their sum is m). */
int oc_copass_partition(const int64_t* keys, const uint64_t* start, const uint64_t* len, uint32_t k, uint64_t m,
                        uint64_t* m_out, oc_copass_info* info);

typedef struct {
  uint64_t aux_peak;        /* most elements the auxiliary array ever held (Eq. A3: max_i N_i) */
  uint64_t moved;           /* elements written while shifting right partitions (Fig. 6E) */
  uint32_t partitions;      /* partition calls */
  uint32_t iterations;      /* summed over them */
  uint32_t last_step_1, last_step_2;
} oc_copass_stats;

/* In-place sort of A = k blocks of sizes N[i], stored one after the other in keys / vals (vals[j] travels with
 * keys[j]).  max_extract < k stops after that many output blocks (Fig. 6 C-F repeated max_extract times) and
 * writes the logical subarrays left over to sub_start / sub_len (k entries each, may be NULL); max_extract >= k
 * runs to the end.  stats may be NULL. */
int oc_copass_block_sort(int64_t* keys, uint32_t* vals, const uint64_t* N, uint32_t k, uint32_t max_extract,
                         uint64_t* sub_start, uint64_t* sub_len, oc_copass_stats* stats);

#ifdef __cplusplus
}
#endif
#endif
