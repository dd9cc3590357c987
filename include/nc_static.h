/*
 * nc_static.h -- one entry point of libnc.so that never allocates device memory: the group index of PAPER.md:121-132
 * (group heads, src_offsets, p_i of Eq. 14, G_i) over connections that are already organised, i.e. what nc_finalize
 * builds as its last step, for callers that hold the organised source / delay arrays themselves.
 *
 * Who this is for.  Every other call of the library takes its working memory from nc_config.mem or cudaMalloc.  Some
 * callers cannot do that at the point where they need the index:
 *   - code that runs inside a loop with a latency budget (a simulation that re-organises or re-indexes connections between
 *     time steps): cudaMalloc and cudaFree make the whole device wait and take a driver lock, so one call stalls every
 *     stream of the process;
 *   - a process whose own pool already holds all of the device's memory (a simulator that reserved the card at start-up, a
 *     framework allocator that was told to take everything): a cudaMalloc from inside a library then simply fails;
 *   - code that was handed a stream and a set of buffers by its host application and was told to touch nothing else.
 * For them nc_index_static keeps the scratch it needs -- one 64-bit status word per tile of 16,384 connections, a tile
 * ticket -- in an array that is part of the library image itself (a file-scope `static __device__` array in
 * csrc/nc_index_static.cu, NC_INDEX_STATIC_SCRATCH_BYTES = 524,544 bytes).  Every GPU on which the library is loaded holds
 * that array from the moment the module is loaded until the process exits, whether the entry point is ever called or not.
 * The price is the fixed maximum below.
 *
 * Everything else is as in nc.h: int status returns, no exception crosses the ABI; pointers named d_* are DEVICE pointers
 * that the caller owns and keeps alive until the work enqueued by the call has finished.
 */
#ifndef NC_STATIC_H_
#define NC_STATIC_H_

#include "nc.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Largest n the entry point takes: 2^30 connections = 65,536 tiles = 512 KB of status words.  (configs[2], the full-scale
 * cortical microcircuit, has 2.99 * 10^8.) */
#define NC_INDEX_STATIC_MAX_CONNECTIONS (1ull << 30)
#define NC_INDEX_STATIC_SCRATCH_BYTES (65536ull * 8ull + 256ull)

/* bits of *d_error */
enum {
  NC_INDEX_STATIC_LOOKBACK = 1u, /* a tile waited for its predecessors longer than the spin limit (the device was
                                    time-sliced or halted under a debugger); the outputs are incomplete */
  NC_INDEX_STATIC_GROUPS = 2u    /* more than group_capacity groups: group_start / group_delay hold the first
                                    group_capacity of them, every other output is complete and *d_total_groups says how
                                    many entries the group arrays need */
};

/* Index over n organised connections (D11 of DESIGN.md), same arrays as nc_index_view:
 *   in   d_source[n], d_delay[n]   source node id and delay in steps of every connection, ascending by (source, delay);
 *                                  ids < n_nodes; both arrays aligned to 16 bytes.  Neither is checked on the device.
 *   out  d_src_offsets[n_nodes+1]  positions of the connections of source s: d_src_offsets[s] .. d_src_offsets[s+1]
 *        d_group_ptr[n_nodes+1]    p_s of Eq. 14; d_group_ptr[n_nodes] = number of groups
 *        d_group_count[n_nodes]    G_s (may be NULL: not written)
 *        d_group_start[group_capacity], d_group_delay[group_capacity]
 *                                  first position and delay of group g, g < min(groups, group_capacity).  A capacity of
 *                                  min(n, n_nodes * largest delay) always suffices.
 *        d_total_groups[1]         number of groups
 *        d_error[1]                0, or NC_INDEX_STATIC_* bits (cleared by the call before the kernel runs)
 *   cuda_stream                    cudaStream_t (NULL = the legacy default stream) of the calling thread's CURRENT device,
 *                                  which is also the device the pointers must belong to.
 * The call enqueues a few small memsets and at most two kernels on that stream and returns without waiting; the outputs
 * are valid for work enqueued later on the same stream.  It calls no cudaMalloc, cudaFree or any routine that allocates,
 * and copies nothing to or from the host.
 *
 * Set-up: the first call on a device looks up the device address of the scratch array (cudaGetSymbolAddress with that
 * device current; with CUDA's lazy loading this is also what loads the module on that device) and keeps it for the life
 * of the process.  Make that first call once per device during start-up, outside any stream capture and before the
 * latency-critical part begins; n = 0 is enough.
 *
 * Sharing: there is ONE scratch array per device, shared by every call from every thread.  The call clears the part it
 * uses on `cuda_stream` before its kernel, so calls that follow one another on one stream -- or that are otherwise ordered
 * on the GPU -- are independent of what the previous call left behind.  Two calls that may run at the same time on one
 * device (different streams without an event between them, different host threads with their own streams) RACE on the
 * status words and give wrong indexes or NC_INDEX_STATIC_LOOKBACK; ordering them is the caller's job.
 *
 * Errors: NC_ERR_CAPACITY when n > NC_INDEX_STATIC_MAX_CONNECTIONS (nothing is enqueued; nc_finalize, which allocates, is
 * the path for larger networks) or when the current device's ordinal is above 63; NC_ERR_INVALID_ARG for a NULL or
 * misaligned array or connections without nodes (n > 0 with n_nodes = 0); NC_ERR_CUDA when a CUDA call fails.  If err_msg
 * is not NULL a NUL-terminated description of the failure (at most err_cap bytes) is written there; it is left untouched
 * on NC_OK. */
int nc_index_static(const uint32_t* d_source, const uint16_t* d_delay, uint64_t n, uint32_t n_nodes,
                    uint32_t* d_src_offsets, uint32_t* d_group_ptr, uint32_t* d_group_count, uint32_t* d_group_start,
                    uint16_t* d_group_delay, uint64_t group_capacity, uint32_t* d_total_groups, uint32_t* d_error,
                    void* cuda_stream, char* err_msg, size_t err_cap);

#ifdef __cplusplus
}
#endif
#endif /* NC_STATIC_H_ */
