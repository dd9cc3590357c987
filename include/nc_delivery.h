/*
 * nc_delivery.h -- C ABI of spike delivery over the index built by nc_finalize (libnc.so).
 *
 * PAPER.md:136 (Sec. II.C, "The spike buffer"): every spike a node emits is buffered with a time index and a
 * connection-group index, both zero; every step the time indexes grow by one; a spike whose time index equals the
 * delay of the group it points at enters the spike array as (source, group, multiplicity) and moves on to the
 * source's next group (delays ascend inside a source); the connections of the groups in the spike
 * array are then delivered in parallel, one thread per connection.
 *
 * Readings: F1 one step = advance, collect matured, deliver, then insert the spikes
 * emitted in this step, so a spike emitted in step k reaches a connection of delay d in step k + d; F2 the input of
 * a node is one fp32 accumulator per (receptor port, node), every connection adds weight * multiplicity;
 * F3 group indexes in the spike array are global (group_ptr[source] + local index, Eq. 14).
 *
 * Conventions as in nc.h: int status returns, no exceptions; all work is enqueued on the context's stream; the
 * nc_delivery object borrows the context's sorted arrays and index and allocates from it: it must be destroyed before the
 * context, and nc_destroy returns NC_ERR_STATE (destroying nothing) while a delivery object of the context still exists.
 * Pointers named d_* are DEVICE pointers owned by the caller; the others are HOST pointers.
 */
#ifndef NC_DELIVERY_H_
#define NC_DELIVERY_H_

#include "nc.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nc_delivery nc_delivery; /* opaque */

/* capacity = the largest number of spikes that may be buffered at once (roughly spikes per step x largest delay in
 * steps).  The context must be finalized (else NC_ERR_STATE).  Allocates 2 x 16 B + 2 x 8 B per unit of capacity. */
int nc_delivery_create(nc_context* ctx, uint32_t capacity, nc_delivery** out);
int nc_delivery_destroy(nc_delivery* d);

/* Number of receptor ports in use: 1 + the largest port any projection was given (nc_set_connection_attributes,
 * PAPER.md:53); 1 unless ports were set. */
int nc_delivery_num_ports(nc_delivery* d, uint32_t* n_ports);

/* One simulation step (asynchronous).  d_nodes[n_new]: nodes that emit a spike in this step; d_mult[n_new]: their
 * multiplicities (NULL = 1 each; 0 = no spike).  d_input[n_ports * n_nodes] (fp32; the input of receptor port p of
 * node t is entry p * n_nodes + t) is ACCUMULATED into with atomic adds, so
 * the caller zeroes it when a neuron model has consumed it.  A node id >= n_nodes or a full buffer drops the spike
 * and is reported by nc_delivery_counts (never silently). */
int nc_delivery_step(nc_delivery* d, const uint32_t* d_nodes, const uint32_t* d_mult, uint32_t n_new, float* d_input);

/* n_steps consecutive steps over a raster that is known beforehand (asynchronous): step k emits the spikes
 * d_nodes[offsets[k] .. offsets[k+1]) (d_mult likewise, or NULL); offsets is a HOST array of n_steps + 1 entries.
 * The same as n_steps calls of nc_delivery_step, without returning to the caller in between; d_input accumulates
 * over all of them. */
int nc_delivery_run(nc_delivery* d, uint32_t n_steps, const uint32_t* d_nodes, const uint32_t* d_mult,
                    const uint64_t* offsets, float* d_input);

/* The spike array of the last step, in no particular order (synchronises): global group index and multiplicity of
 * each entry; *n = number of entries, of which min(*n, cap) are copied. */
int nc_delivery_read_spike_array(nc_delivery* d, uint32_t* group, uint32_t* mult, uint32_t cap, uint32_t* n);

/* buffered = spikes waiting in the buffers; events = connections delivered since creation; dropped = spikes lost to
 * a full buffer; bad_nodes = spikes with a node id outside the network (synchronises).  Any pointer may be NULL. */
int nc_delivery_counts(nc_delivery* d, uint64_t* buffered, uint64_t* events, uint64_t* dropped, uint64_t* bad_nodes);

#ifdef __cplusplus
}
#endif
#endif /* NC_DELIVERY_H_ */
