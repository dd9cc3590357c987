/*
 * delivery.h -- CPU oracle of spike delivery over the built index (Sec. II.C).
 * TEST INFRASTRUCTURE, like oracle.h: plain single-threaded C++, fp64 accumulation, shares no code with the CUDA
 * path; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may use it.
 *
 * The paper's structure, followed literally: every node has a queue of outgoing spikes (time index, connection
 * group index, multiplicity).  A spike enters with both indexes zero.  Every step the time indexes of all buffered
 * spikes grow by one; a spike whose time index equals the delay of the connection group its group index points at
 * goes into the spike array as (source, group, multiplicity) and its group index moves to the next group (delays
 * ascend inside a source); after its last group it leaves the queue.  Then every connection of every
 * group in the spike array adds weight * multiplicity to the input of its target.
 *
 * Readings: F1 one step = advance, collect matured, deliver, THEN insert the spikes
 * emitted in this step (time index 0), so a spike emitted in step k reaches a connection of delay d in step k + d;
 * F2 the "input" of a node is one fp accumulator per (receptor port, node), summed here in fp64;
 * F3 the group index in the spike array is the global one, group_ptr[source] + local index (Eq. 14).
 */
#ifndef ORACLE_DELIVERY_H_
#define ORACLE_DELIVERY_H_
#include <stdint.h>
#include "oracle.h"
#ifdef __cplusplus
extern "C" {
#endif
typedef struct oc_delivery oc_delivery;
/* ctx must be finalized and outlive the delivery object */
int oc_delivery_create(oc_context* ctx, oc_delivery** out);
int oc_delivery_destroy(oc_delivery* d);
/* One step.  nodes/mult: the n_new spikes emitted in this step (mult NULL = 1 each).  input[n_ports * n_nodes] (fp64,
 * entry port * n_nodes + node; n_ports = 1 + the largest receptor port in use) is ACCUMULATED into.  Returns OC_OK or a negative oc status (node out of range). */
int oc_delivery_step(oc_delivery* d, const uint32_t* nodes, const uint32_t* mult, uint32_t n_new, double* input);
/* the spike array of the last step: global group index and multiplicity per entry, in queue order */
int oc_delivery_spike_array(oc_delivery* d, const uint32_t** group, const uint32_t** mult, uint32_t* n);
int oc_delivery_num_ports(oc_delivery* d, uint32_t* n_ports);
/* spikes still buffered, and connections delivered so far */
int oc_delivery_counts(oc_delivery* d, uint64_t* buffered, uint64_t* events);
#ifdef __cplusplus
}
#endif
#endif
