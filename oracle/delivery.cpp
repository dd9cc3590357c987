// delivery.cpp -- see delivery.h.  Plain loops in the paper's order; test infrastructure only.
#include "delivery.h"

#include <algorithm>
#include <deque>
#include <vector>

namespace {
struct Spike {
  uint32_t time_idx, group_idx, mult;
};
}  // namespace

struct oc_delivery {
  oc_connections_view conn;  // sorted view
  oc_index_view idx;
  std::vector<std::deque<Spike>> queue;  // one per node
  std::vector<uint32_t> arr_group, arr_mult;
  std::vector<uint8_t> port;  // receptor port of every organised connection
  uint32_t n_ports = 1;
  uint64_t events = 0;
};

extern "C" {

int oc_delivery_create(oc_context* ctx, oc_delivery** out) {
  if (!ctx || !out) return -1;
  oc_delivery* d = new oc_delivery();
  int rc = oc_get_connections(ctx, 1, &d->conn);
  if (rc == 0) rc = oc_get_index(ctx, &d->idx);
  if (rc != 0) {
    delete d;
    return rc;
  }
  d->queue.resize(d->idx.n_nodes);
  d->port.resize(d->conn.n);
  if (d->conn.n && oc_read_connection_attributes(ctx, 1, 0, d->conn.n, d->port.data(), nullptr) != 0) {
    delete d;
    return -1;
  }
  for (uint8_t p : d->port) d->n_ports = std::max<uint32_t>(d->n_ports, (uint32_t)p + 1u);
  *out = d;
  return 0;
}

int oc_delivery_destroy(oc_delivery* d) {
  delete d;
  return 0;
}

int oc_delivery_step(oc_delivery* d, const uint32_t* nodes, const uint32_t* mult, uint32_t n_new, double* input) {
  if (!d || !input || (n_new && !nodes)) return -1;
  for (uint32_t k = 0; k < n_new; ++k)
    if (nodes[k] >= d->idx.n_nodes) return -1;
  d->arr_group.clear();
  d->arr_mult.clear();
  // time indexes grow by one; matured spikes go to the spike array and point at their next group
  for (uint32_t s = 0; s < d->idx.n_nodes; ++s) {
    std::deque<Spike>& q = d->queue[s];
    const uint32_t G = d->idx.group_count[s], p = d->idx.group_ptr[s];
    for (Spike& sp : q) {
      sp.time_idx += 1;
      if (sp.group_idx < G && d->idx.group_delay[p + sp.group_idx] == sp.time_idx) {
        d->arr_group.push_back(p + sp.group_idx);
        d->arr_mult.push_back(sp.mult);
        sp.group_idx += 1;
      }
    }
    while (!q.empty() && q.front().group_idx >= G) q.pop_front();  // spikes leave in arrival order
  }
  // every connection of every group in the spike array
  for (size_t e = 0; e < d->arr_group.size(); ++e) {
    const uint32_t g = d->arr_group[e];
    const uint64_t c0 = d->idx.group_start[g];
    const uint64_t c1 = g + 1 < d->idx.total_groups ? d->idx.group_start[g + 1] : d->conn.n;
    for (uint64_t c = c0; c < c1; ++c)  // reading F2: one input per (receptor port, node), port-major
      input[(uint64_t)d->port[c] * d->idx.n_nodes + d->conn.target[c]] += (double)d->conn.weight[c] * (double)d->arr_mult[e];
    d->events += c1 - c0;
  }
  // the spikes emitted in this step (a node without outgoing connections buffers nothing)
  for (uint32_t k = 0; k < n_new; ++k) {
    const uint32_t m = mult ? mult[k] : 1u;
    if (m && d->idx.group_count[nodes[k]]) d->queue[nodes[k]].push_back(Spike{0u, 0u, m});
  }
  return 0;
}

int oc_delivery_spike_array(oc_delivery* d, const uint32_t** group, const uint32_t** mult, uint32_t* n) {
  if (!d || !group || !mult || !n) return -1;
  *group = d->arr_group.data();
  *mult = d->arr_mult.data();
  *n = (uint32_t)d->arr_group.size();
  return 0;
}

int oc_delivery_num_ports(oc_delivery* d, uint32_t* n_ports) {
  if (!d || !n_ports) return -1;
  *n_ports = d->n_ports;
  return 0;
}

int oc_delivery_counts(oc_delivery* d, uint64_t* buffered, uint64_t* events) {
  if (!d) return -1;
  uint64_t b = 0;
  for (auto& q : d->queue) b += q.size();
  if (buffered) *buffered = b;
  if (events) *events = d->events;
  return 0;
}

}  // extern "C"
