// nc_internal.h -- what the other translation units of libnc may ask of a context (not part of the C ABI).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>
#include "../../include/nc.h"

struct nc_organised_view {  // borrowed device pointers, valid until nc_destroy
  const uint32_t* target;       // flat organised arrays; NULL when the organised connections live in the storage blocks
  const float* weight;
  // COPASS organisation (NC_FLAG_ORGANISE_COPASS): organised position j is entry j % block_size of block j / block_size
  const uint64_t* block_table;  // device array of block base addresses, NULL for the flat arrays
  uint64_t block_size, off_target, off_weight;
  const uint32_t* group_ptr;    // [n_nodes + 1]
  const uint32_t* group_start;  // [total_groups]
  const uint16_t* group_delay;  // [total_groups]
  const uint8_t* port;          // receptor port of every organised connection, NULL when every port is 0
  uint32_t n_ports;             // 1 + the largest port in use
  uint32_t n_nodes, total_groups;
  uint64_t n;
  cudaStream_t stream;
};
int nc_internal_organised_view(nc_context* c, nc_organised_view* out);  // NC_ERR_STATE before nc_finalize
void* nc_internal_alloc(nc_context* c, size_t bytes);
void nc_internal_free(nc_context* c, void* p);
int nc_internal_fail(nc_context* c, int code, const char* msg);
void nc_internal_attach(nc_context* c, int delta);  // a delivery object was created on (+1) / destroyed from (-1) this context
