// comparators.cu -- TEST-ONLY device-side comparators (SURVEY 8(c) "what pins each part"): library routines that the
// product never links, used by tests/test_gpu_comparators.py to check the CUDA path against something other than
// the oracle:
//   * cuRAND's own Philox4x32-10 round function (curand_philox4x32_x.h) for the device Philox of the library;
//   * cub::DeviceRadixSort::SortPairs -- the sort underneath the paper's COPASS block-sort --
//     for the permutation nc_finalize produces, and as a context timing on the same keys.
// Built by the test with nvcc into tests/cuda/libcmp.so (git-ignored).  Nothing under paper_2306_09855_b200/ includes
// or loads this file.
#include <cub/device/device_radix_sort.cuh>
#include <cuda_runtime.h>
#include <curand_philox4x32_x.h>
#include <stdint.h>

namespace {

__global__ void curand_philox_kernel(uint32_t n, const uint4* ctr, const uint2* key, uint4* out) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = curand_Philox4x32_10(ctr[i], key[i]);
}

__global__ void iota_kernel(uint32_t* v, uint32_t n) {
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) v[i] = i;
}

}  // namespace

extern "C" {

// out[4 i ..] = curand_Philox4x32_10(ctr[4 i ..], key[2 i ..]); host arrays.  Returns 0 or a cudaError_t.
int cmp_curand_philox(uint32_t n, const uint32_t* ctr, const uint32_t* key, uint32_t* out) {
  uint4 *d_ctr = nullptr, *d_out = nullptr;
  uint2* d_key = nullptr;
  cudaError_t e;
  if ((e = cudaMalloc(&d_ctr, (size_t)n * 16)) || (e = cudaMalloc(&d_out, (size_t)n * 16)) ||
      (e = cudaMalloc(&d_key, (size_t)n * 8)))
    return (int)e;
  cudaMemcpy(d_ctr, ctr, (size_t)n * 16, cudaMemcpyHostToDevice);
  cudaMemcpy(d_key, key, (size_t)n * 8, cudaMemcpyHostToDevice);
  curand_philox_kernel<<<(n + 255) / 256, 256>>>(n, d_ctr, d_key, d_out);
  e = cudaMemcpy(out, d_out, (size_t)n * 16, cudaMemcpyDeviceToHost);
  cudaFree(d_ctr);
  cudaFree(d_key);
  cudaFree(d_out);
  return (int)e;
}

// Stable sort of (keys[i], i) by bits [begin_bit, end_bit) of the key: d_keys (device, n entries, left untouched),
// d_perm_out (device, n entries).  *ms = device time of the second of two identical SortPairs calls (the first warms
// up); *temp_bytes = CUB's temporary storage.  Returns 0 or a cudaError_t.
int cmp_cub_sort_pairs(uint32_t n, const uint32_t* d_keys, uint32_t* d_perm_out, int begin_bit, int end_bit, float* ms,
                       uint64_t* temp_bytes) {
  uint32_t *d_keys_out = nullptr, *d_iota = nullptr;
  void* d_temp = nullptr;
  size_t bytes = 0;
  cudaError_t e;
  if ((e = cudaMalloc(&d_keys_out, (size_t)n * 4)) || (e = cudaMalloc(&d_iota, (size_t)n * 4))) return (int)e;
  iota_kernel<<<1024, 256>>>(d_iota, n);
  cub::DeviceRadixSort::SortPairs(nullptr, bytes, d_keys, d_keys_out, d_iota, d_perm_out, (int)n, begin_bit, end_bit);
  if ((e = cudaMalloc(&d_temp, bytes))) return (int)e;
  cudaEvent_t a, b;
  cudaEventCreate(&a);
  cudaEventCreate(&b);
  for (int rep = 0; rep < 2; ++rep) {
    cudaEventRecord(a);
    cub::DeviceRadixSort::SortPairs(d_temp, bytes, d_keys, d_keys_out, d_iota, d_perm_out, (int)n, begin_bit, end_bit);
    cudaEventRecord(b);
  }
  e = cudaEventSynchronize(b);
  if (ms) cudaEventElapsedTime(ms, a, b);
  if (temp_bytes) *temp_bytes = bytes;
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  cudaFree(d_temp);
  cudaFree(d_keys_out);
  cudaFree(d_iota);
  return (int)e;
}

}  // extern "C"
