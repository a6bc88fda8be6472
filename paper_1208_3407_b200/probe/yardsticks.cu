// yardsticks.cu -- library yardsticks for bench.py, NOT part of libbits_b200 and never linked into it
// (SURVEY.md section 8(d) "Yardsticks"): with no reference kernel to beat, these put the library's sort
// keys/s and searched intervals/s next to what the CUDA toolkit's own primitives reach on the same
// arrays on the same box:
//   (i)  cub::DeviceRadixSort::SortKeys on uint32 keys (the library radix sort the paper's BITS-CUDA
//        would call today);
//   (ii) thrust::upper_bound / thrust::lower_bound, vectorised over a query array, on sorted keys
//        (Algorithm 1's two BSEARCHes, as two library calls).
// Plain C ABI, device pointers owned by the caller, timing by CUDA events on the given stream.
#include <cuda_runtime.h>
#include <stdint.h>

#include <cub/device/device_radix_sort.cuh>
#include <thrust/binary_search.h>
#include <thrust/execution_policy.h>
#include <thrust/system/cuda/execution_policy.h>

extern "C" {

// Bytes of temporary storage cub needs to sort n uint32 keys.
size_t yard_cub_sort_temp_bytes(uint64_t n) {
  size_t bytes = 0;
  cub::DeviceRadixSort::SortKeys(nullptr, bytes, (const uint32_t*)nullptr, (uint32_t*)nullptr, (int64_t)n);
  return bytes;
}

// Sorts keys_in -> keys_out `reps` times (after two warm-ups); returns the best time of one sort in ms
// (negative on a CUDA error).  begin_bit .. end_bit as in cub (0, 32 = the whole key).
double yard_cub_sort_keys_ms(const uint32_t* keys_in, uint32_t* keys_out, uint64_t n, void* temp, size_t temp_bytes,
                             int begin_bit, int end_bit, int reps, void* stream) {
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -1.0;
  double best = 1e30;
  for (int i = 0; i < reps + 2; ++i) {
    cudaEventRecord(e0, st);
    if (cub::DeviceRadixSort::SortKeys(temp, temp_bytes, keys_in, keys_out, (int64_t)n, begin_bit, end_bit, st) != cudaSuccess) return -1.0;
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) return -1.0;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (i >= 2 && ms < best) best = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return best;
}

// first_out[i] = #{b_s <= q_end[i]} (upper bound), last_out[i] = #{b_e < q_start[i]} (lower bound): the two
// vectorised library searches of one counting call.  Returns the best time of the pair of calls in ms.
double yard_thrust_bounds_ms(const uint32_t* b_s, const uint32_t* b_e, uint64_t n_b, const uint32_t* q_end,
                             const uint32_t* q_start, uint64_t n_q, uint32_t* first_out, uint32_t* last_out, int reps,
                             void* stream) {
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -1.0;
  double best = 1e30;
  auto pol = thrust::cuda::par_nosync.on(st);
  for (int i = 0; i < reps + 2; ++i) {
    cudaEventRecord(e0, st);
    thrust::upper_bound(pol, b_s, b_s + n_b, q_end, q_end + n_q, first_out);
    thrust::lower_bound(pol, b_e, b_e + n_b, q_start, q_start + n_q, last_out);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) return -1.0;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (i >= 2 && ms < best) best = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return best;
}

}  // extern "C"
