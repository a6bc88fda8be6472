// l2_probe.cu -- yardsticks for bench.py, NOT part of libbits_b200: the two L2 figures SURVEY.md 8(d)
// asks for as denominators of the search kernels (MEASURED_PEAKS.json has none):
//   (i)  streaming read bandwidth over a buffer that fits the 126 MB L2 (default 48 MB),
//   (ii) random 32-byte-sector gather throughput over an L2-resident buffer (default 80 MB).
// Plain C ABI, device pointers owned by the caller, timing by CUDA events on the given stream.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__global__ void __launch_bounds__(256) stream_read_kernel(const uint4* __restrict__ p, uint64_t n16, uint32_t* sink) {
  uint32_t acc = 0;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (uint64_t)gridDim.x * blockDim.x) {
    const uint4 v = __ldcg(p + i);           // L2 only: every request goes to the L2
    acc ^= v.x ^ v.y ^ v.z ^ v.w;
  }
  if (acc == 0x12345678u) *sink = acc;       // keeps the loads alive
}

// Every thread touches `per_thread` pseudo-random 32-byte sectors, one 16-byte load per sector, eight
// independent loads in flight.
__global__ void __launch_bounds__(256) gather_sector_kernel(const uint4* __restrict__ p, uint64_t n_sectors, uint32_t per_thread,
                                                            uint32_t* sink) {
  uint32_t s = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u, acc = 0;
  for (uint32_t k = 0; k < per_thread; k += 8) {
    uint64_t idx[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      s = s * 1664525u + 1013904223u;
      idx[j] = ((uint64_t)s * n_sectors) >> 32;
    }
    uint4 v[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) v[j] = __ldcg(p + 2 * idx[j]);
#pragma unroll
    for (int j = 0; j < 8; ++j) acc ^= v[j].x;
  }
  if (acc == 0x12345678u) *sink = acc;
}

float time_launches(cudaStream_t st, int reps, void (*launch)(cudaStream_t, void*), void* arg) {
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  for (int i = 0; i < 3; ++i) launch(st, arg);
  float best = 1e30f;
  for (int i = 0; i < reps; ++i) {
    cudaEventRecord(e0, st); launch(st, arg); cudaEventRecord(e1, st);
    cudaEventSynchronize(e1);
    float ms = 0.f; cudaEventElapsedTime(&ms, e0, e1);
    best = ms < best ? ms : best;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return best;
}

struct Arg { const uint4* p; uint64_t n; uint32_t per_thread; uint32_t* sink; };
void launch_stream(cudaStream_t st, void* a) { Arg* x = (Arg*)a; stream_read_kernel<<<148 * 16, 256, 0, st>>>(x->p, x->n, x->sink); }
void launch_gather(cudaStream_t st, void* a) { Arg* x = (Arg*)a; gather_sector_kernel<<<148 * 32, 256, 0, st>>>(x->p, x->n, x->per_thread, x->sink); }

}  // namespace

extern "C" {

// GB/s of a streaming read of `bytes` (multiple of 16) from buf, best of `reps` (buffer warmed into L2 first).
double l2_probe_stream_gbs(const void* buf, uint64_t bytes, uint32_t* sink, int reps, void* stream) {
  Arg a{(const uint4*)buf, bytes / 16, 0, sink};
  const float ms = time_launches((cudaStream_t)stream, reps, launch_stream, &a);
  return cudaGetLastError() == cudaSuccess ? (double)bytes / (ms * 1e-3) / 1e9 : -1.0;
}

// 1e9 sectors/s of random 32-byte sector reads over `bytes` of buf, best of `reps`.
double l2_probe_gather_gsectors(const void* buf, uint64_t bytes, uint32_t* sink, int reps, void* stream) {
  Arg a{(const uint4*)buf, bytes / 32, 64, sink};
  const float ms = time_launches((cudaStream_t)stream, reps, launch_gather, &a);
  const double sectors = 148.0 * 32 * 256 * 64;
  return cudaGetLastError() == cudaSuccess ? sectors / (ms * 1e-3) / 1e9 : -1.0;
}

}  // extern "C"
