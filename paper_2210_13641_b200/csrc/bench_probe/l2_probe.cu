// l2_probe.cu — bench-only micro-benchmark (NOT part of libnsm.so or of include/nsm.h): built as its own shared object,
// libnsm_bench_probe.so, and loaded by bench.py alone.  It measures, inside the bench run, the peak the encoder (S4) and
// the scatter (S12) are quoted against while the tables fit the L2 ("measure L2 bandwidth and
// atomic throughput yourself; MEASURED_PEAKS.json has HBM and bf16 only"): random 8-byte gathers and random
// red.global.add.v2.f32 over a table of a given size -- those kernels' access pattern with every locality removed.
// One launch is timed with CUDA events after warm-up launches; best of 8.
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__device__ __forceinline__ uint32_t pmix(uint32_t x) {
  x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
  return x;
}

// each thread: 8 independent accesses to random 8-byte entries
__global__ void probe_gather_kernel(const float2 *__restrict__ tab, uint32_t n_entries, uint32_t seed, uint64_t n_threads,
                                    float *__restrict__ sink) {
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_threads) return;
  const uint32_t h = pmix(seed ^ (uint32_t)i);
  float acc = 0.f;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const float2 v = __ldg(tab + pmix(h + k * 0x9e3779b9u) % n_entries);
    acc += v.x + v.y;
  }
  if (acc == 123.456f) *sink = acc;
}

__global__ void probe_red_kernel(float2 *__restrict__ tab, uint32_t n_entries, uint32_t seed, uint64_t n_threads) {
  const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_threads) return;
  const uint32_t h = pmix(seed ^ (uint32_t)i);
#pragma unroll
  for (int k = 0; k < 8; ++k) atomicAdd(tab + pmix(h + k * 0x9e3779b9u) % n_entries, make_float2(1.f, 2.f));
}

}  // namespace

// returns 0 on success, 1 bad argument, 2 out of memory, 3 CUDA error; *seconds_out = duration of one launch
extern "C" int nsm_bench_probe_l2(uint64_t table_bytes, uint64_t n_accesses, int reductions, double *seconds_out) {
  if (!seconds_out || table_bytes < 64 || n_accesses < 8) return 1;
  float2 *tab = nullptr;
  float *sink = nullptr;
  if (cudaMalloc(&tab, table_bytes) != cudaSuccess || cudaMalloc(&sink, 4) != cudaSuccess) {
    cudaGetLastError();
    cudaFree(tab);
    return 2;
  }
  cudaMemset(tab, 0, table_bytes);
  const uint32_t n_entries = (uint32_t)(table_bytes / 8);
  const uint64_t n_threads = n_accesses / 8;
  const unsigned grid = (unsigned)((n_threads + 255) / 256);
  cudaEvent_t a, b;
  cudaEventCreate(&a);
  cudaEventCreate(&b);
  float best = 1e30f;
  for (int rep = 0; rep < 12; ++rep) {   // 4 warm-up launches bring the table into the L2 if it fits
    cudaEventRecord(a);
    if (reductions) probe_red_kernel<<<grid, 256>>>(tab, n_entries, 7919u * rep + 1u, n_threads);
    else probe_gather_kernel<<<grid, 256>>>(tab, n_entries, 7919u * rep + 1u, n_threads, sink);
    cudaEventRecord(b);
    cudaEventSynchronize(b);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    if (rep >= 4 && ms < best) best = ms;
  }
  cudaEventDestroy(a);
  cudaEventDestroy(b);
  cudaFree(tab);
  cudaFree(sink);
  if (cudaGetLastError() != cudaSuccess) return 3;
  *seconds_out = (double)best * 1e-3;
  return 0;
}
