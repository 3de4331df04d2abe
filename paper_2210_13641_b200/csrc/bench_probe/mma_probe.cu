// mma_probe.cu — bench-only micro-benchmark (part of libnsm_bench_probe.so, NOT of libnsm.so or include/nsm.h): what a
// stream of the small tcgen05.mma instructions the MLP kernels consist of costs on this GPU.  One CTA, an elected lane
// issues n MMAs (cta_group::1, kind::f16, M = 128, K = 16, the given N) on zeroed shared-memory operands and one commit;
// cycles from the first issue to the mbarrier flip (clock64, SM clock), best of 4.  The MLPs of this path are bound by
// this dispatch rate and by the fixed issue-to-completion latency, not by tensor math (profiles/r2d): bench.py quotes
// mlp_fwd / mlp_bwd against the floor it implies.
#include <cuda_runtime.h>
#include <stdint.h>

#include "../tc_common.cuh"

namespace {

using namespace tc;

__global__ void __launch_bounds__(128) mma_chain_kernel(uint32_t N, uint32_t n_mma, long long *out) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t sbase = smem_u32(smem);
  const uint32_t bar = sbase + 65536, tslot = sbase + 65544;
  for (uint32_t i = threadIdx.x; i < 65536 / 16; i += 128) reinterpret_cast<uint4 *>(smem)[i] = make_uint4(0, 0, 0, 0);
  if (threadIdx.x == 0) { mbar_init(bar, 1); fence_async_smem(); }
  if (threadIdx.x < 32) tmem_alloc<256>(tslot);
  fence_async_smem(); fence_before(); __syncthreads(); fence_after();
  const uint32_t tm = *reinterpret_cast<volatile uint32_t *>(smem + 65544);
  const uint32_t idesc = make_idesc(0, 128, N, 0, 0);
  uint32_t ph = 0;
  long long best = 1ll << 62;
  for (int rep = 0; rep < 4; ++rep) {
    __syncthreads();
    const long long t0 = clock64();
    if (threadIdx.x < 32 && elect_one()) {
      const uint64_t da = make_desc(sbase, 128 * 16, 128), db = make_desc(sbase + 32768, N * 16, 128);
      for (uint32_t i = 0; i < n_mma; ++i) mma_ss(tm, da, db, idesc, 1);
      mma_commit(bar);
    }
    mbar_wait(bar, ph); ph ^= 1;
    const long long t = clock64() - t0;
    if (t < best) best = t;
  }
  if (threadIdx.x == 0) *out = best;
  __syncthreads();
  if (threadIdx.x < 32) tmem_free<256>(tm);
}

}  // namespace

// cycles (SM clock) from the first issue to completion of n_mma MMAs of width N (16 <= N <= 256, a multiple of 16).
// returns 0 on success, 1 bad argument, 3 CUDA error
extern "C" int nsm_bench_probe_mma(uint32_t N, uint32_t n_mma, long long *cycles_out) {
  if (!cycles_out || N < 16 || N > 256 || (N & 15u) || n_mma == 0) return 1;
  long long *d = nullptr;
  if (cudaMalloc(&d, sizeof(long long)) != cudaSuccess) { cudaGetLastError(); return 3; }
  cudaFuncSetAttribute(mma_chain_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 66048);
  mma_chain_kernel<<<1, 128, 66048>>>(N, n_mma, d);
  const cudaError_t e = cudaMemcpy(cycles_out, d, sizeof(long long), cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess || cudaGetLastError() != cudaSuccess) return 3;
  return 0;
}
