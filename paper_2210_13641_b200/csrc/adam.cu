// adam.cu — S13 of DESIGN.md "Algorithm": Adam with bias correction (the paper names no
// optimiser, PAPER.md:133 only says L_M is minimised; reading R16).  Tables: only the entries
// of the structural touched set U are updated when sparse_table_adam = 1 — untouched entries
// keep theta, m, v bit-unchanged.  The gradient words are reset to "untouched" in the same pass,
// so the next step's scatter starts clean without a separate memset.
#include "nsm_internal.cuh"
#include "table_ops.cuh"

namespace {

using namespace tableops;

// One block per chunk of ADAM_CHUNK_FLOATS / F consecutive entries, two phases.
//  1. The chunk's gradient words are read densely (coalesced 16-byte loads, four independent ones
//     per thread; the array is L2-hot, the scatter has just written it).  Entries whose first word
//     is not -0.0f (FieldParams: "referenced this step") are compacted into shared memory
//     (index + gradient), warp-aggregated.
//  2. The block walks the compact list: every thread has a touched entry, loads its theta (compact
//     array) and its moment record (m | v; 16 bytes for F = 2; two entries in flight per thread),
//     updates and stores them.  The 16-byte gradient words that held a touched entry are then reset to
//     -0.0f, so the next step's scatter starts from "untouched" without a separate pass.
// sparse = 0 (dense Adam, textbook): every entry goes through phase 2.
template <int F>
__global__ void __launch_bounds__(ADAM_THREADS) adam_table_kernel(float *__restrict__ theta, float *__restrict__ mv, float *__restrict__ grad,
                                                                  uint64_t first_entry, uint64_t n_entries, int sparse, AdamConst c,
                                                                  unsigned long long *tl, int theta_resident, int reverse) {
  constexpr int CH = ADAM_CHUNK_FLOATS / F;
  __shared__ float list_g[ADAM_CHUNK_FLOATS];          // compacted gradients, F floats per touched entry
  __shared__ uint16_t list_e[CH];                      // compacted local entry indices
  __shared__ uint32_t cnt;
  pdl_wait();
  pdl_trigger();
  tl_mark(tl, K_ADAM_TABLE, 0);
  // reverse (tables beyond the L2): chunks from the END of the arrays to their start.  The scatter in front of this
  // kernel walks the levels upwards there, so the gradient lines it wrote last -- the finest levels' -- are the ones
  // still (dirty) in the L2, and the coarse levels this kernel then ends with are what the next encoder starts with
  // (config 4: adam_table 509 -> 494 us, encode 146 -> 142 us).  With tables inside the L2 it costs (config 2: +2.3 us).
  // In that order the theta stores also take the default policy instead of evict_first (486 us; the moment records'
  // stores stay evict_first: 494 us with both default).
  const uint32_t chunk = reverse ? gridDim.x - 1 - blockIdx.x : blockIdx.x;
  adam_chunk<F>(theta, mv, grad, first_entry + (uint64_t)chunk * CH, n_entries, sparse, c, list_g, list_e, &cnt, theta_resident || reverse);
  tl_mark(tl, K_ADAM_TABLE, 1);
}

__global__ void adam_dense_kernel(float *__restrict__ theta, float *__restrict__ m, float *__restrict__ v,
                                  float *__restrict__ grad, uint64_t n, AdamConst c) {
  pdl_wait();
  pdl_trigger();
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
    float th = theta[i], mm = m[i], vv = v[i];
    adam_one(th, mm, vv, grad[i], c);
    theta[i] = th; m[i] = mm; v[i] = vv; grad[i] = 0.f;
  }
}

}  // namespace

int launch_adam_table(const FieldParams &fp, uint32_t F, int sparse, float lr, float beta1, float beta2, float eps,
                      float inv_bc1, float inv_bc2, cudaStream_t st, unsigned long long *tl, uint64_t max_samples) {
  AdamConst c{lr, beta1, beta2, eps, inv_bc1, inv_bc2};
  const uint64_t chunk = ADAM_CHUNK_FLOATS / F, first_entry = 0, end_entry = fp.n_entries;
  dim3 grid((unsigned)((end_entry - first_entry + chunk - 1) / chunk)), block(ADAM_THREADS);
  // the panel encoder's case (launch_encode): tables that fit the L2 and a large step, whose encoder re-reads every table
  // line many times -- the updated theta then stays in the L2 for it (config 3: encode 128.7 -> 119.7 us against +3 us
  // here); with small steps (config 2) the same costs 2.7 us per step, so it is tied to the step's size
  const int theta_resident = fp.n_entries * F * sizeof(float) <= (96ull << 20) && max_samples >= (1ull << 20);
  const int reverse = fp.n_entries * F * sizeof(float) > (96ull << 20);   // the bound launch_scatter prefetches beyond
  switch (F) {
    case 1: launch_pdl(adam_table_kernel<1>, grid, block, 0, st, fp.theta, fp.mv, fp.grad, first_entry, end_entry, sparse, c, tl, theta_resident, reverse); break;
    case 2: launch_pdl(adam_table_kernel<2>, grid, block, 0, st, fp.theta, fp.mv, fp.grad, first_entry, end_entry, sparse, c, tl, theta_resident, reverse); break;
    case 4: launch_pdl(adam_table_kernel<4>, grid, block, 0, st, fp.theta, fp.mv, fp.grad, first_entry, end_entry, sparse, c, tl, theta_resident, reverse); break;
    default: launch_pdl(adam_table_kernel<8>, grid, block, 0, st, fp.theta, fp.mv, fp.grad, first_entry, end_entry, sparse, c, tl, theta_resident, reverse); break;
  }
  return 1;
}

int launch_adam_mlp(const FieldParams &fp, float lr, float beta1, float beta2, float eps, float inv_bc1, float inv_bc2,
                    cudaStream_t st) {
  AdamConst c{lr, beta1, beta2, eps, inv_bc1, inv_bc2};
  launch_pdl(adam_dense_kernel, dim3((unsigned)((fp.n_mlp + 255) / 256)), dim3(256), 0, st, fp.mlp_theta, fp.mlp_m, fp.mlp_v, fp.mlp_grad,
             fp.n_mlp, c);
  return 1;
}
