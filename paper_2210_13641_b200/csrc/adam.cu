// adam.cu — S13 of DESIGN.md "Algorithm": Adam with bias correction (the paper names no
// optimiser, PAPER.md:133 only says L_M is minimised; reading R16).  Tables: only the entries
// of the structural touched set U are updated when sparse_table_adam = 1 — untouched entries
// keep theta, m, v bit-unchanged.  The gradients of the touched entries are zeroed and the touched bits
// cleared in the same pass, so the next step's scatter starts clean without a separate memset.
#include "nsm_internal.cuh"
#include "table_ops.cuh"

namespace {

using namespace tableops;

// One block per ADAM_ENTRIES consecutive table entries (body: tableops::adam_block).  The touched set arrives as a bitmap
// written by the scatter; the block walks its 512 bytes of it and then touches only what the touched entries need: their
// gradient, their theta, their moment record.  Nothing is scanned densely (round 1's kernel read all of the gradient
// array to find the touched 25 %: 48.8 MB at config 2, 719 MB at config 4).
template <int F>
__global__ void __launch_bounds__(ADAM_THREADS) adam_table_kernel(float *__restrict__ theta, float *__restrict__ mv, float *__restrict__ grad,
                                                                  uint32_t *__restrict__ touched, uint64_t n_entries, int sparse,
                                                                  AdamConst c, unsigned long long *tl) {
  __shared__ uint16_t list_e[ADAM_ENTRIES];            // local indices of the block's touched entries, ascending
  __shared__ uint32_t warp_tot[ADAM_WORDS / 32];
  pdl_wait();
  pdl_trigger();
  tl_mark(tl, K_ADAM_TABLE, 0);
  adam_block<F>(theta, mv, grad, touched, (uint64_t)blockIdx.x * ADAM_ENTRIES, n_entries, sparse, c, list_e, warp_tot);
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
                      float inv_bc1, float inv_bc2, cudaStream_t st, unsigned long long *tl) {
  AdamConst c{lr, beta1, beta2, eps, inv_bc1, inv_bc2};
  dim3 grid((unsigned)((fp.n_entries + ADAM_ENTRIES - 1) / ADAM_ENTRIES)), block(ADAM_THREADS);
  switch (F) {
    case 1: launch_pdl(adam_table_kernel<1>, grid, block, 0, st, fp.theta, fp.mv, fp.grad, fp.touched, fp.n_entries, sparse, c, tl); break;
    case 2: launch_pdl(adam_table_kernel<2>, grid, block, 0, st, fp.theta, fp.mv, fp.grad, fp.touched, fp.n_entries, sparse, c, tl); break;
    case 4: launch_pdl(adam_table_kernel<4>, grid, block, 0, st, fp.theta, fp.mv, fp.grad, fp.touched, fp.n_entries, sparse, c, tl); break;
    default: launch_pdl(adam_table_kernel<8>, grid, block, 0, st, fp.theta, fp.mv, fp.grad, fp.touched, fp.n_entries, sparse, c, tl); break;
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
