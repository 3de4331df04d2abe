// adam.cu — S13 of DESIGN.md "Algorithm": Adam with bias correction (the paper names no
// optimiser, PAPER.md:133 only says L_M is minimised; reading R16).  Tables: only the entries
// of the structural touched set U are updated when sparse_table_adam = 1 — untouched entries
// keep theta, m, v bit-unchanged.  The gradient and the touched flag are cleared in the same
// pass, so the next step's scatter starts from zero without a separate memset.
#include "nsm_internal.cuh"

namespace {

struct AdamConst {
  float lr, b1, b2, eps, inv_bc1, inv_bc2;
};

__device__ __forceinline__ void adam_one(float &th, float &m, float &v, float g, const AdamConst &c) {
  m = c.b1 * m + (1.f - c.b1) * g;
  v = c.b2 * v + (1.f - c.b2) * g * g;
  float mhat = m * c.inv_bc1, vhat = v * c.inv_bc2;
  th = th - c.lr * mhat / (sqrtf(vhat) + c.eps);
}

template <int F>
__global__ void __launch_bounds__(256) adam_table_kernel(float *__restrict__ theta, float *__restrict__ m,
                                                         float *__restrict__ v, float *__restrict__ grad,
                                                         uint8_t *__restrict__ touched, uint64_t n_entries,
                                                         int sparse, AdamConst c) {
  for (uint64_t e = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_entries;
       e += (uint64_t)gridDim.x * blockDim.x) {
    const uint8_t t = touched[e];
    if (sparse && !t) continue;
    float th[F], mm[F], vv[F], gg[F];
#pragma unroll
    for (int f = 0; f < F; ++f) {
      th[f] = theta[e * F + f]; mm[f] = m[e * F + f]; vv[f] = v[e * F + f]; gg[f] = grad[e * F + f];
    }
#pragma unroll
    for (int f = 0; f < F; ++f) adam_one(th[f], mm[f], vv[f], gg[f], c);
#pragma unroll
    for (int f = 0; f < F; ++f) {
      theta[e * F + f] = th[f]; m[e * F + f] = mm[f]; v[e * F + f] = vv[f];
      if (t) grad[e * F + f] = 0.f;
    }
    if (t) touched[e] = 0;
  }
}

__global__ void adam_dense_kernel(float *__restrict__ theta, float *__restrict__ m, float *__restrict__ v,
                                  float *__restrict__ grad, uint64_t n, AdamConst c) {
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x) {
    float th = theta[i], mm = m[i], vv = v[i];
    adam_one(th, mm, vv, grad[i], c);
    theta[i] = th; m[i] = mm; v[i] = vv; grad[i] = 0.f;
  }
}

}  // namespace

int launch_adam_table(const FieldParams &fp, uint32_t F, int sparse, float lr, float beta1, float beta2, float eps,
                      float inv_bc1, float inv_bc2, int n_sms, cudaStream_t st) {
  AdamConst c{lr, beta1, beta2, eps, inv_bc1, inv_bc2};
  dim3 grid(n_sms * 8), block(256);
  switch (F) {
    case 1: adam_table_kernel<1><<<grid, block, 0, st>>>(fp.theta, fp.m, fp.v, fp.grad, fp.touched, fp.n_entries, sparse, c); break;
    case 2: adam_table_kernel<2><<<grid, block, 0, st>>>(fp.theta, fp.m, fp.v, fp.grad, fp.touched, fp.n_entries, sparse, c); break;
    case 4: adam_table_kernel<4><<<grid, block, 0, st>>>(fp.theta, fp.m, fp.v, fp.grad, fp.touched, fp.n_entries, sparse, c); break;
    default: adam_table_kernel<8><<<grid, block, 0, st>>>(fp.theta, fp.m, fp.v, fp.grad, fp.touched, fp.n_entries, sparse, c); break;
  }
  return 1;
}

int launch_adam_mlp(const FieldParams &fp, float lr, float beta1, float beta2, float eps, float inv_bc1, float inv_bc2,
                    cudaStream_t st) {
  AdamConst c{lr, beta1, beta2, eps, inv_bc1, inv_bc2};
  adam_dense_kernel<<<(unsigned)((fp.n_mlp + 255) / 256), 256, 0, st>>>(fp.theta + fp.n_table, fp.m + fp.n_table,
                                                                       fp.v + fp.n_table, fp.grad + fp.n_table,
                                                                       fp.n_mlp, c);
  return 1;
}
