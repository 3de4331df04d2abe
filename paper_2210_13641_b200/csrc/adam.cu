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

// One thread per B consecutive entries: their flag bytes come in one coalesced load; the records
// of the touched ones (4F floats each; one 32 B sector for F = 2) are ALL requested before any is
// used, so a thread keeps up to B record loads in flight (the kernel is latency-, not
// bandwidth-limited at 25 % touched).
template <int F>
__global__ void __launch_bounds__(256) adam_table_kernel(float *__restrict__ rec, uint8_t *__restrict__ touched,
                                                         uint64_t n_entries, int sparse, AdamConst c) {
  constexpr int B = (F <= 2) ? 8 : 4;
  const uint64_t n_groups = (n_entries + B - 1) / B;
  for (uint64_t q = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; q < n_groups; q += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t e0 = q * B;
    uint64_t flags = 0;
    if (e0 + B <= n_entries) {
      if (B == 8) flags = *reinterpret_cast<const uint64_t *>(touched + e0);
      else flags = *reinterpret_cast<const uint32_t *>(touched + e0);
    } else {
      for (uint64_t e = e0; e < n_entries; ++e) flags |= (uint64_t)touched[e] << (8 * (e - e0));
    }
    if (sparse && flags == 0) continue;
    float4 x[B][F];
    bool act[B];
#pragma unroll
    for (int j = 0; j < B; ++j) {
      act[j] = (e0 + j < n_entries) && (!sparse || ((flags >> (8 * j)) & 0xffu));
      if (act[j]) {
        const float4 *r4 = reinterpret_cast<const float4 *>(rec + (e0 + j) * 4 * F);
#pragma unroll
        for (int i = 0; i < F; ++i) x[j][i] = r4[i];
      }
    }
#pragma unroll
    for (int j = 0; j < B; ++j) {
      if (!act[j]) continue;
      float vals[4 * F];
#pragma unroll
      for (int i = 0; i < F; ++i) {
        vals[4 * i] = x[j][i].x; vals[4 * i + 1] = x[j][i].y; vals[4 * i + 2] = x[j][i].z; vals[4 * i + 3] = x[j][i].w;
      }
#pragma unroll
      for (int f = 0; f < F; ++f) {
        adam_one(vals[f], vals[2 * F + f], vals[3 * F + f], vals[F + f], c);
        vals[F + f] = 0.f;   // the gradient is consumed
      }
      float4 *r4 = reinterpret_cast<float4 *>(rec + (e0 + j) * 4 * F);
#pragma unroll
      for (int i = 0; i < F; ++i) r4[i] = make_float4(vals[4 * i], vals[4 * i + 1], vals[4 * i + 2], vals[4 * i + 3]);
    }
    if (flags) {
      if (e0 + B <= n_entries) {
        if (B == 8) *reinterpret_cast<uint64_t *>(touched + e0) = 0ull;
        else *reinterpret_cast<uint32_t *>(touched + e0) = 0u;
      } else {
        for (uint64_t e = e0; e < n_entries; ++e) touched[e] = 0;
      }
    }
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
    case 1: adam_table_kernel<1><<<grid, block, 0, st>>>(fp.rec, fp.touched, fp.n_entries, sparse, c); break;
    case 2: adam_table_kernel<2><<<grid, block, 0, st>>>(fp.rec, fp.touched, fp.n_entries, sparse, c); break;
    case 4: adam_table_kernel<4><<<grid, block, 0, st>>>(fp.rec, fp.touched, fp.n_entries, sparse, c); break;
    default: adam_table_kernel<8><<<grid, block, 0, st>>>(fp.rec, fp.touched, fp.n_entries, sparse, c); break;
  }
  return 1;
}

int launch_adam_mlp(const FieldParams &fp, float lr, float beta1, float beta2, float eps, float inv_bc1, float inv_bc2,
                    cudaStream_t st) {
  AdamConst c{lr, beta1, beta2, eps, inv_bc1, inv_bc2};
  adam_dense_kernel<<<(unsigned)((fp.n_mlp + 255) / 256), 256, 0, st>>>(fp.mlp_theta, fp.mlp_m, fp.mlp_v, fp.mlp_grad, fp.n_mlp, c);
  return 1;
}
