// adam.cu — S13 of DESIGN.md "Algorithm": Adam with bias correction (the paper names no
// optimiser, PAPER.md:133 only says L_M is minimised; reading R16).  Tables: only the entries
// of the structural touched set U are updated when sparse_table_adam = 1 — untouched entries
// keep theta, m, v bit-unchanged.  The gradient words are reset to "untouched" in the same pass,
// so the next step's scatter starts clean without a separate memset.
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

// One thread per B consecutive entries (B*F = 4 gradient floats = one coalesced 16-byte load, two
// for F = 8).  The gradient array is read densely (it is L2-hot: the scatter has just written it);
// only the records of touched entries (bits(g) != -0.0f, see FieldParams) are loaded, updated and
// stored, and their gradient words are reset to -0.0f, so the next step's scatter starts from
// "untouched" without a separate clearing pass.
template <int F>
__global__ void __launch_bounds__(256) adam_table_kernel(float *__restrict__ rec, float *__restrict__ grad,
                                                         uint64_t n_entries, int sparse, AdamConst c) {
  constexpr int B = F >= 4 ? 1 : 4 / F;
  constexpr int NV = B * F / 4;        // float4 loads of gradient per thread
  const uint64_t q = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const uint64_t e0 = q * B;
  if (e0 >= n_entries) return;
  float g[B * F];
  if (e0 + B <= n_entries) {
    const float4 *g4 = reinterpret_cast<const float4 *>(grad + e0 * F);
#pragma unroll
    for (int i = 0; i < NV; ++i) {
      const float4 t = g4[i];
      g[4 * i] = t.x; g[4 * i + 1] = t.y; g[4 * i + 2] = t.z; g[4 * i + 3] = t.w;
    }
  } else {
#pragma unroll
    for (int i = 0; i < B * F; ++i) g[i] = (e0 * F + i < n_entries * F) ? grad[e0 * F + i] : __uint_as_float(NSM_GRAD_UNTOUCHED);
  }
  bool act[B];
  float th[B][F], m[B][F], v[B][F];
#pragma unroll
  for (int j = 0; j < B; ++j) {
    act[j] = (e0 + j < n_entries) && (!sparse || __float_as_uint(g[j * F]) != NSM_GRAD_UNTOUCHED);
    if (act[j]) {
      const float *r = rec + (e0 + j) * 4 * F;
      if constexpr (F == 1) {
        const float4 t = *reinterpret_cast<const float4 *>(r);
        th[j][0] = t.x; m[j][0] = t.z; v[j][0] = t.w;
      } else if constexpr (F == 2) {
        const float4 a = *reinterpret_cast<const float4 *>(r), b = *reinterpret_cast<const float4 *>(r + 4);
        th[j][0] = a.x; th[j][1] = a.y; m[j][0] = b.x; m[j][1] = b.y; v[j][0] = b.z; v[j][1] = b.w;
      } else {
#pragma unroll
        for (int i = 0; i < F / 4; ++i) {
          const float4 a = *reinterpret_cast<const float4 *>(r + 4 * i), b = *reinterpret_cast<const float4 *>(r + 2 * F + 4 * i),
                       d = *reinterpret_cast<const float4 *>(r + 3 * F + 4 * i);
          th[j][4 * i] = a.x; th[j][4 * i + 1] = a.y; th[j][4 * i + 2] = a.z; th[j][4 * i + 3] = a.w;
          m[j][4 * i] = b.x; m[j][4 * i + 1] = b.y; m[j][4 * i + 2] = b.z; m[j][4 * i + 3] = b.w;
          v[j][4 * i] = d.x; v[j][4 * i + 1] = d.y; v[j][4 * i + 2] = d.z; v[j][4 * i + 3] = d.w;
        }
      }
    }
  }
  bool any = false;
#pragma unroll
  for (int j = 0; j < B; ++j) {
    if (!act[j]) continue;
    any = true;
#pragma unroll
    for (int f = 0; f < F; ++f) {
      adam_one(th[j][f], m[j][f], v[j][f], g[j * F + f], c);
      g[j * F + f] = __uint_as_float(NSM_GRAD_UNTOUCHED);   // the gradient is consumed
    }
    float *r = rec + (e0 + j) * 4 * F;
    if constexpr (F == 1) {
      r[0] = th[j][0];
      *reinterpret_cast<float2 *>(r + 2) = make_float2(m[j][0], v[j][0]);
    } else if constexpr (F == 2) {
      *reinterpret_cast<float2 *>(r) = make_float2(th[j][0], th[j][1]);
      *reinterpret_cast<float4 *>(r + 4) = make_float4(m[j][0], m[j][1], v[j][0], v[j][1]);
    } else {
#pragma unroll
      for (int i = 0; i < F / 4; ++i) {
        *reinterpret_cast<float4 *>(r + 4 * i) = make_float4(th[j][4 * i], th[j][4 * i + 1], th[j][4 * i + 2], th[j][4 * i + 3]);
        *reinterpret_cast<float4 *>(r + 2 * F + 4 * i) = make_float4(m[j][4 * i], m[j][4 * i + 1], m[j][4 * i + 2], m[j][4 * i + 3]);
        *reinterpret_cast<float4 *>(r + 3 * F + 4 * i) = make_float4(v[j][4 * i], v[j][4 * i + 1], v[j][4 * i + 2], v[j][4 * i + 3]);
      }
    }
  }
  if (any) {
    if (e0 + B <= n_entries) {
      float4 *g4 = reinterpret_cast<float4 *>(grad + e0 * F);
#pragma unroll
      for (int i = 0; i < NV; ++i) g4[i] = make_float4(g[4 * i], g[4 * i + 1], g[4 * i + 2], g[4 * i + 3]);
    } else {
#pragma unroll
      for (int i = 0; i < B * F; ++i)
        if (e0 * F + i < n_entries * F) grad[e0 * F + i] = g[i];
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
  (void)n_sms;
  AdamConst c{lr, beta1, beta2, eps, inv_bc1, inv_bc2};
  const uint64_t per_thread = F >= 4 ? 1 : 4 / F;
  const uint64_t n_threads = (fp.n_entries + per_thread - 1) / per_thread;
  dim3 grid((unsigned)((n_threads + 255) / 256)), block(256);
  switch (F) {
    case 1: adam_table_kernel<1><<<grid, block, 0, st>>>(fp.rec, fp.grad, fp.n_entries, sparse, c); break;
    case 2: adam_table_kernel<2><<<grid, block, 0, st>>>(fp.rec, fp.grad, fp.n_entries, sparse, c); break;
    case 4: adam_table_kernel<4><<<grid, block, 0, st>>>(fp.rec, fp.grad, fp.n_entries, sparse, c); break;
    default: adam_table_kernel<8><<<grid, block, 0, st>>>(fp.rec, fp.grad, fp.n_entries, sparse, c); break;
  }
  return 1;
}

int launch_adam_mlp(const FieldParams &fp, float lr, float beta1, float beta2, float eps, float inv_bc1, float inv_bc2,
                    cudaStream_t st) {
  AdamConst c{lr, beta1, beta2, eps, inv_bc1, inv_bc2};
  adam_dense_kernel<<<(unsigned)((fp.n_mlp + 255) / 256), 256, 0, st>>>(fp.mlp_theta, fp.mlp_m, fp.mlp_v, fp.mlp_grad, fp.n_mlp, c);
  return 1;
}
