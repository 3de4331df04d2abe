// pose.cu — row f2: gradients of the mapping loss with respect to the rays, i.e. to the keyframe
// poses (L_M(T, Theta) is minimised over the poses T as well as the field).  Per ray
//     g_o = dL/do                          (translation part of the keyframe's se(3) gradient: sum over its rays)
//     tau = d/d(omega) L,  d <- exp(omega^) d   (rotation part: d x dL/dd -- tangential, so how Y is continued off the
//                                                unit sphere does not matter)
// through the two places a ray enters the step: the sample positions x = (o + t d - aabb_min) / extent (S4's trilinear
// weights: dL/dx_c = sum_l N_l sum_corners (d omega / d w_c) theta[corner] . dL/de_l) and the direction encoding Y(d)
// (S6; dL/dY comes out of the colour MLP's first-layer dgrad).  Liveness, t and delta are piecewise constant in the pose.
//
// pose_dx_kernel: 16 or 32 lanes per sample, lane = level: the 8 corner gathers of S4 once more (theta is still the
// pre-update theta: this runs between the MLP backward and Adam), dotted with dL/de; warp-reduced over levels.
// pose_ray_kernel: one warp per ray: sums dL/dx, t dL/dx and dL/dY over the ray's samples, applies the polynomial SH
// Jacobian (S6, degree <= 4) and the cross products.
#include "nsm_internal.cuh"
#include "table_ops.cuh"

namespace {

using namespace tableops;

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int s = 16; s > 0; s >>= 1) v += __shfl_xor_sync(0xffffffffu, v, s);
  return v;
}

// LPS lanes per sample (16 when L <= 16: two samples per warp; else 32), lane = level.
// n_pose: the levels l < n_pose carry the position's derivative (coarse-to-fine pose refinement, DESIGN.md 8d reading R26)
template <int F, int LPS>
__global__ void __launch_bounds__(256) pose_dx_kernel(LevelTable lv, const float *__restrict__ theta, Workspace ws,
                                                      const uint32_t *__restrict__ d_S, uint32_t n_pose) {
  const uint64_t S = *d_S;
  const uint32_t lane = threadIdx.x & (LPS - 1);
  const uint64_t group0 = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) / LPS, n_groups = ((uint64_t)gridDim.x * blockDim.x) / LPS;
  const uint64_t S_pad = (S + (32 / LPS) - 1) / (32 / LPS) * (32 / LPS);   // whole warps stay converged for the shuffles
  for (uint64_t s = group0; s < S_pad; s += n_groups) {
    float acc[3] = {0.f, 0.f, 0.f};
    if (s < S && lane < n_pose) {
      const uint32_t l = lane;
      const CornerIndex ci = corner_index(lv, l, ws.s_x[s], ws.s_x[ws.cap + s], ws.s_x[2 * ws.cap + s]);
      float de[F];
#pragma unroll
      for (int f = 0; f < F; ++f) de[f] = ws.de[(size_t)(l * F + f) * ws.cap + s];
      const float *tab = theta + lv.offset[l] * F;
      const float Nf = __uint2float_rn(lv.res[l]);
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        float th[F];
        load_entry<F>(tab + (size_t)ci.slot[k] * F, th);
        float dot = 0.f;
#pragma unroll
        for (int f = 0; f < F; ++f) dot = fmaf(th[f], de[f], dot);
        const float wx = (k & 1) ? ci.w[0] : 1.f - ci.w[0], wy = (k & 2) ? ci.w[1] : 1.f - ci.w[1],
                    wz = (k & 4) ? ci.w[2] : 1.f - ci.w[2];
        const float sx = (k & 1) ? 1.f : -1.f, sy = (k & 2) ? 1.f : -1.f, sz = (k & 4) ? 1.f : -1.f;
        acc[0] = fmaf(Nf * sx * wy * wz, dot, acc[0]);
        acc[1] = fmaf(Nf * wx * sy * wz, dot, acc[1]);
        acc[2] = fmaf(Nf * wx * wy * sz, dot, acc[2]);
      }
    }
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int sft = LPS / 2; sft > 0; sft >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], sft);
    if (s < S && lane < 3) ws.dx[(size_t)lane * ws.cap + s] = lane == 0 ? acc[0] : (lane == 1 ? acc[1] : acc[2]);
  }
}

// sum_j gY[j] grad Y_j(d), polynomial real SH of DESIGN.md S6 (no Condon-Shortley phase), n <= 4
__device__ __forceinline__ void sh_grad_dot(uint32_t n, float x, float y, float z, const float *gY, float g[3]) {
  g[0] = g[1] = g[2] = 0.f;
  if (n < 2) return;
  const float a = 0.4886025119029199f;
  g[1] += a * gY[1]; g[2] += a * gY[2]; g[0] += a * gY[3];
  if (n < 3) return;
  const float b = 1.0925484305920792f, c = 0.31539156525252005f, e = 0.5462742152960396f;
  g[0] += b * y * gY[4];          g[1] += b * x * gY[4];
  g[1] += b * z * gY[5];          g[2] += b * y * gY[5];
  g[2] += c * 6.f * z * gY[6];
  g[0] += b * z * gY[7];          g[2] += b * x * gY[7];
  g[0] += e * 2.f * x * gY[8];    g[1] -= e * 2.f * y * gY[8];
  if (n < 4) return;
  const float f = 0.5900435899266435f, q = 2.890611442640554f, h = 0.4570457994644658f, k = 0.3731763325901154f,
              m = 1.445305721320277f;
  const float xx = x * x, yy = y * y, zz = z * z;
  g[0] += f * 6.f * x * y * gY[9];          g[1] += f * 3.f * (xx - yy) * gY[9];
  g[0] += q * y * z * gY[10];               g[1] += q * x * z * gY[10];      g[2] += q * x * y * gY[10];
  g[1] += h * (5.f * zz - 1.f) * gY[11];    g[2] += h * 10.f * y * z * gY[11];
  g[2] += k * (15.f * zz - 3.f) * gY[12];
  g[0] += h * (5.f * zz - 1.f) * gY[13];    g[2] += h * 10.f * x * z * gY[13];
  g[0] += m * 2.f * x * z * gY[14];         g[1] -= m * 2.f * y * z * gY[14]; g[2] += m * (xx - yy) * gY[14];
  g[0] += f * 3.f * (xx - yy) * gY[15];     g[1] -= f * 6.f * x * y * gY[15];
}

__global__ void __launch_bounds__(256) pose_ray_kernel(Workspace ws, uint32_t R, const float *__restrict__ dirs, float inv_extent,
                                                       uint32_t sh_degree, float *__restrict__ g_o, float *__restrict__ tau) {
  const uint32_t r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (r >= R) return;
  const uint32_t off = ws.offsets[r], n = ws.offsets[r + 1] - off;
  const uint32_t n_sh = sh_degree * sh_degree;
  float so[3] = {0.f, 0.f, 0.f}, sd[3] = {0.f, 0.f, 0.f}, gY[16];
#pragma unroll
  for (int j = 0; j < 16; ++j) gY[j] = 0.f;
  for (uint32_t i = lane; i < n; i += 32) {
    const uint64_t s = (uint64_t)off + i;
    const float t = ws.s_t[s];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const float v = ws.dx[(size_t)c * ws.cap + s] * inv_extent;
      so[c] += v;
      sd[c] = fmaf(t, v, sd[c]);
    }
#pragma unroll
    for (int j = 0; j < 16; ++j)
      if ((uint32_t)j < n_sh) gY[j] += ws.dY[(size_t)j * ws.cap + s];
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) { so[c] = warp_sum(so[c]); sd[c] = warp_sum(sd[c]); }
#pragma unroll
  for (int j = 0; j < 16; ++j) gY[j] = warp_sum(gY[j]);
  if (lane == 0) {
    const float x = __ldg(dirs + 3 * (size_t)r), y = __ldg(dirs + 3 * (size_t)r + 1), z = __ldg(dirs + 3 * (size_t)r + 2);
    float g[3];
    sh_grad_dot(sh_degree, x, y, z, gY, g);
#pragma unroll
    for (int c = 0; c < 3; ++c) g[c] += sd[c];
    const float t0 = y * g[2] - z * g[1], t1 = z * g[0] - x * g[2], t2 = x * g[1] - y * g[0];
    g_o[3 * (size_t)r] = so[0]; g_o[3 * (size_t)r + 1] = so[1]; g_o[3 * (size_t)r + 2] = so[2];
    tau[3 * (size_t)r] = t0; tau[3 * (size_t)r + 1] = t1; tau[3 * (size_t)r + 2] = t2;
  }
}

// Per-keyframe se(3) gradient (translation | rotation | number of rays | pad): one block per keyframe scans the batch
// for its rays and sums their g_o and tau.  Deterministic, and no hot atomics: with ~10 keyframes the obvious
// atomicAdd per ray puts 16 K reductions on each of 70 addresses (33 us of same-address serialisation at 2^14 rays).
__global__ void __launch_bounds__(256) pose_kf_reduce_kernel(uint32_t R, const uint32_t *__restrict__ ray_kf, const float *__restrict__ g_o,
                                                             const float *__restrict__ tau, float *__restrict__ kf_grad) {
  __shared__ float red[8][7];
  const uint32_t k = blockIdx.x, lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  float acc[7] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  for (uint32_t r = threadIdx.x; r < R; r += blockDim.x) {
    if (ray_kf[r] == k) {
#pragma unroll
      for (int c = 0; c < 3; ++c) { acc[c] += g_o[3 * (size_t)r + c]; acc[3 + c] += tau[3 * (size_t)r + c]; }
      acc[6] += 1.f;
    }
  }
#pragma unroll
  for (int i = 0; i < 7; ++i) {
    acc[i] = warp_sum(acc[i]);
    if (lane == 0) red[wid][i] = acc[i];
  }
  __syncthreads();
  if (threadIdx.x < 7) {
    float v = 0.f;
    for (int w = 0; w < 8; ++w) v += red[w][threadIdx.x];
    kf_grad[NSM_KF_GRAD_STRIDE * (size_t)k + threadIdx.x] = v;
  }
}

// F2, the update: Adam on every keyframe's 6-vector that received rays in this batch, then t <- t - delta_t and
// R <- exp(-[delta_omega]x) R (Rodrigues), written into the device-side keyframe directory.  One thread per keyframe;
// the few transcendental operations run in double.
__global__ void pose_step_kernel(KeyframeDev *__restrict__ kfs, uint32_t n_kf, const float *__restrict__ kf_grad,
                                 float *__restrict__ pm, float *__restrict__ pv, uint32_t *__restrict__ pcnt, float lr_t, float lr_r,
                                 float beta1, float beta2, float eps) {
  const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= n_kf) return;
  const float *g = kf_grad + NSM_KF_GRAD_STRIDE * (size_t)k;
  if (!(g[6] > 0.f)) return;                       // no ray of this keyframe in the batch: untouched
  const uint32_t cnt = pcnt[k] + 1;
  const double bc1 = 1.0 - pow((double)beta1, (double)cnt), bc2 = 1.0 - pow((double)beta2, (double)cnt);
  double delta[6];
#pragma unroll
  for (int i = 0; i < 6; ++i) {
    const float m = beta1 * pm[6 * k + i] + (1.f - beta1) * g[i];
    const float v = beta2 * pv[6 * k + i] + (1.f - beta2) * g[i] * g[i];
    pm[6 * k + i] = m; pv[6 * k + i] = v;
    delta[i] = (double)(i < 3 ? lr_t : lr_r) * ((double)m / bc1) / (sqrt((double)v / bc2) + (double)eps);
  }
  KeyframeDev kf = kfs[k];
#pragma unroll
  for (int i = 0; i < 3; ++i) kf.t[i] = (float)((double)kf.t[i] - delta[i]);
  const double w0 = delta[3], w1 = delta[4], w2 = delta[5];
  const double a2 = w0 * w0 + w1 * w1 + w2 * w2, a = sqrt(a2);
  const double A = a > 1e-12 ? sin(a) / a : 1.0, B = a > 1e-12 ? (1.0 - cos(a)) / a2 : 0.5;
  const double K[9] = {0.0, -w2, w1, w2, 0.0, -w0, -w1, w0, 0.0};
  double E[9], Rn[9];
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      double k2 = 0.0;
#pragma unroll
      for (int q = 0; q < 3; ++q) k2 += K[3 * i + q] * K[3 * q + j];
      E[3 * i + j] = (i == j ? 1.0 : 0.0) - A * K[3 * i + j] + B * k2;
    }
#pragma unroll
  for (int i = 0; i < 3; ++i)
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      double acc = 0.0;
#pragma unroll
      for (int q = 0; q < 3; ++q) acc += E[3 * i + q] * (double)kf.R[3 * q + j];
      Rn[3 * i + j] = acc;
    }
#pragma unroll
  for (int i = 0; i < 9; ++i) kf.R[i] = (float)Rn[i];
  kfs[k] = kf;
  pcnt[k] = cnt;
}

}  // namespace

int launch_pose_step(KeyframeDev *kfs, uint32_t n_kf, const float *kf_grad, float *pm, float *pv, uint32_t *pcnt, float lr_t,
                     float lr_r, float beta1, float beta2, float eps, cudaStream_t st) {
  pose_step_kernel<<<(n_kf + 63) / 64, 64, 0, st>>>(kfs, n_kf, kf_grad, pm, pv, pcnt, lr_t, lr_r, beta1, beta2, eps);
  return 1;
}

int launch_pose_gradients(const LevelTable &lv, const float *theta, const Workspace &ws, const uint32_t *d_S, uint32_t R,
                          const float *dirs, float inv_extent, uint32_t sh_degree, float *g_o, float *tau, const uint32_t *ray_kf,
                          float *kf_grad, uint32_t n_kf, int n_sms, cudaStream_t st, uint32_t pose_levels) {
  dim3 grid(n_sms * 8), block(256);
  const uint32_t n_pose = (pose_levels == 0 || pose_levels > lv.n_levels) ? lv.n_levels : pose_levels;
  const bool half = lv.n_levels <= 16;
  switch (lv.n_features) {
    case 1: if (half) pose_dx_kernel<1, 16><<<grid, block, 0, st>>>(lv, theta, ws, d_S, n_pose); else pose_dx_kernel<1, 32><<<grid, block, 0, st>>>(lv, theta, ws, d_S, n_pose); break;
    case 2: if (half) pose_dx_kernel<2, 16><<<grid, block, 0, st>>>(lv, theta, ws, d_S, n_pose); else pose_dx_kernel<2, 32><<<grid, block, 0, st>>>(lv, theta, ws, d_S, n_pose); break;
    case 4: if (half) pose_dx_kernel<4, 16><<<grid, block, 0, st>>>(lv, theta, ws, d_S, n_pose); else pose_dx_kernel<4, 32><<<grid, block, 0, st>>>(lv, theta, ws, d_S, n_pose); break;
    default: if (half) pose_dx_kernel<8, 16><<<grid, block, 0, st>>>(lv, theta, ws, d_S, n_pose); else pose_dx_kernel<8, 32><<<grid, block, 0, st>>>(lv, theta, ws, d_S, n_pose); break;
  }
  pose_ray_kernel<<<(R + 7) / 8, 256, 0, st>>>(ws, R, dirs, inv_extent, sh_degree, g_o, tau);
  if (ray_kf && n_kf) pose_kf_reduce_kernel<<<n_kf, 256, 0, st>>>(R, ray_kf, g_o, tau, kf_grad);
  return ray_kf && n_kf ? 3 : 2;
}
