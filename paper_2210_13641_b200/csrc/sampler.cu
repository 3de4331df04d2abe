// sampler.cu — row F1: the ray-batch sampler over the device-side keyframe store.  The mapping
// thread optimises over all keyframes received so far, each with its pose, image, depth map and depth variance
// (PAPER.md:157-159); one training batch is n_rays (keyframe, pixel) pairs drawn uniformly.  DESIGN.md "F1":
//   kf  = (h(seed, draw, r, 0xffff0001) * n_kf)  >> 32        pix = (h(seed, draw, r, 0xffff0002) * (W H)) >> 32
//   (xc, yc) = ((u - cx) / fx, (v - cy) / fy),  n2 = fma(xc, xc, fma(yc, yc, 1)),  n = sqrt(n2)
//   d = R (xc, yc, 1) / n (fma chain below),  o = t,  range = z-depth * n,  variance * n2
// Index-path rule: every float operation is an explicit round-to-nearest intrinsic in the order of the oracle, so
// the batch is bit-identical to the oracle's.  One thread per ray: a pure gather (5 floats from a random pixel).
#include "nsm_internal.cuh"

namespace {

__global__ void __launch_bounds__(256) sample_batch_kernel(const KeyframeDev *__restrict__ kfs, uint32_t n_kf, uint64_t seed,
                                                           uint32_t draw, uint32_t n_rays, float *__restrict__ origins,
                                                           float *__restrict__ dirs, float *__restrict__ rgb,
                                                           float *__restrict__ depth, float *__restrict__ depth_var,
                                                           uint32_t *__restrict__ ray_kf) {
  const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n_rays) return;
  const uint32_t hp = nsm_hash_prefix(seed, draw, r);
  const uint32_t kf = (uint32_t)(((uint64_t)nsm_mix32(hp ^ 0xffff0001u) * (uint64_t)n_kf) >> 32);
  const KeyframeDev k = kfs[kf];
  const uint32_t pix = (uint32_t)(((uint64_t)nsm_mix32(hp ^ 0xffff0002u) * ((uint64_t)k.W * k.H)) >> 32);
  const uint32_t u = pix % k.W, v = pix / k.W;
  const float xc = __fdiv_rn(__fsub_rn(__uint2float_rn(u), k.cx), k.fx);
  const float yc = __fdiv_rn(__fsub_rn(__uint2float_rn(v), k.cy), k.fy);
  const float n2 = __fmaf_rn(xc, xc, __fmaf_rn(yc, yc, 1.0f));
  const float n = __fsqrt_rn(n2);
  const float dx = __fdiv_rn(xc, n), dy = __fdiv_rn(yc, n), dz = __fdiv_rn(1.0f, n);
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    float acc = __fmul_rn(k.R[3 * i + 2], dz);
    acc = __fmaf_rn(k.R[3 * i + 1], dy, acc);
    acc = __fmaf_rn(k.R[3 * i + 0], dx, acc);
    dirs[3 * (size_t)r + i] = acc;
    origins[3 * (size_t)r + i] = k.t[i];
    rgb[3 * (size_t)r + i] = __ldg(k.rgb + 3 * (size_t)pix + i);
  }
  depth[r] = __fmul_rn(__ldg(k.depth + pix), n);
  depth_var[r] = __fmul_rn(__ldg(k.var + pix), n2);
  if (ray_kf) ray_kf[r] = kf;
}

}  // namespace

int launch_sample_batch(const KeyframeDev *kfs, uint32_t n_kf, uint64_t seed, uint32_t draw, uint32_t n_rays, float *origins,
                        float *dirs, float *rgb, float *depth, float *depth_var, uint32_t *ray_kf, cudaStream_t st) {
  sample_batch_kernel<<<(n_rays + 255) / 256, 256, 0, st>>>(kfs, n_kf, seed, draw, n_rays, origins, dirs, rgb, depth, depth_var, ray_kf);
  return 1;
}
