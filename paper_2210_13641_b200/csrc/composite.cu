// composite.cu — S8 (transmittance + alpha compositing, Eqs. 5, 6 and the colour sum at
// PAPER.md:151), S9 (loss, Eqs. 3, 4, 7) and S10 (its derivative w.r.t. sigma_i and c_i) in ONE
// kernel: a ray's loss gradient depends only on that ray's own C and D_hat (L is a mean over
// rays), so the backward sweep can follow the forward sweep without leaving the warp.
//
// One warp per ray.  Forward: 32 samples at a time, a warp inclusive scan of a_i = sigma_i delta_i
// gives T_i = exp(-sum_{j<i} a_j) (Eq. 6); the carry crosses chunks (rays have up to K = 512
// samples).  Backward: chunks in reverse, a warp suffix scan of w_j q_j.
#include "nsm_internal.cuh"

namespace {

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int s = 16; s > 0; s >>= 1) v += __shfl_xor_sync(0xffffffffu, v, s);
  return v;
}

__device__ __forceinline__ float warp_incl_scan(float v, uint32_t lane) {
#pragma unroll
  for (int s = 1; s < 32; s <<= 1) {
    float y = __shfl_up_sync(0xffffffffu, v, s);
    if (lane >= (uint32_t)s) v += y;
  }
  return v;
}

// suffix (reverse inclusive) scan
__device__ __forceinline__ float warp_suffix_scan(float v, uint32_t lane) {
#pragma unroll
  for (int s = 1; s < 32; s <<= 1) {
    float y = __shfl_down_sync(0xffffffffu, v, s);
    if (lane + s < 32) v += y;
  }
  return v;
}

template <bool TRAIN>
__global__ void __launch_bounds__(256) composite_kernel(Workspace ws, uint32_t R, const float *__restrict__ tgt_rgb,
                                                        const float *__restrict__ tgt_depth,
                                                        const float *__restrict__ tgt_var, float lambda_d,
                                                        float bg0, float bg1, float bg2, float cut,
                                                        float *__restrict__ out_rgb, float *__restrict__ out_depth,
                                                        float *__restrict__ out_opacity) {
  pdl_wait();
  pdl_trigger();
  tl_mark(ws.timeline, K_COMPOSITE, 0);
  const uint32_t r = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  float l_rgb = 0.0f, l_d = 0.0f;  // lane 0 holds the ray's loss terms
  float gmax = 0.0f;               // max |gradient entering the MLP backward| seen by this thread
  if (r < R) {
    const uint32_t off = ws.offsets[r], n = ws.offsets[r + 1] - off;
    // ---- forward (S8) ----
    float carry = 0.0f;  // sum of a_j over previous chunks
    float C0 = 0.f, C1 = 0.f, C2 = 0.f, D = 0.f, O = 0.f;
    bool stopped = false;
    for (uint32_t base = 0; base < n && !stopped; base += 32) {
      const uint32_t i = base + lane;
      const bool ok = i < n;
      const uint64_t s = (uint64_t)off + i;
      float sg = ok ? ws.sigma[s] : 0.f, dl = ok ? ws.s_delta[s] : 0.f, t = ok ? ws.s_t[s] : 0.f;
      float c0 = ok ? ws.rgb[3 * s] : 0.f, c1 = ok ? ws.rgb[3 * s + 1] : 0.f, c2 = ok ? ws.rgb[3 * s + 2] : 0.f;
      float a = sg * dl;
      float incl = warp_incl_scan(a, lane);
      float Ti = expf(-(carry + (incl - a)));   // Eq. 6
      float alpha = -expm1f(-a);                // 1 - exp(-sigma_i delta_i)
      float w = Ti * alpha;
      if (!TRAIN && cut > 0.f) {
        // S15: the ray stops after the first sample whose T_{i+1} < cut
        float Tnext = expf(-(carry + incl));
        uint32_t below = __ballot_sync(0xffffffffu, ok && Tnext < cut);
        if (below) {
          uint32_t first = __ffs(below) - 1;
          if (lane > first) w = 0.f, a = 0.f;
          stopped = true;
          incl = __shfl_sync(0xffffffffu, incl, first);  // carry ends at the stopping sample
        }
      }
      if (TRAIN && ok) ws.T_excl[s] = Ti;
      C0 += w * c0; C1 += w * c1; C2 += w * c2; D += w * t; O += w;
      carry += stopped ? incl : __shfl_sync(0xffffffffu, incl, 31);
    }
    C0 = warp_sum(C0); C1 = warp_sum(C1); C2 = warp_sum(C2); D = warp_sum(D); O = warp_sum(O);
    const float T_end = expf(-carry);
    C0 += T_end * bg0; C1 += T_end * bg1; C2 += T_end * bg2;
    if (!TRAIN) {
      if (lane == 0) {
        out_rgb[3 * (size_t)r] = C0; out_rgb[3 * (size_t)r + 1] = C1; out_rgb[3 * (size_t)r + 2] = C2;
        out_depth[r] = D;
        if (out_opacity) out_opacity[r] = O;
      }
    } else {
      if (lane == 0) {
        ws.C[3 * (size_t)r] = C0; ws.C[3 * (size_t)r + 1] = C1; ws.C[3 * (size_t)r + 2] = C2;
        ws.D_hat[r] = D; ws.O[r] = O;
      }
      // ---- loss (S9) and per-ray gradients ----
      const float invR = 1.0f / (float)R;
      float e0 = C0 - tgt_rgb[3 * (size_t)r], e1 = C1 - tgt_rgb[3 * (size_t)r + 1], e2 = C2 - tgt_rgb[3 * (size_t)r + 2];
      l_rgb = e0 * e0 + e1 * e1 + e2 * e2;                                     // Eq. 7
      float gC0 = 2.f * invR * e0, gC1 = 2.f * invR * e1, gC2 = 2.f * invR * e2;
      float dsl = tgt_depth[r], var = tgt_var[r], gD = 0.f;
      if (dsl > 0.f && var > 0.f && isfinite(var)) {                           // R13 mask
        float ed = D - dsl;
        l_d = ed * ed / var;                                                   // Eq. 4
        gD = 2.f * lambda_d * invR * ed / var;
      }
      const float bgdot = bg0 * gC0 + bg1 * gC1 + bg2 * gC2;
      // ---- backward (S10): chunks in reverse ----
      float suffix_carry = 0.f;  // sum_{j in later chunks} w_j q_j
      const uint32_t n_chunks = (n + 31) >> 5;
      for (uint32_t ch = n_chunks; ch-- > 0;) {
        const uint32_t i = ch * 32 + lane;
        const bool ok = i < n;
        const uint64_t s = (uint64_t)off + i;
        float sg = ok ? ws.sigma[s] : 0.f, dl = ok ? ws.s_delta[s] : 0.f, t = ok ? ws.s_t[s] : 0.f;
        float c0 = ok ? ws.rgb[3 * s] : 0.f, c1 = ok ? ws.rgb[3 * s + 1] : 0.f, c2 = ok ? ws.rgb[3 * s + 2] : 0.f;
        float Ti = ok ? ws.T_excl[s] : 0.f;
        float a = sg * dl;
        float ea = expf(-a);
        float w = Ti * (-expm1f(-a));
        float Tn = Ti * ea;                                                    // T_{i+1}
        float q = c0 * gC0 + c1 * gC1 + c2 * gC2 + t * gD;
        float wq = w * q;
        float sfx_incl = warp_suffix_scan(wq, lane);
        float sfx = suffix_carry + (sfx_incl - wq);                            // sum_{j>i} w_j q_j
        if (ok) {
          const float ds = dl * (Tn * q - sfx - T_end * bgdot);
          ws.dsigma[s] = ds;
          ws.drgb[3 * s] = w * gC0; ws.drgb[3 * s + 1] = w * gC1; ws.drgb[3 * s + 2] = w * gC2;
          // what S11 starts from: dL/dg0 = dsigma*sigma and dL/d(pre-sigmoid) = dc * c(1-c)
          gmax = fmaxf(gmax, fabsf(ds * sg));
          gmax = fmaxf(gmax, 0.25f * w * fmaxf(fabsf(gC0), fmaxf(fabsf(gC1), fabsf(gC2))));
        }
        suffix_carry += __shfl_sync(0xffffffffu, sfx_incl, 0);
      }
    }
  }
  if (TRAIN) {
    // block reduction of the loss terms, one double atomic per block and term
    __shared__ float red[2][8];
    const uint32_t wid = threadIdx.x >> 5;
    if (lane == 0) { red[0][wid] = l_rgb; red[1][wid] = l_d; }
    __syncthreads();
    if (threadIdx.x < 2) {
      double acc = 0.0;
      for (uint32_t w = 0; w < (blockDim.x >> 5); ++w) acc += (double)red[threadIdx.x][w];
      atomicAdd(ws.loss_acc + threadIdx.x, acc);
    }
#pragma unroll
    for (int sft = 16; sft > 0; sft >>= 1) gmax = fmaxf(gmax, __shfl_xor_sync(0xffffffffu, gmax, sft));
    if (lane == 0 && gmax > 0.f && isfinite(gmax)) atomicMax(ws.grad_absmax, __float_as_uint(gmax));
  }
  tl_mark(ws.timeline, K_COMPOSITE, 1);
}

}  // namespace

int launch_composite_train(const Workspace &ws, uint32_t R, const float *rgb, const float *depth,
                           const float *depth_var, float lambda_d, const float bg[3], cudaStream_t st) {
  dim3 grid((R + 7) / 8), block(256);
  launch_pdl(composite_kernel<true>, grid, block, 0, st, ws, R, rgb, depth, depth_var, lambda_d, bg[0], bg[1], bg[2], 0.f,
             (float *)nullptr, (float *)nullptr, (float *)nullptr);
  return 1;
}

int launch_composite_render(const Workspace &ws, uint32_t R, float cut, const float bg[3], float *out_rgb,
                            float *out_depth, float *out_opacity, cudaStream_t st) {
  dim3 grid((R + 7) / 8), block(256);
  launch_pdl(composite_kernel<false>, grid, block, 0, st, ws, R, (const float *)nullptr, (const float *)nullptr,
             (const float *)nullptr, 0.f, bg[0], bg[1], bg[2], cut, out_rgb, out_depth, out_opacity);
  return 1;
}
