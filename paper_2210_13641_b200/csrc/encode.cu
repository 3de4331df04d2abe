// encode.cu — S4 (multiresolution hash-grid encoding, forward gather) and S12 (table-gradient
// scatter) of DESIGN.md "Algorithm".  PAPER.md:65,143,167 delegate the encoding to [17]; the
// vertex grid, dense-vs-hashed rule and XOR-of-products hash are readings R11.
//
// Work decomposition: one thread per (level, sample), level-major, so that a warp holds 32
// consecutive samples (neighbours along a ray) of ONE level: their corners share cache lines at
// coarse levels, the whole chip works on one level's table slice at a time (L2/L1 locality), and
// the feature planes e[l*F+f][s] are written / read fully coalesced.
#include <cuda_bf16.h>
#include <cuda_fp16.h>

#include "nsm_internal.cuh"

namespace {

struct CornerIndex {
  uint32_t slot[8];
  float w[3];
};

// Index path of S4 (fp32 ops explicit; integers bit-exact against the oracle).
__device__ __forceinline__ CornerIndex corner_index(const LevelTable &lv, uint32_t l, float x0,
                                                    float x1, float x2) {
  CornerIndex ci;
  const uint32_t N = lv.res[l];
  const float Nf = __uint2float_rn(N);
  uint32_t c0[3];
  const float x[3] = {x0, x1, x2};
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    float pos = __fmul_rn(x[a], Nf);
    int c = min(__float2int_rd(pos), (int)N - 1);
    c = max(c, 0);
    c0[a] = (uint32_t)c;
    ci.w[a] = __fsub_rn(pos, __int2float_rn(c));
  }
  if (lv.dense[l]) {
    const uint32_t side = N + 1;
#pragma unroll
    for (uint32_t k = 0; k < 8; ++k)
      ci.slot[k] = (c0[0] + (k & 1u)) + side * ((c0[1] + ((k >> 1) & 1u)) + side * (c0[2] + ((k >> 2) & 1u)));
  } else {
#pragma unroll
    for (uint32_t k = 0; k < 8; ++k)
      ci.slot[k] = ((c0[0] + (k & 1u)) ^ ((c0[1] + ((k >> 1) & 1u)) * 2654435761u) ^
                    ((c0[2] + ((k >> 2) & 1u)) * 805459861u)) & lv.t_mask;
  }
  return ci;
}

__device__ __forceinline__ float corner_weight(uint32_t k, const float w[3]) {
  float a = (k & 1u) ? w[0] : 1.0f - w[0];
  float b = (k & 2u) ? w[1] : 1.0f - w[1];
  float c = (k & 4u) ? w[2] : 1.0f - w[2];
  return a * b * c;
}

template <int F> struct Vec;
template <> struct Vec<1> { using T = float; };
template <> struct Vec<2> { using T = float2; };
template <> struct Vec<4> { using T = float4; };

// the same through an L2 cache-policy (hashed levels: stream, evict first)
template <int F>
__device__ __forceinline__ void load_entry_hint(const float *p, float out[F], uint64_t pol) {
  if constexpr (F == 8) {
    float4 a = ld_hint_f4(p, pol), b = ld_hint_f4(p + 4, pol);
    out[0] = a.x; out[1] = a.y; out[2] = a.z; out[3] = a.w;
    out[4] = b.x; out[5] = b.y; out[6] = b.z; out[7] = b.w;
  } else if constexpr (F == 4) {
    float4 a = ld_hint_f4(p, pol);
    out[0] = a.x; out[1] = a.y; out[2] = a.z; out[3] = a.w;
  } else if constexpr (F == 2) {
    float2 a = ld_hint_f2(p, pol);
    out[0] = a.x; out[1] = a.y;
  } else {
    out[0] = ld_hint_f1(p, pol);
  }
}

template <int F>
__device__ __forceinline__ void load_entry(const float *p, float out[F]) {
  if constexpr (F == 8) {
    float4 a = __ldg(reinterpret_cast<const float4 *>(p)), b = __ldg(reinterpret_cast<const float4 *>(p) + 1);
    out[0] = a.x; out[1] = a.y; out[2] = a.z; out[3] = a.w;
    out[4] = b.x; out[5] = b.y; out[6] = b.z; out[7] = b.w;
  } else if constexpr (F == 4) {
    float4 a = __ldg(reinterpret_cast<const float4 *>(p));
    out[0] = a.x; out[1] = a.y; out[2] = a.z; out[3] = a.w;
  } else if constexpr (F == 2) {
    float2 a = __ldg(reinterpret_cast<const float2 *>(p));
    out[0] = a.x; out[1] = a.y;
  } else {
    out[0] = __ldg(p);
  }
}

// MODE 0: e -> fp32 planes [l*F+f][cap].  MODE 1 / 2: e -> fp16 / bf16 operand-tile blob of the
// tensor-core MLP kernels ([tile][8-column panel][128 rows][8 x 16 bit], mlp_tc.cu); the rows of
// the last tile beyond S are zero-filled so the MMA never reads stale data.
template <int F, int MODE>
__global__ void __launch_bounds__(256) encode_forward_kernel(LevelTable lv, const float *__restrict__ theta,
                                                             Workspace ws, const uint32_t *__restrict__ d_S) {
  pdl_wait();
  pdl_trigger();
  tl_mark(ws.timeline, K_ENCODE, 0);
  const uint64_t S = *d_S;
  const uint64_t S_it = MODE == 0 ? S : ((S + NSM_TILE - 1) / NSM_TILE) * NSM_TILE;
  const uint64_t total = S_it * lv.n_levels;
  const uint32_t LF = lv.n_levels * F;
  const uint64_t pol_first = l2_evict_first();
  for (uint64_t wi = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; wi < total;
       wi += (uint64_t)gridDim.x * blockDim.x) {
    const uint32_t l = (uint32_t)(wi / S_it);
    const uint64_t s = wi - (uint64_t)l * S_it;
    float acc[F];
#pragma unroll
    for (int f = 0; f < F; ++f) acc[f] = 0.0f;
    if (s < S) {
      CornerIndex ci = corner_index(lv, l, ws.s_x[s], ws.s_x[ws.cap + s], ws.s_x[2 * ws.cap + s]);
      const float *tab = theta + lv.offset[l] * F;
      float v[8][F];
#pragma unroll
      if (lv.dense[l]) {   // coarse levels are re-read every step: normal policy; hashed levels stream through L2
#pragma unroll
        for (int k = 0; k < 8; ++k) load_entry<F>(tab + (size_t)ci.slot[k] * F, v[k]);  // 8 gathers in flight
      } else {
#pragma unroll
        for (int k = 0; k < 8; ++k) load_entry_hint<F>(tab + (size_t)ci.slot[k] * F, v[k], pol_first);
      }
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        float om = corner_weight(k, ci.w);
#pragma unroll
        for (int f = 0; f < F; ++f) acc[f] = fmaf(om, v[k][f], acc[f]);
      }
    }
    if (MODE == 0) {
#pragma unroll
      for (int f = 0; f < F; ++f) ws.e[(size_t)(l * F + f) * ws.cap + s] = acc[f];
    } else {
      const uint32_t c = l * F;   // F consecutive columns never straddle an 8-column panel (F | 8)
      // two-term tile: [hi: LF*256 bytes][lo: LF*256 bytes] per 128-sample tile (e = hi + lo)
      const size_t half = (size_t)LF * NSM_TILE * 2;
      uint8_t *dst = ws.blob_e + (s >> 7) * (2 * half) + (c >> 3) * (NSM_TILE * 16) + (s & 127) * 16 + (c & 7) * 2;
#pragma unroll
      for (int f = 0; f < F; ++f) {
        if (MODE == 1) {
          const __half hi = __float2half_rn(acc[f]);
          reinterpret_cast<__half *>(dst)[f] = hi;
          reinterpret_cast<__half *>(dst + half)[f] = __float2half_rn(acc[f] - __half2float(hi));
        } else {
          const __nv_bfloat16 hi = __float2bfloat16_rn(acc[f]);
          reinterpret_cast<__nv_bfloat16 *>(dst)[f] = hi;
          reinterpret_cast<__nv_bfloat16 *>(dst + half)[f] = __float2bfloat16_rn(acc[f] - __bfloat162float(hi));
        }
      }
    }
  }
  tl_mark(ws.timeline, K_ENCODE, 1);
}

template <int F>
__device__ __forceinline__ void red_add_entry(float *p, const float g[F], uint64_t pol) {
  // vectorised no-return reductions (red.global.add.v2/v4.f32, sm_90+); the gradient array stays in L2
  if constexpr (F == 8) {
    red_hint_f4(p, make_float4(g[0], g[1], g[2], g[3]), pol);
    red_hint_f4(p + 4, make_float4(g[4], g[5], g[6], g[7]), pol);
  } else if constexpr (F == 4) {
    red_hint_f4(p, make_float4(g[0], g[1], g[2], g[3]), pol);
  } else if constexpr (F == 2) {
    red_hint_f2(p, make_float2(g[0], g[1]), pol);
  } else {
    red_hint_f1(p, g[0], pol);
  }
}

// S12: d theta[(offset_l + slot) F + f] += omega * dL/de[l F + f].  The touched set U is structural
// (every referenced entry, independent of the gradient's value): it is carried by the gradient words
// themselves, see FieldParams in nsm_internal.cuh.
template <int F>
__global__ void __launch_bounds__(256) scatter_backward_kernel(LevelTable lv, float *__restrict__ grad, Workspace ws,
                                                               const uint32_t *__restrict__ d_S, uint32_t l0, uint32_t l1) {
  pdl_wait();
  pdl_trigger();
  tl_mark(ws.timeline, K_SCATTER, 0);
  const uint64_t S = *d_S;
  const uint64_t total = S * (l1 - l0);
  const uint64_t pol_last = l2_evict_last();
  for (uint64_t wi = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; wi < total;
       wi += (uint64_t)gridDim.x * blockDim.x) {
    const uint32_t l = l0 + (uint32_t)(wi / S);
    const uint64_t s = wi - (uint64_t)(l - l0) * S;
    CornerIndex ci = corner_index(lv, l, ws.s_x[s], ws.s_x[ws.cap + s], ws.s_x[2 * ws.cap + s]);
    float de[F];
#pragma unroll
    for (int f = 0; f < F; ++f) de[f] = ws.de[(size_t)(l * F + f) * ws.cap + s];
    float *tab = grad + lv.offset[l] * F;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      float om = corner_weight(k, ci.w);
      float g[F];
#pragma unroll
      for (int f = 0; f < F; ++f) {
        const float v = om * de[f];
        g[f] = fabsf(v) < NSM_GRAD_MIN_ADDEND ? 0.0f : v;   // never -0.0, never near-subnormal; NaN stays NaN
      }
      red_add_entry<F>(tab + (size_t)ci.slot[k] * F, g, pol_last);
    }
  }
  tl_mark(ws.timeline, K_SCATTER, 1);
}

// gradient array <- canonical gradient and flags (debug / test entry point)
__global__ void set_grad_kernel(float *__restrict__ grad, uint32_t F, uint64_t n_entries, const float *__restrict__ src,
                                const uint8_t *__restrict__ touched) {
  const uint64_t total = n_entries * F;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t e = i / F;
    const bool t = src && (!touched || touched[e]);
    const float v = t ? src[i] : 0.f;
    grad[i] = t ? (fabsf(v) < NSM_GRAD_MIN_ADDEND ? 0.0f : v) : __uint_as_float(NSM_GRAD_UNTOUCHED);
  }
}

__global__ void get_touched_kernel(const float *__restrict__ grad, uint32_t F, uint64_t n_entries, uint8_t *__restrict__ dst) {
  for (uint64_t e = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_entries; e += (uint64_t)gridDim.x * blockDim.x)
    dst[e] = __float_as_uint(grad[e * F]) != NSM_GRAD_UNTOUCHED;
}

__global__ void debug_slots_kernel(LevelTable lv, Workspace ws, const uint32_t *__restrict__ d_S,
                                   uint32_t *slots, float *w) {
  const uint64_t S = *d_S;
  const uint64_t total = S * lv.n_levels;
  for (uint64_t wi = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; wi < total;
       wi += (uint64_t)gridDim.x * blockDim.x) {
    const uint32_t l = (uint32_t)(wi / S);
    const uint64_t s = wi - (uint64_t)l * S;
    CornerIndex ci = corner_index(lv, l, ws.s_x[s], ws.s_x[ws.cap + s], ws.s_x[2 * ws.cap + s]);
    if (slots)
      for (int k = 0; k < 8; ++k) slots[(s * lv.n_levels + l) * 8 + k] = ci.slot[k];
    if (w)
      for (int a = 0; a < 3; ++a) w[(s * lv.n_levels + l) * 3 + a] = ci.w[a];
  }
}

__global__ void planes_to_rows_kernel(const float *__restrict__ planes, uint64_t cap, uint32_t n_planes,
                                      const uint32_t *__restrict__ d_S, float *__restrict__ rows) {
  const uint64_t S = *d_S;
  const uint64_t total = S * n_planes;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total;
       i += (uint64_t)gridDim.x * blockDim.x) {
    uint64_t s = i / n_planes;
    uint32_t p = (uint32_t)(i - s * n_planes);
    rows[i] = planes[(size_t)p * cap + s];
  }
}

__device__ __forceinline__ uint64_t param_index(uint32_t F, uint64_t e, uint32_t f, int which) {
  return which == 0 ? e * F + f : e * 2 * F + (which == 3 ? F : 0) + f;
}

__global__ void pack_records_kernel(float *__restrict__ theta, float *__restrict__ mv, uint32_t F, uint64_t n_entries, int which,
                                    const float *__restrict__ src) {
  const uint64_t total = n_entries * F;
  float *dst = which == 0 ? theta : mv;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t e = i / F;
    dst[param_index(F, e, (uint32_t)(i - e * F), which)] = src ? src[i] : 0.f;
  }
}

__global__ void unpack_records_kernel(const float *__restrict__ theta, const float *__restrict__ mv, uint32_t F, uint64_t n_entries,
                                      int which, float *__restrict__ dst) {
  const uint64_t total = n_entries * F;
  const float *src = which == 0 ? theta : mv;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t e = i / F;
    dst[i] = src[param_index(F, e, (uint32_t)(i - e * F), which)];
  }
}

}  // namespace

int launch_pack_records(const FieldParams &fp, int which, const float *src, cudaStream_t st) {
  pack_records_kernel<<<2048, 256, 0, st>>>(fp.theta, fp.mv, fp.F, fp.n_entries, which, src);
  return 1;
}

int launch_unpack_records(const FieldParams &fp, int which, float *dst, cudaStream_t st) {
  unpack_records_kernel<<<2048, 256, 0, st>>>(fp.theta, fp.mv, fp.F, fp.n_entries, which, dst);
  return 1;
}

template <int F>
static void launch_encode_f(const LevelTable &lv, const float *theta, const Workspace &ws, const uint32_t *d_S, int out_mode,
                            dim3 grid, dim3 block, cudaStream_t st) {
  if (out_mode == 0) launch_pdl(encode_forward_kernel<F, 0>, grid, block, 0, st, lv, theta, ws, d_S);
  else if (out_mode == 1) launch_pdl(encode_forward_kernel<F, 1>, grid, block, 0, st, lv, theta, ws, d_S);
  else launch_pdl(encode_forward_kernel<F, 2>, grid, block, 0, st, lv, theta, ws, d_S);
}

int launch_encode(const LevelTable &lv, const float *theta, const Workspace &ws, const uint32_t *d_S, int out_mode,
                  int n_sms, cudaStream_t st) {
  dim3 grid(n_sms * 8), block(256);
  switch (lv.n_features) {
    case 1: launch_encode_f<1>(lv, theta, ws, d_S, out_mode, grid, block, st); break;
    case 2: launch_encode_f<2>(lv, theta, ws, d_S, out_mode, grid, block, st); break;
    case 4: launch_encode_f<4>(lv, theta, ws, d_S, out_mode, grid, block, st); break;
    default: launch_encode_f<8>(lv, theta, ws, d_S, out_mode, grid, block, st); break;
  }
  return 1;
}

int launch_set_grad(const FieldParams &fp, const float *src, const uint8_t *touched, cudaStream_t st) {
  set_grad_kernel<<<2048, 256, 0, st>>>(fp.grad, fp.F, fp.n_entries, src, touched);
  return 1;
}

int launch_get_touched(const FieldParams &fp, uint8_t *dst, cudaStream_t st) {
  get_touched_kernel<<<2048, 256, 0, st>>>(fp.grad, fp.F, fp.n_entries, dst);
  return 1;
}

int launch_scatter(const LevelTable &lv, float *grad, const Workspace &ws,
                   const uint32_t *d_S, uint32_t l0, uint32_t l1, int n_sms, cudaStream_t st) {
  dim3 grid(n_sms * 8), block(256);
  switch (lv.n_features) {
    case 1: launch_pdl(scatter_backward_kernel<1>, grid, block, 0, st, lv, grad, ws, d_S, l0, l1); break;
    case 2: launch_pdl(scatter_backward_kernel<2>, grid, block, 0, st, lv, grad, ws, d_S, l0, l1); break;
    case 4: launch_pdl(scatter_backward_kernel<4>, grid, block, 0, st, lv, grad, ws, d_S, l0, l1); break;
    default: launch_pdl(scatter_backward_kernel<8>, grid, block, 0, st, lv, grad, ws, d_S, l0, l1); break;
  }
  return 1;
}

int launch_debug_slots(const LevelTable &lv, const Workspace &ws, const uint32_t *d_S, uint32_t *slots,
                       float *w, cudaStream_t st) {
  debug_slots_kernel<<<1024, 256, 0, st>>>(lv, ws, d_S, slots, w);
  return 1;
}

int launch_planes_to_rows(const float *planes, uint64_t cap, uint32_t n_planes, const uint32_t *d_S,
                          float *rows, cudaStream_t st) {
  planes_to_rows_kernel<<<1024, 256, 0, st>>>(planes, cap, n_planes, d_S, rows);
  return 1;
}
