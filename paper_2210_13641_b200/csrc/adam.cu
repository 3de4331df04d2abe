// adam.cu — S13 of DESIGN.md "Algorithm": Adam with bias correction (the paper names no
// optimiser, PAPER.md:133 only says L_M is minimised; reading R16).  Tables: only the entries
// of the structural touched set U are updated when sparse_table_adam = 1 — untouched entries
// keep theta, m, v bit-unchanged.  The gradient words are reset to "untouched" in the same pass,
// so the next step's scatter starts clean without a separate memset.
#include "nsm_internal.cuh"

namespace {

// One block per chunk of ADAM_CHUNK_FLOATS / F consecutive entries, two phases.
//  1. The chunk's gradient words are read densely (coalesced 16-byte loads, four independent ones
//     per thread; the array is L2-hot, the scatter has just written it).  Entries whose first word
//     is not -0.0f (FieldParams: "referenced this step") are compacted into shared memory
//     (index + gradient), warp-aggregated.
//  2. The block walks the compact list: every thread has a touched entry, loads its theta (compact
//     array) and its moment record (m | v; 16 bytes for F = 2; two entries in flight per thread),
//     updates and stores them.  The whole gradient chunk is then reset to -0.0f with coalesced
//     stores, so the next step's scatter starts from "untouched" without a separate pass.
// sparse = 0 (dense Adam, textbook): every entry goes through phase 2.
constexpr int ADAM_CHUNK_FLOATS = 4096;
constexpr int ADAM_THREADS = 256;

// one touched entry: theta (F floats of the compact array) and its moment record (m | v, 2F floats)
template <int F>
__device__ __forceinline__ void adam_entry(float *__restrict__ th_p, float *__restrict__ mv_p, const float *g, const AdamConst &c,
                                           uint64_t pol_ld, uint64_t pol_st) {
  float th[F], m[F], v[F];
  if constexpr (F == 1) {
    th[0] = ld_hint_f1(th_p, pol_ld);
    const float2 t = ld_hint_f2(mv_p, pol_ld);
    m[0] = t.x; v[0] = t.y;
  } else if constexpr (F == 2) {
    const float2 a = ld_hint_f2(th_p, pol_ld);
    const float4 b = ld_hint_f4(mv_p, pol_ld);
    th[0] = a.x; th[1] = a.y; m[0] = b.x; m[1] = b.y; v[0] = b.z; v[1] = b.w;
  } else {
#pragma unroll
    for (int i = 0; i < F / 4; ++i) {
      const float4 a = ld_hint_f4(th_p + 4 * i, pol_ld), b = ld_hint_f4(mv_p + 4 * i, pol_ld), d = ld_hint_f4(mv_p + F + 4 * i, pol_ld);
      th[4 * i] = a.x; th[4 * i + 1] = a.y; th[4 * i + 2] = a.z; th[4 * i + 3] = a.w;
      m[4 * i] = b.x; m[4 * i + 1] = b.y; m[4 * i + 2] = b.z; m[4 * i + 3] = b.w;
      v[4 * i] = d.x; v[4 * i + 1] = d.y; v[4 * i + 2] = d.z; v[4 * i + 3] = d.w;
    }
  }
#pragma unroll
  for (int f = 0; f < F; ++f) adam_one(th[f], m[f], v[f], g[f], c);
  if constexpr (F == 1) {
    st_hint_f1(th_p, th[0], pol_st);
    st_hint_f2(mv_p, make_float2(m[0], v[0]), pol_st);
  } else if constexpr (F == 2) {
    st_hint_f2(th_p, make_float2(th[0], th[1]), pol_st);
    st_hint_f4(mv_p, make_float4(m[0], m[1], v[0], v[1]), pol_st);
  } else {
#pragma unroll
    for (int i = 0; i < F / 4; ++i) {
      st_hint_f4(th_p + 4 * i, make_float4(th[4 * i], th[4 * i + 1], th[4 * i + 2], th[4 * i + 3]), pol_st);
      st_hint_f4(mv_p + 4 * i, make_float4(m[4 * i], m[4 * i + 1], m[4 * i + 2], m[4 * i + 3]), pol_st);
      st_hint_f4(mv_p + F + 4 * i, make_float4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]), pol_st);
    }
  }
}

template <int F>
__global__ void __launch_bounds__(ADAM_THREADS) adam_table_kernel(float *__restrict__ theta, float *__restrict__ mv, float *__restrict__ grad,
                                                                  uint64_t first_entry, uint64_t n_entries, int sparse, AdamConst c,
                                                                  unsigned long long *tl) {
  constexpr int CH = ADAM_CHUNK_FLOATS / F;            // entries per chunk
  constexpr int NV = ADAM_CHUNK_FLOATS / 4 / ADAM_THREADS;   // float4 loads per thread
  __shared__ float list_g[ADAM_CHUNK_FLOATS];          // compacted gradients, F floats per touched entry
  __shared__ uint16_t list_e[CH];                      // compacted local entry indices
  __shared__ uint32_t cnt;
  const uint32_t tid = threadIdx.x, lane = tid & 31;
  pdl_wait();
  pdl_trigger();
  tl_mark(tl, K_ADAM_TABLE, 0);
  const uint64_t e_base = first_entry + (uint64_t)blockIdx.x * CH;   // first_entry is a multiple of 4 entries (16-byte loads)
  const uint64_t n_float = n_entries * F;
  const float *g4 = grad + e_base * F;
  const uint64_t pol_first = l2_evict_first(), pol_last = l2_evict_last(), pol_ld = l2_evict_normal();
  if (tid == 0) cnt = 0;
  float4 gv[NV];
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const uint32_t q = j * ADAM_THREADS + tid;         // float4 index inside the chunk
    gv[j] = (e_base * F + 4ull * q < n_float) ? ld_hint_f4(g4 + 4 * q, pol_last) : make_float4(0.f, 0.f, 0.f, 0.f);   // the array is padded to 256 B
  }
  __syncthreads();
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const uint32_t q = j * ADAM_THREADS + tid;
    const float w[4] = {gv[j].x, gv[j].y, gv[j].z, gv[j].w};
    if constexpr (F <= 4) {
      constexpr int EPV = 4 / F;                       // entries per float4
#pragma unroll
      for (int i = 0; i < EPV; ++i) {
        const uint32_t le = q * EPV + i;               // local entry index
        const bool t = (e_base + le < n_entries) && (!sparse || __float_as_uint(w[i * F]) != NSM_GRAD_UNTOUCHED);
        const uint32_t mk = __ballot_sync(0xffffffffu, t);
        uint32_t base = 0;
        if (lane == 0 && mk) base = atomicAdd(&cnt, (uint32_t)__popc(mk));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (t) {
          const uint32_t pos = base + __popc(mk & ((1u << lane) - 1u));
          list_e[pos] = (uint16_t)le;
#pragma unroll
          for (int f = 0; f < F; ++f) list_g[pos * F + f] = w[i * F + f];
        }
      }
    } else {                                           // F = 8: an entry spans two float4 (q even: first half)
      const uint32_t le = q >> 1;
      const uint32_t first_word = __float_as_uint(__shfl_sync(0xffffffffu, w[0], lane & ~1u));
      const bool t = (e_base + le < n_entries) && (!sparse || first_word != NSM_GRAD_UNTOUCHED);
      const uint32_t mk = __ballot_sync(0xffffffffu, t && !(lane & 1u));
      uint32_t base = 0;
      if (lane == 0 && mk) base = atomicAdd(&cnt, (uint32_t)__popc(mk));
      base = __shfl_sync(0xffffffffu, base, 0);
      if (t) {
        const uint32_t pos = base + __popc(mk & ((1u << (lane & ~1u)) - 1u));
        if (!(lane & 1u)) list_e[pos] = (uint16_t)le;
#pragma unroll
        for (int f = 0; f < 4; ++f) list_g[pos * F + (lane & 1u) * 4 + f] = w[f];
      }
    }
  }
  __syncthreads();
  const uint32_t n = cnt;
  if (n == 0) { tl_mark(tl, K_ADAM_TABLE, 1); return; }
  // phase 2: two records in flight per thread
  for (uint32_t i0 = tid; i0 < n; i0 += 2 * ADAM_THREADS) {
    const uint32_t i1 = i0 + ADAM_THREADS;
    const uint64_t e0 = e_base + list_e[i0], e1 = e_base + list_e[i1 < n ? i1 : i0];
    if constexpr (F == 2) {   // touch the second entry's moment record early
      asm volatile("prefetch.global.L2 [%0];" ::"l"(mv + e1 * 2 * F));
    }
    adam_entry<F>(theta + e0 * F, mv + e0 * 2 * F, list_g + i0 * F, c, pol_ld, pol_first);
    if (i1 < n) adam_entry<F>(theta + e1 * F, mv + e1 * 2 * F, list_g + i1 * F, c, pol_ld, pol_first);
  }
  // reset the chunk's gradient words
  float *o4 = grad + e_base * F;
  const float nz = __uint_as_float(NSM_GRAD_UNTOUCHED);
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const uint32_t q = j * ADAM_THREADS + tid;
    if (e_base * F + 4ull * q < n_float) st_hint_f4(o4 + 4 * q, make_float4(nz, nz, nz, nz), pol_last);
  }
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

// entries [first_entry, end_entry): a level group (first_entry must be a multiple of 4)
int launch_adam_table(const FieldParams &fp, uint32_t F, int sparse, float lr, float beta1, float beta2, float eps,
                      float inv_bc1, float inv_bc2, uint64_t first_entry, uint64_t end_entry, cudaStream_t st,
                      unsigned long long *tl) {
  AdamConst c{lr, beta1, beta2, eps, inv_bc1, inv_bc2};
  const uint64_t chunk = ADAM_CHUNK_FLOATS / F;
  dim3 grid((unsigned)((end_entry - first_entry + chunk - 1) / chunk)), block(ADAM_THREADS);
  switch (F) {
    case 1: launch_pdl(adam_table_kernel<1>, grid, block, 0, st, fp.theta, fp.mv, fp.grad, first_entry, end_entry, sparse, c, tl); break;
    case 2: launch_pdl(adam_table_kernel<2>, grid, block, 0, st, fp.theta, fp.mv, fp.grad, first_entry, end_entry, sparse, c, tl); break;
    case 4: launch_pdl(adam_table_kernel<4>, grid, block, 0, st, fp.theta, fp.mv, fp.grad, first_entry, end_entry, sparse, c, tl); break;
    default: launch_pdl(adam_table_kernel<8>, grid, block, 0, st, fp.theta, fp.mv, fp.grad, first_entry, end_entry, sparse, c, tl); break;
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
