// table_ops.cuh — device code shared by the table kernels: the index path of S4 (corner slots and weights), the
// eight-corner gather / vector reduction of one (sample, level), and the touched-only Adam update of one chunk of
// entries.  Used by encode.cu (S4, S12) and adam.cu (S13).
#pragma once
#include "nsm_internal.cuh"

namespace tableops {

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

// The touched set U (S12: every entry referenced this step, whatever its gradient's value) is one bit per table entry,
// bit (e & 31) of word (e >> 5), e = offset_l + slot.  Test first, set only if clear: the test is an ordinary load that
// may be served by a stale L1 line (then the atomic is merely redundant -- bits are only ever SET while the scatter
// runs), so an entry costs one L2 atomic per step instead of one per reference.  The 0.76 MB (config 2) / 5.6 MB
// (config 4) bitmap stays cache-resident; the table Adam walks it instead of the gradient array.
__device__ __forceinline__ void mark_touched(uint32_t *__restrict__ touched, uint64_t e, uint32_t bits) {
  uint32_t *w = touched + (e >> 5);
  bits <<= (uint32_t)(e & 31u);
  if ((*w & bits) != bits) atomicOr(w, bits);
}

// S12 for one cell of one level: the eight corner reductions d theta[(offset_l + slot) F + f] += val[corner][f], and the
// eight touched bits.
template <int F>
__device__ __forceinline__ void issue_corner_reds(const LevelTable &lv, float *__restrict__ grad, uint32_t *__restrict__ touched,
                                                  uint32_t l, const uint32_t slot[8], float val[8][F], uint64_t pol_last) {
  const uint64_t e_l = lv.offset[l];
  float *tab = grad + e_l * F;
#pragma unroll
  for (int k = 0; k < 8; k += 2) {
    // The two x-neighbour corners (k, k+1) are adjacent entries whenever their slots differ in bit 0 only (always on
    // a dense level, for even cell x on a hashed one: the hash XORs x in unmultiplied): one bitmap word, and for
    // F = 2, if the pair is also 16-byte aligned in the array, one red.v4 covers both entries (~25 % fewer
    // reductions at the L2).
    const uint64_t a0 = e_l + slot[k], a1 = e_l + slot[k + 1];
    const bool pair = (a0 ^ a1) == 1ull;
    if (pair) {
      mark_touched(touched, a0 & ~1ull, 3u);
    } else {
      mark_touched(touched, a0, 1u);
      mark_touched(touched, a1, 1u);
    }
    if (F == 2 && pair) {
      float *p = grad + (a0 & ~1ull) * 2;
      if (a0 & 1ull) red_hint_f4(p, make_float4(val[k + 1][0], val[k + 1][1], val[k][0], val[k][1]), pol_last);
      else red_hint_f4(p, make_float4(val[k][0], val[k][1], val[k + 1][0], val[k + 1][1]), pol_last);
    } else {
      red_add_entry<F>(tab + (size_t)slot[k] * F, val[k], pol_last);
      red_add_entry<F>(tab + (size_t)slot[k + 1] * F, val[k + 1], pol_last);
    }
  }
}

// the corner slots of (sample s, level l) and its eight contributions omega_corner * dL/de[l F + f]
template <int F>
__device__ __forceinline__ void corner_contributions(const LevelTable &lv, const Workspace &ws, uint32_t l, uint64_t s,
                                                     uint32_t slot[8], float val[8][F]) {
  const CornerIndex ci = corner_index(lv, l, ws.s_x[s], ws.s_x[ws.cap + s], ws.s_x[2 * ws.cap + s]);
  float de[F];
#pragma unroll
  for (int f = 0; f < F; ++f) de[f] = ws.de[(size_t)(l * F + f) * ws.cap + s];
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    slot[k] = ci.slot[k];
    const float om = corner_weight(k, ci.w);
#pragma unroll
    for (int f = 0; f < F; ++f) val[k][f] = om * de[f];
  }
}

template <int F>
__device__ __forceinline__ void scatter_sample_level(const LevelTable &lv, float *__restrict__ grad, uint32_t *__restrict__ touched,
                                                     const Workspace &ws, uint32_t l, uint64_t s, uint64_t pol_last) {
  uint32_t slot[8];
  float val[8][F];
  corner_contributions<F>(lv, ws, l, s, slot, val);
  issue_corner_reds<F>(lv, grad, touched, l, slot, val, pol_last);
}

constexpr int ADAM_WORDS = 128;                    // bitmap words per block
constexpr int ADAM_ENTRIES = ADAM_WORDS * 32;      // = 4096 table entries per block
constexpr int ADAM_THREADS = 256;

template <int F>
__device__ __forceinline__ void store_entry_hint(float *p, const float v[F], uint64_t pol) {
  if constexpr (F == 8) {
    st_hint_f4(p, make_float4(v[0], v[1], v[2], v[3]), pol);
    st_hint_f4(p + 4, make_float4(v[4], v[5], v[6], v[7]), pol);
  } else if constexpr (F == 4) {
    st_hint_f4(p, make_float4(v[0], v[1], v[2], v[3]), pol);
  } else if constexpr (F == 2) {
    st_hint_f2(p, make_float2(v[0], v[1]), pol);
  } else {
    st_hint_f1(p, v[0], pol);
  }
}

// One touched entry in flight: its gradient and theta (F floats of the compact arrays each) and its moment record
// (m | v, 2F floats).  load() issues the four accesses, step() updates and stores and zeroes the gradient.
template <int F>
struct AdamRec {
  float g[F], th[F], m[F], v[F];
  __device__ __forceinline__ void load(const float *g_p, const float *th_p, const float *mv_p, uint64_t pol_g, uint64_t pol_th,
                                       uint64_t pol_mv) {
    load_entry_hint<F>(g_p, g, pol_g);
    load_entry_hint<F>(th_p, th, pol_th);
    if constexpr (F == 1) {
      const float2 t = ld_hint_f2(mv_p, pol_mv);
      m[0] = t.x; v[0] = t.y;
    } else if constexpr (F == 2) {
      const float4 t = ld_hint_f4(mv_p, pol_mv);
      m[0] = t.x; m[1] = t.y; v[0] = t.z; v[1] = t.w;
    } else {
      load_entry_hint<F>(mv_p, m, pol_mv);
      load_entry_hint<F>(mv_p + F, v, pol_mv);
    }
  }
  __device__ __forceinline__ void step(float *g_p, float *th_p, float *mv_p, const AdamConst &c, uint64_t pol_g, uint64_t pol_th,
                                       uint64_t pol_mv) {
#pragma unroll
    for (int f = 0; f < F; ++f) adam_one(th[f], m[f], v[f], g[f], c);
    store_entry_hint<F>(th_p, th, pol_th);
    if constexpr (F == 1) {
      st_hint_f2(mv_p, make_float2(m[0], v[0]), pol_mv);
    } else if constexpr (F == 2) {
      st_hint_f4(mv_p, make_float4(m[0], m[1], v[0], v[1]), pol_mv);
    } else {
      store_entry_hint<F>(mv_p, m, pol_mv);
      store_entry_hint<F>(mv_p + F, v, pol_mv);
    }
#pragma unroll
    for (int f = 0; f < F; ++f) g[f] = 0.f;
    store_entry_hint<F>(g_p, g, pol_g);
  }
};

// S13 for the ADAM_ENTRIES consecutive entries starting at e_base (a multiple of 32), by a block of ADAM_THREADS threads.
// The block reads its ADAM_WORDS words of the touched bitmap (512 contiguous bytes; the scatter set the bits), clears
// them, and expands the set bits into a list of local entry indices in shared memory -- ascending, so the threads of a
// warp update neighbouring touched entries and share sectors.  Every thread then takes UNROLL list entries at a time:
// all their loads (gradient, theta, moment record) are issued before the first update, so a thread keeps 3 x UNROLL
// independent DRAM / L2 accesses in flight.  Neither the gradient array nor theta / m|v of untouched entries is read:
// the traffic is what the touched set needs and nothing else.  sparse = 0 (dense Adam, textbook): every entry.
template <int F>
__device__ __forceinline__ void adam_block(float *__restrict__ theta, float *__restrict__ mv, float *__restrict__ grad,
                                           uint32_t *__restrict__ touched, uint64_t e_base, uint64_t n_entries, int sparse,
                                           const AdamConst &c, uint16_t *list_e, uint32_t *warp_tot) {
  constexpr int UNROLL = F <= 2 ? 4 : (F == 4 ? 2 : 1);
  const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  uint32_t wv = 0;
  if (tid < ADAM_WORDS) {
    const uint64_t e0 = e_base + 32ull * tid;
    if (e0 < n_entries) {
      uint32_t *wp = touched + (e0 >> 5);
      const uint32_t t = *wp;
      if (t) *wp = 0u;
      wv = sparse ? t : 0xffffffffu;
      const uint64_t rem = n_entries - e0;
      if (rem < 32) wv &= (1u << (uint32_t)rem) - 1u;
    }
  }
  // exclusive scan of the per-word counts over the ADAM_WORDS / 32 loading warps
  const uint32_t cnt = __popc(wv);
  uint32_t incl = cnt;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t y = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= (uint32_t)d) incl += y;
  }
  if (lane == 31 && warp < ADAM_WORDS / 32) warp_tot[warp] = incl;
  __syncthreads();
  uint32_t n = 0, pos = incl - cnt;
#pragma unroll
  for (uint32_t w = 0; w < ADAM_WORDS / 32; ++w) {
    const uint32_t t = warp_tot[w];
    if (w < warp) pos += t;
    n += t;
  }
  if (n == 0) return;
  while (wv) {
    const uint32_t b = (uint32_t)__ffs(wv) - 1u;
    wv &= wv - 1u;
    list_e[pos++] = (uint16_t)(tid * 32u + b);
  }
  __syncthreads();
  // L2 policies: the moment records are a pure stream (read once, written once per step): evict_first both ways.  The
  // gradient words were just written by the scatter (evict_last there) and theta is re-read by the next step's encoder.
  const uint64_t pol_n = l2_evict_normal(), pol_first = l2_evict_first();
  for (uint32_t i0 = tid; i0 < n; i0 += UNROLL * ADAM_THREADS) {
    AdamRec<F> r[UNROLL];
    uint64_t e[UNROLL];
#pragma unroll
    for (int u = 0; u < UNROLL; ++u) {
      const uint32_t i = i0 + u * ADAM_THREADS;
      e[u] = e_base + list_e[i < n ? i : i0];
      if (i < n) r[u].load(grad + e[u] * F, theta + e[u] * F, mv + e[u] * 2 * F, pol_n, pol_n, pol_first);
    }
#pragma unroll
    for (int u = 0; u < UNROLL; ++u) {
      const uint32_t i = i0 + u * ADAM_THREADS;
      if (i < n) r[u].step(grad + e[u] * F, theta + e[u] * F, mv + e[u] * 2 * F, c, pol_n, pol_first, pol_first);
    }
  }
}

}  // namespace tableops
