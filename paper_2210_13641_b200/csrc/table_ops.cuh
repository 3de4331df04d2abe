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

// L2 cache-policy words as compile-time constants (the values createpolicy.fractional.L2::evict_*.b64 ..., 1.0 returns;
// published in CUTLASS as CacheHintSm90).  A policy that is an immediate lives in a uniform register: with a policy held in
// a per-thread variable every hinted load paid two R2UR moves (the encoder's instruction stream, not its memory traffic,
// was what bounded it: profiles/r2k).
constexpr uint64_t NSM_L2_EVICT_NORMAL = 0x1000000000000000ull, NSM_L2_EVICT_FIRST = 0x12F0000000000000ull,
                   NSM_L2_EVICT_LAST = 0x14F0000000000000ull;
template <uint64_t POL>
__device__ __forceinline__ void st_pol_u4(void *p, uint4 v) {
  asm volatile("st.global.L2::cache_hint.v4.b32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "l"(POL) : "memory");
}
template <uint64_t POL>
__device__ __forceinline__ float4 ld_pol_f4(const float *p) {
  float4 v;
  asm volatile("ld.global.L2::cache_hint.v4.f32 {%0, %1, %2, %3}, [%4], %5;"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(POL) : "memory");
  return v;
}
template <uint64_t POL>
__device__ __forceinline__ float2 ld_pol_f2(const float *p) {
  float2 v;
  asm volatile("ld.global.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(POL) : "memory");
  return v;
}

// S4's gather for one (sample, level): the eight corner entries of the level slice `tab` (= theta + offset_l F, 16-byte
// aligned: EntryMap).  F = 2: the x-neighbour corners (k, k + 1) are one aligned 16-byte pair of entries whenever their
// slots differ in bit 0 only -- on a dense level for every even slot, on a hashed level for every even cell x (the hash
// XORs x in unmultiplied) -- and then come in with one load.  All index arithmetic is 32-bit.
template <int F, uint64_t POL>
__device__ __forceinline__ void gather_corners(const float *__restrict__ tab, const uint32_t slot[8], float v[8][F]) {
  // the slice pointer as one opaque 64-bit register pair: every address below is then a single IMAD.WIDE (left to itself
  // the compiler re-adds table base, level offset and slot with carries for each of the twelve loads)
  asm volatile("" : "+l"(tab));
  if constexpr (F == 2) {
#pragma unroll
    for (int k = 0; k < 8; k += 2) {
      const uint32_t s0 = slot[k], s1 = slot[k + 1];
      if ((s0 ^ s1) == 1u) {
        const float4 q = ld_pol_f4<POL>(tab + 4 * (size_t)(s0 >> 1));
        const bool odd = s0 & 1u;
        v[k][0] = odd ? q.z : q.x; v[k][1] = odd ? q.w : q.y;
        v[k + 1][0] = odd ? q.x : q.z; v[k + 1][1] = odd ? q.y : q.w;
      } else {
        const float2 a = ld_pol_f2<POL>(tab + 2 * (size_t)s0), b = ld_pol_f2<POL>(tab + 2 * (size_t)s1);
        v[k][0] = a.x; v[k][1] = a.y; v[k + 1][0] = b.x; v[k + 1][1] = b.y;
      }
    }
  } else {
#pragma unroll
    for (int k = 0; k < 8; ++k) load_entry_hint<F>(tab + (size_t)slot[k] * F, v[k], POL);   // 8 gathers in flight
  }
}

// S12 for one cell of one level: the eight corner reductions d theta[(offset_l + slot) F + f] += val[corner][f].
// Addends are canonicalised here (never -0.0, never near-subnormal; NaN stays NaN): the touched set U is structural
// (every referenced entry, independent of the gradient's value) and is carried by the gradient words themselves, see
// FieldParams in nsm_internal.cuh.
template <int F>
__device__ __forceinline__ void issue_corner_reds(const LevelTable &lv, float *__restrict__ grad, uint32_t l, const uint32_t slot[8],
                                                  float val[8][F], uint64_t pol_last) {
#pragma unroll
  for (int k = 0; k < 8; ++k)
#pragma unroll
    for (int f = 0; f < F; ++f) val[k][f] = fabsf(val[k][f]) < NSM_GRAD_MIN_ADDEND ? 0.0f : val[k][f];
  float *tab = grad + lv.offset[l] * F;
  if constexpr (F == 2) {
    // The two x-neighbour corners (k, k+1) are adjacent entries whenever their slots differ in bit 0 only (always on
    // a dense level, for even cell x on a hashed one: the hash XORs x in unmultiplied).  If the pair is also
    // 16-byte aligned in the array, one red.v4 covers both entries: ~25 % fewer reductions at the L2.
    // (the level slice starts on a 16-byte boundary, EntryMap: the pair test needs the slots only)
#pragma unroll
    for (int k = 0; k < 8; k += 2) {
      const uint32_t s0 = slot[k], s1 = slot[k + 1];
      if ((s0 ^ s1) == 1u) {
        float *p = tab + 2 * (size_t)(s0 & ~1u);
        if (s0 & 1u) red_hint_f4(p, make_float4(val[k + 1][0], val[k + 1][1], val[k][0], val[k][1]), pol_last);
        else red_hint_f4(p, make_float4(val[k][0], val[k][1], val[k + 1][0], val[k + 1][1]), pol_last);
      } else {
        red_add_entry<2>(tab + (size_t)slot[k] * 2, val[k], pol_last);
        red_add_entry<2>(tab + (size_t)slot[k + 1] * 2, val[k + 1], pol_last);
      }
    }
  } else {
#pragma unroll
    for (int k = 0; k < 8; ++k) red_add_entry<F>(tab + (size_t)slot[k] * F, val[k], pol_last);
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
__device__ __forceinline__ void scatter_sample_level(const LevelTable &lv, float *__restrict__ grad, const Workspace &ws,
                                                     uint32_t l, uint64_t s, uint64_t pol_last) {
  uint32_t slot[8];
  float val[8][F];
  corner_contributions<F>(lv, ws, l, s, slot, val);
  issue_corner_reds<F>(lv, grad, l, slot, val, pol_last);
}

constexpr int ADAM_CHUNK_FLOATS = 4096;
constexpr int ADAM_THREADS = 256;

// one touched entry: theta (F floats of the compact array) and its moment record (m | v, 2F floats)
template <int F>
__device__ __forceinline__ void adam_entry(float *__restrict__ th_p, float *__restrict__ mv_p, const float *g, const AdamConst &c,
                                           uint64_t pol_ld, uint64_t pol_st, uint64_t pol_th) {
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
    st_hint_f1(th_p, th[0], pol_th);
    st_hint_f2(mv_p, make_float2(m[0], v[0]), pol_st);
  } else if constexpr (F == 2) {
    st_hint_f2(th_p, make_float2(th[0], th[1]), pol_th);
    st_hint_f4(mv_p, make_float4(m[0], m[1], v[0], v[1]), pol_st);
  } else {
#pragma unroll
    for (int i = 0; i < F / 4; ++i) {
      st_hint_f4(th_p + 4 * i, make_float4(th[4 * i], th[4 * i + 1], th[4 * i + 2], th[4 * i + 3]), pol_th);
      st_hint_f4(mv_p + 4 * i, make_float4(m[4 * i], m[4 * i + 1], m[4 * i + 2], m[4 * i + 3]), pol_st);
      st_hint_f4(mv_p + F + 4 * i, make_float4(v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]), pol_st);
    }
  }
}

// S13 for one chunk of ADAM_CHUNK_FLOATS / F consecutive entries starting at e_base (e_base * F a multiple of 4),
// by a whole block of ADAM_THREADS threads.  Shared memory: list_g [ADAM_CHUNK_FLOATS], list_e [CH], cnt_p.  The caller
// must __syncthreads() before reusing the shared arrays.
template <int F>
__device__ __forceinline__ void adam_chunk(float *__restrict__ theta, float *__restrict__ mv, float *__restrict__ grad,
                                           uint64_t e_base, uint64_t n_entries, int sparse, const AdamConst &c, float *list_g,
                                           uint16_t *list_e, uint32_t *cnt_p, int theta_resident) {
  constexpr int CH = ADAM_CHUNK_FLOATS / F;            // entries per chunk
  constexpr int NV = ADAM_CHUNK_FLOATS / 4 / ADAM_THREADS;   // float4 loads per thread
  const uint32_t tid = threadIdx.x, lane = tid & 31;
  const uint64_t n_float = n_entries * F;
  const float *g4 = grad + e_base * F;
  // L2 policies, swept on B200 (profiles/r1k): theta / moment stores evict_first, everything else default.  Marking
  // Adam's own gradient reads and resets evict_last (as the scatter's reductions are) costs 4 us per step.
  // theta_resident (tables that fit the L2): the updated theta stays for the next step's encoder (default policy)
  const uint64_t pol_ld = l2_evict_normal(), pol_first = l2_evict_first(), pol_last = pol_ld;
  const uint64_t pol_th = theta_resident ? pol_ld : pol_first;
  if (tid == 0) *cnt_p = 0;
  float4 gv[NV];
  uint32_t dirty = 0;                                  // bit j: the thread's j-th 16-byte word holds a touched entry
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
        if (t) dirty |= 1u << j;
        const uint32_t mk = __ballot_sync(0xffffffffu, t);
        uint32_t base = 0;
        if (lane == 0 && mk) base = atomicAdd(cnt_p, (uint32_t)__popc(mk));
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
      if (t) dirty |= 1u << j;
      const uint32_t mk = __ballot_sync(0xffffffffu, t && !(lane & 1u));
      uint32_t base = 0;
      if (lane == 0 && mk) base = atomicAdd(cnt_p, (uint32_t)__popc(mk));
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
  const uint32_t n = *cnt_p;
  if (n == 0) return;
  // phase 2: two records in flight per thread
  for (uint32_t i0 = tid; i0 < n; i0 += 2 * ADAM_THREADS) {
    const uint32_t i1 = i0 + ADAM_THREADS;
    const uint64_t e0 = e_base + list_e[i0], e1 = e_base + list_e[i1 < n ? i1 : i0];
    if constexpr (F == 2) {   // touch the second entry's moment record early
      asm volatile("prefetch.global.L2 [%0];" ::"l"(mv + e1 * 2 * F));
    }
    adam_entry<F>(theta + e0 * F, mv + e0 * 2 * F, list_g + i0 * F, c, pol_ld, pol_first, pol_th);
    if (i1 < n) adam_entry<F>(theta + e1 * F, mv + e1 * 2 * F, list_g + i1 * F, c, pol_ld, pol_first, pol_th);
  }
  // reset the chunk's gradient words
  float *o4 = grad + e_base * F;
  const float nz = __uint_as_float(NSM_GRAD_UNTOUCHED);
#pragma unroll
  for (int j = 0; j < NV; ++j) {
    const uint32_t q = j * ADAM_THREADS + tid;
    // only the words that held a touched entry: the others are -0.0 already (with tables far larger than the L2 the
    // dense rewrite was half of this kernel's DRAM traffic)
    if (((dirty >> j) & 1u) && e_base * F + 4ull * q < n_float) st_hint_f4(o4 + 4 * q, make_float4(nz, nz, nz, nz), pol_last);
  }
}

}  // namespace tableops
