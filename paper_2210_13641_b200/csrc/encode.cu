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
#include "table_ops.cuh"

namespace {

using namespace tableops;

#ifndef NSM_PANEL_HASHED_POL
#define NSM_PANEL_HASHED_POL NSM_L2_EVICT_LAST
#endif

// MODE 0: e -> fp32 planes [l*F+f][cap].  MODE 1 / 2: e -> fp16 / bf16 operand-tile blob of the
// tensor-core MLP kernels ([tile][8-column panel][128 rows][8 x 16 bit], mlp_tc.cu); the rows of
// the last tile beyond S are zero-filled so the MMA never reads stale data.
// TWO_TERM = false (forward-only uses: render, occupancy refresh -- their MLP kernel reads the hi tile only): the lo term is
// neither computed nor stored.
// F = 4: capped at 64 registers (80 otherwise) for four blocks per SM: with tables beyond the L2 the kernel waits for
// DRAM and a fourth block's gathers in flight are worth 2 % (config 4: 148.8 -> 146.2 us; five blocks spill: 151.8 us).
// (0 = no minimum, the compiler's own choice: 47 registers at F = 2; a minimum of 1 lets it take 72.)
template <int F, int MODE, bool TWO_TERM = true>
__global__ void __launch_bounds__(256, F == 4 ? 4 : 0) encode_forward_kernel(LevelTable lv, const float *__restrict__ theta,
                                                             Workspace ws, const uint32_t *__restrict__ d_S, uint32_t seq,
                                                             uint32_t stream_hashed) {
  __shared__ uint32_t chunk_s;
  pdl_wait();
  pdl_trigger();
  tl_mark(ws.timeline, K_ENCODE, 0);
  const uint64_t S = *d_S;
  const uint64_t S_it = MODE == 0 ? S : ((S + NSM_TILE - 1) / NSM_TILE) * NSM_TILE;
  const uint64_t total = S_it * lv.n_levels;
  const uint32_t LF = lv.n_levels * F;
  const uint32_t lane = threadIdx.x & 31;
  ChunkQueue q(ws.work_ctr, seq);
  for (;;) {   // 256 consecutive (level, sample) items at a time, handed out in order (see ChunkQueue); warp-uniform
    const uint64_t cb = q.next(&chunk_s);
    if (cb >= total) break;                        // block-uniform
    const uint64_t wb = cb + (threadIdx.x & ~31u);
    if (wb >= total) continue;                     // warp-uniform (the last, partial chunk)
    const uint64_t wi = wb + lane;
    const bool in_range = wi < total;
    const uint32_t l = (uint32_t)((in_range ? wi : wb) / S_it);
    const uint64_t s = (in_range ? wi : wb) - (uint64_t)l * S_it;
    const bool live = in_range && s < S;
    float acc[F];
#pragma unroll
    for (int f = 0; f < F; ++f) acc[f] = 0.0f;
    // On a dense (coarse) level consecutive samples of a ray share their cell for several steps: when the warp holds one
    // dense level, only the first lane of each run of equal cells gathers the eight corners, the others take them by
    // shuffle (the L2's random-access rate bounds this kernel, profiles/r1p).
    const uint32_t l_first = __shfl_sync(0xffffffffu, l, 0);
    const bool one_dense_level = __all_sync(0xffffffffu, l == l_first) && lv.dense[l_first];
    CornerIndex ci;
    if (live) ci = corner_index(lv, l, ws.s_x[s], ws.s_x[ws.cap + s], ws.s_x[2 * ws.cap + s]);
    uint32_t head_lane = lane;
    bool gathers = live;
    if (one_dense_level) {
      const uint32_t key = live ? ci.slot[0] : 0xffffffffu - lane;
      const uint32_t prev = __shfl_up_sync(0xffffffffu, key, 1);
      const uint32_t heads = __ballot_sync(0xffffffffu, lane == 0 || key != prev);
      head_lane = 31u - (uint32_t)__clz(heads & (0xffffffffu >> (31u - lane)));
      gathers = live && head_lane == lane;
    }
    float v[8][F];
#pragma unroll
    for (int k = 0; k < 8; ++k)
#pragma unroll
      for (int f = 0; f < F; ++f) v[k][f] = 0.f;
    if (gathers) {
      const float *tab = theta + lv.offset[l] * F;
      // coarse (dense) levels are re-read every step: default policy.  Hashed levels: evict_first where the tables are
      // L2-sized and a small step references an entry less than once (stream_hashed, config 2: the lines would only push the
      // gradient array out, scatter 19 -> 24 us with the default policy); default where the tables dwarf the L2 (config 4:
      // a fetched sector is met again by the next samples of the ray within microseconds, and "evict first" lines do not
      // live that long under 0.5 GB of misses: encode 142 -> 117 us)
      if (lv.dense[l] || !stream_hashed) gather_corners<F, NSM_L2_EVICT_NORMAL>(tab, ci.slot, v);
      else gather_corners<F, NSM_L2_EVICT_FIRST>(tab, ci.slot, v);
    }
    if (one_dense_level) {
#pragma unroll
      for (int k = 0; k < 8; ++k)
#pragma unroll
        for (int f = 0; f < F; ++f) v[k][f] = __shfl_sync(0xffffffffu, v[k][f], head_lane);
    }
    if (live) {
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        float om = corner_weight(k, ci.w);
#pragma unroll
        for (int f = 0; f < F; ++f) acc[f] = fmaf(om, v[k][f], acc[f]);
      }
    }
    if (!in_range) continue;
    if (MODE == 0) {
#pragma unroll
      for (int f = 0; f < F; ++f) ws.e[(size_t)(l * F + f) * ws.cap + s] = acc[f];
    } else {
      const uint32_t c = l * F;   // F consecutive columns never straddle an 8-column panel (F | 8)
      // two-term tile: [hi: LF*256 bytes][lo: LF*256 bytes] per 128-sample tile (e = hi + lo)
      const size_t half = (size_t)LF * NSM_TILE * 2;
      uint8_t *dst = ws.blob_e + (s >> 7) * (2 * half) + (c >> 3) * (NSM_TILE * 16) + (s & 127) * 16 + (c & 7) * 2;
      // the F columns of the level are adjacent 16-bit elements of one panel row: one store per term (F = 2: 4 bytes)
      uint16_t hi16[F], lo16[F];
#pragma unroll
      for (int f = 0; f < F; ++f) {
        if (MODE == 1) {
          const __half hi = __float2half_rn(acc[f]);
          hi16[f] = __half_as_ushort(hi);
          lo16[f] = TWO_TERM ? __half_as_ushort(__float2half_rn(acc[f] - __half2float(hi))) : (uint16_t)0;
        } else {
          const __nv_bfloat16 hi = __float2bfloat16_rn(acc[f]);
          hi16[f] = __bfloat16_as_ushort(hi);
          lo16[f] = TWO_TERM ? __bfloat16_as_ushort(__float2bfloat16_rn(acc[f] - __bfloat162float(hi))) : (uint16_t)0;
        }
      }
      if constexpr (F == 1) {
        *reinterpret_cast<uint16_t *>(dst) = hi16[0];
        if (TWO_TERM) *reinterpret_cast<uint16_t *>(dst + half) = lo16[0];
      } else {
        uint32_t hw[F / 2], lw[F / 2];
#pragma unroll
        for (int i = 0; i < F / 2; ++i) {
          hw[i] = (uint32_t)hi16[2 * i] | ((uint32_t)hi16[2 * i + 1] << 16);
          lw[i] = (uint32_t)lo16[2 * i] | ((uint32_t)lo16[2 * i + 1] << 16);
        }
        if constexpr (F == 2) {
          *reinterpret_cast<uint32_t *>(dst) = hw[0];
          if (TWO_TERM) *reinterpret_cast<uint32_t *>(dst + half) = lw[0];
        } else if constexpr (F == 4) {
          *reinterpret_cast<uint2 *>(dst) = make_uint2(hw[0], hw[1]);
          if (TWO_TERM) *reinterpret_cast<uint2 *>(dst + half) = make_uint2(lw[0], lw[1]);
        } else {
          *reinterpret_cast<uint4 *>(dst) = make_uint4(hw[0], hw[1], hw[2], hw[3]);
          if (TWO_TERM) *reinterpret_cast<uint4 *>(dst + half) = make_uint4(lw[0], lw[1], lw[2], lw[3]);
        }
      }
    }
  }
  tl_mark(ws.timeline, K_ENCODE, 1);
}

// The same for the tensor-core path, one thread per (PANEL of 8 columns, sample): the 8 / F levels whose features fill one
// 8-column panel of the operand tile.  The thread then owns a whole 16-byte panel row chunk of the hi and of the lo tile:
// a warp writes 512 contiguous bytes per store instead of 4-byte pieces at a 16-byte stride (partial-sector writes were
// what the L2 spent its time on: one store per term and level took config 3's encoder from 200.8 to 175.1 us, this
// mapping to 155.4 us), and the sample position is loaded once per panel.  Items are panel-major, 256 per chunk, in
// order.  launch_encode picks between the two mappings.
template <int F, int MODE, bool TWO_TERM = true>
__global__ void __launch_bounds__(256) encode_forward_panel_kernel(LevelTable lv, const float *__restrict__ theta, Workspace ws,
                                                                   const uint32_t *__restrict__ d_S, uint32_t seq) {
  static_assert(MODE == 1 || MODE == 2, "operand-tile output only");
  constexpr int LPG = 8 / F;                       // levels per panel
  __shared__ uint32_t chunk_s;
  pdl_wait();
  pdl_trigger();
  tl_mark(ws.timeline, K_ENCODE, 0);
  const uint64_t S = *d_S;
  const uint64_t S_it = ((S + NSM_TILE - 1) / NSM_TILE) * NSM_TILE;     // whole tiles: rows beyond S are zero-filled
  const uint32_t LF = lv.n_levels * F, n_panels = LF / 8;               // LF is a multiple of 16 on this path
  const uint64_t total = S_it * n_panels;
  const uint32_t lane = threadIdx.x & 31;
  const size_t half = (size_t)LF * NSM_TILE * 2;   // two-term tile: [hi: LF*256 bytes][lo: LF*256 bytes] per 128-sample tile
  ChunkQueue q(ws.work_ctr, seq);
  for (;;) {
    const uint64_t cb = q.next(&chunk_s);
    if (cb >= total) break;                        // block-uniform
    const uint64_t wi = cb + threadIdx.x;          // S_it is a multiple of 128: a warp never straddles two panels
    if (wi >= total) continue;                     // (total is a multiple of 128 too: warp-uniform)
    const uint32_t g = (uint32_t)(wi / S_it);
    const uint64_t s = wi - (uint64_t)g * S_it;
    const bool live = s < S;
    float x0 = 0.f, x1 = 0.f, x2 = 0.f;
    if (live) { x0 = ws.s_x[s]; x1 = ws.s_x[ws.cap + s]; x2 = ws.s_x[2 * ws.cap + s]; }
    uint32_t hw[4] = {0u, 0u, 0u, 0u}, lw[4] = {0u, 0u, 0u, 0u};        // the 8 columns of the panel row, hi and lo terms
#pragma unroll
    for (int j = 0; j < LPG; ++j) {
      const uint32_t l = g * LPG + j;              // warp-uniform
      float acc[F];
#pragma unroll
      for (int f = 0; f < F; ++f) acc[f] = 0.0f;
      const bool dense = lv.dense[l];
      CornerIndex ci;
      if (live) ci = corner_index(lv, l, x0, x1, x2);
      // dense (coarse) level: only the first lane of each run of equal cells gathers, the run takes the corners by shuffle
      uint32_t head_lane = lane;
      bool gathers = live;
      if (dense) {
        const uint32_t key = live ? ci.slot[0] : 0xffffffffu - lane;
        const uint32_t prev = __shfl_up_sync(0xffffffffu, key, 1);
        const uint32_t heads = __ballot_sync(0xffffffffu, lane == 0 || key != prev);
        head_lane = 31u - (uint32_t)__clz(heads & (0xffffffffu >> (31u - lane)));
        gathers = live && head_lane == lane;
      }
      float v[8][F];
#pragma unroll
      for (int k = 0; k < 8; ++k)
#pragma unroll
        for (int f = 0; f < F; ++f) v[k][f] = 0.f;
      if (gathers) {
        const float *tab = theta + lv.offset[l] * F;
        if (dense) gather_corners<F, NSM_L2_EVICT_NORMAL>(tab, ci.slot, v);
        else gather_corners<F, NSM_PANEL_HASHED_POL>(tab, ci.slot, v);
      }
      if (dense) {
#pragma unroll
        for (int k = 0; k < 8; ++k)
#pragma unroll
          for (int f = 0; f < F; ++f) v[k][f] = __shfl_sync(0xffffffffu, v[k][f], head_lane);
      }
      if (live) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          const float om = corner_weight(k, ci.w);
#pragma unroll
          for (int f = 0; f < F; ++f) acc[f] = fmaf(om, v[k][f], acc[f]);
        }
      }
#pragma unroll
      for (int f = 0; f < F; ++f) {
        uint32_t h16, l16;
        if (MODE == 1) {
          const __half hi = __float2half_rn(acc[f]);
          h16 = __half_as_ushort(hi);
          l16 = TWO_TERM ? __half_as_ushort(__float2half_rn(acc[f] - __half2float(hi))) : 0u;
        } else {
          const __nv_bfloat16 hi = __float2bfloat16_rn(acc[f]);
          h16 = __bfloat16_as_ushort(hi);
          l16 = TWO_TERM ? __bfloat16_as_ushort(__float2bfloat16_rn(acc[f] - __bfloat162float(hi))) : 0u;
        }
        const int col = j * F + f;                 // column inside the panel, compile-time
        hw[col >> 1] |= h16 << ((col & 1) * 16);
        lw[col >> 1] |= l16 << ((col & 1) * 16);
      }
    }
    uint8_t *dst = ws.blob_e + (s >> 7) * (2 * half) + (size_t)g * (NSM_TILE * 16) + (s & 127) * 16;
    st_pol_u4<NSM_L2_EVICT_FIRST>(dst, make_uint4(hw[0], hw[1], hw[2], hw[3]));
    if (TWO_TERM) st_pol_u4<NSM_L2_EVICT_FIRST>(dst + half, make_uint4(lw[0], lw[1], lw[2], lw[3]));
  }
  tl_mark(ws.timeline, K_ENCODE, 1);
}

// S12, thread per (level, sample), level-major (see table_ops.cuh).  On DENSE (coarse) levels consecutive samples of a
// ray sit in the same cell for several steps (level 0: ~6 samples per cell at config 3), and every sample of a cell adds
// to the same eight entries: when a warp holds one dense level, the contributions of each run of equal cells are summed
// with a segmented warp scan and only the run's first lane issues the reductions -- the L2 reduction rate is what bounds
// this kernel (profiles/r1p), so fewer reductions is the only way to make it faster.
template <int F>
__global__ void __launch_bounds__(256) scatter_backward_kernel(LevelTable lv, float *__restrict__ grad, Workspace ws,
                                                               const uint32_t *__restrict__ d_S, uint32_t l0, uint32_t l1, int prefetch,
                                                               uint32_t seq) {
  __shared__ uint32_t chunk_s;
  pdl_wait();
  pdl_trigger();
  tl_mark(ws.timeline, K_SCATTER, 0);
  const uint64_t S = *d_S;
  const uint64_t total = S * (l1 - l0);
  const uint64_t pol_last = l2_evict_last();
  const uint32_t lane = threadIdx.x & 31;
  const uint32_t nl = l1 - l0;
  const uint64_t n_sc = (S + 255) / 256;              // 256-sample chunks per level
  const uint64_t n_chunks = prefetch ? (total + 255) / 256 : n_sc * nl;
  const uint64_t stride = (uint64_t)prefetch * 256;   // prefetch distance: that many chunks ahead of the one in hand
  ChunkQueue q(ws.work_ctr, seq);
  for (;;) {   // 256 (level, sample) items at a time, handed out in order; warp-uniform
    const uint64_t c = q.next(&chunk_s) / 256;
    if (c >= n_chunks) break;                          // block-uniform
    // Two chunk orders.  Tables beyond the L2 (prefetch != 0): level-major, chunk c = items [256 c, 256 c + 256) of the
    // level-major item list, so the chip stays inside one level's slice (ChunkQueue).  L2-resident tables: chunk c =
    // samples [256 (c / nl), ...) of level c % nl, so the chunks in flight cover all levels evenly -- with every block
    // on the same coarse level at once, its few thousand entries serialise the whole chip's reductions (measured at
    // config 3: 285 us level-major, 269 us with the levels spread).
    uint64_t wi, wb;                                   // this lane's item and its warp's first item (level-major indices)
    if (prefetch) {
      wb = c * 256 + (threadIdx.x & ~31u);
      wi = wb + lane;
    } else {
      const uint64_t s0 = (c / nl) * 256 + (threadIdx.x & ~31u);
      wb = (uint64_t)(c % nl) * S + s0;
      wi = s0 + lane < S ? wb + lane : total;
      if (s0 >= S) wb = total;
    }
    if (wb >= total) continue;                         // warp-uniform (partial chunks)
    const bool valid = wi < total;
    const uint32_t l = l0 + (uint32_t)((valid ? wi : wb) / S);
    const uint64_t s = (valid ? wi : wb) - (uint64_t)(l - l0) * S;
    const uint32_t l_first = __shfl_sync(0xffffffffu, l, 0);
    const bool one_dense_level = __all_sync(0xffffffffu, l == l_first) && lv.dense[l_first];
    if (prefetch) {
      // Tables far larger than the L2 (config 4): a reduction that misses waits in the L2's atomic unit for its DRAM fill,
      // and that unit tracks far fewer misses than the read path (in situ: 0.98 GB of DRAM traffic in 349 us = 2.8 TB/s,
      // while the encoder's plain loads reach 5.1 TB/s).  So the sectors a LATER chunk's item will reduce into are
      // requested now, as L2 prefetches: by the time the reductions arrive (`prefetch` chunks later) they hit.
      const uint64_t wn = wi + stride;
      if (wn < total) {
        const uint32_t ln = l0 + (uint32_t)(wn / S);
        const uint64_t sn = wn - (uint64_t)(ln - l0) * S;
        if (!lv.dense[ln]) {
          const CornerIndex cn = corner_index(lv, ln, ws.s_x[sn], ws.s_x[ws.cap + sn], ws.s_x[2 * ws.cap + sn]);
          const float *tab = grad + lv.offset[ln] * F;
          // one request per sector: an x-neighbour pair (slots s, s ^ 1) lies in one 32-byte sector for F <= 4 (EntryMap)
#pragma unroll
          for (int k = 0; k < 8; k += 2) {
            asm volatile("prefetch.global.L2::evict_last [%0];" ::"l"(tab + (size_t)cn.slot[k] * F));
            if (F > 4 || (cn.slot[k] ^ cn.slot[k + 1]) != 1u)
              asm volatile("prefetch.global.L2::evict_last [%0];" ::"l"(tab + (size_t)cn.slot[k + 1] * F));
          }
        }
      }
    }
    if (!one_dense_level) {
      if (valid) scatter_sample_level<F>(lv, grad, ws, l, s, pol_last);
      continue;
    }
    uint32_t slot[8];
    float val[8][F];
    corner_contributions<F>(lv, ws, l, s, slot, val);
    // runs of equal cells (slot[0] identifies the cell on a dense level); invalid lanes form runs of their own
    const uint32_t key = valid ? slot[0] : 0xffffffffu - lane;
    const uint32_t prev = __shfl_up_sync(0xffffffffu, key, 1);
    const uint32_t heads = __ballot_sync(0xffffffffu, lane == 0 || key != prev);
    const uint32_t later = lane == 31 ? 0u : heads >> (lane + 1);
    const uint32_t run_end = later ? lane + (uint32_t)__ffs(later) : 32u;      // first lane of the next run
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {   // segmented suffix sum: the run's first lane ends up with the run's total
#pragma unroll
      for (int k = 0; k < 8; ++k)
#pragma unroll
        for (int f = 0; f < F; ++f) {
          const float o = __shfl_down_sync(0xffffffffu, val[k][f], d);
          if (lane + d < run_end) val[k][f] += o;
        }
    }
    if (valid && ((heads >> lane) & 1u)) issue_corner_reds<F>(lv, grad, l, slot, val, pol_last);
  }
  tl_mark(ws.timeline, K_SCATTER, 1);
}

// canonical entry -> storage entry (EntryMap, nsm_internal.cuh)
__device__ __forceinline__ uint64_t storage_entry(const EntryMap &m, uint64_t e_canon) {
  uint32_t l = 0;
  while (l + 1 < m.n_levels && e_canon >= m.canon[l + 1]) ++l;
  return m.storage[l] + (e_canon - m.canon[l]);
}
// storage entry -> canonical entry, or ~0 for a padding entry
__device__ __forceinline__ uint64_t canonical_entry(const EntryMap &m, uint64_t e_storage) {
  uint32_t l = 0;
  while (l + 1 < m.n_levels && e_storage >= m.storage[l + 1]) ++l;
  const uint64_t i = e_storage - m.storage[l];
  return i < m.canon[l + 1] - m.canon[l] ? m.canon[l] + i : ~0ull;
}

// gradient array <- canonical gradient and flags (debug / test entry point); walks the STORAGE array, padding included
__global__ void set_grad_kernel(float *__restrict__ grad, uint32_t F, uint64_t n_entries, EntryMap map, const float *__restrict__ src,
                                const uint8_t *__restrict__ touched) {
  const uint64_t total = n_entries * F;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t es = i / F;
    const uint64_t e = src ? canonical_entry(map, es) : ~0ull;
    const bool t = e != ~0ull && (!touched || touched[e]);
    const float v = t ? src[e * F + (i - es * F)] : 0.f;
    grad[i] = t ? (fabsf(v) < NSM_GRAD_MIN_ADDEND ? 0.0f : v) : __uint_as_float(NSM_GRAD_UNTOUCHED);
  }
}

__global__ void get_touched_kernel(const float *__restrict__ grad, uint32_t F, uint64_t n_canon, EntryMap map, uint8_t *__restrict__ dst) {
  for (uint64_t e = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; e < n_canon; e += (uint64_t)gridDim.x * blockDim.x)
    dst[e] = __float_as_uint(grad[storage_entry(map, e) * F]) != NSM_GRAD_UNTOUCHED;
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
  return which <= 1 ? e * F + f : e * 2 * F + (which == 3 ? F : 0) + f;
}

// walks the STORAGE arrays: padding entries become zeros
__global__ void pack_records_kernel(float *__restrict__ theta, float *__restrict__ mv, uint32_t F, uint64_t n_entries, EntryMap map,
                                    int which, const float *__restrict__ src) {
  const uint64_t total = n_entries * F;
  float *dst = which == 0 ? theta : mv;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t es = i / F;
    const uint32_t f = (uint32_t)(i - es * F);
    const uint64_t e = src ? canonical_entry(map, es) : ~0ull;
    dst[param_index(F, es, f, which)] = e != ~0ull ? src[e * F + f] : 0.f;
  }
}

// walks the canonical array; which == 1: the gradient array ("untouched" words read as -0.0)
__global__ void unpack_records_kernel(const float *__restrict__ theta, const float *__restrict__ mv, const float *__restrict__ grad,
                                      uint32_t F, uint64_t n_canon, EntryMap map, int which, float *__restrict__ dst) {
  const uint64_t total = n_canon * F;
  const float *src = which == 0 ? theta : (which == 1 ? grad : mv);
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t e = i / F;
    dst[i] = src[param_index(F, storage_entry(map, e), (uint32_t)(i - e * F), which)];
  }
}

}  // namespace

int launch_pack_records(const FieldParams &fp, int which, const float *src, cudaStream_t st) {
  pack_records_kernel<<<2048, 256, 0, st>>>(fp.theta, fp.mv, fp.F, fp.n_entries, fp.map, which, src);
  return 1;
}

int launch_unpack_records(const FieldParams &fp, int which, float *dst, cudaStream_t st) {
  unpack_records_kernel<<<2048, 256, 0, st>>>(fp.theta, fp.mv, fp.grad, fp.F, fp.n_canon, fp.map, which, dst);
  return 1;
}

template <int F, bool TT>
static void launch_encode_ft(const LevelTable &lv, const float *theta, const Workspace &ws, const uint32_t *d_S, int out_mode,
                             dim3 grid, dim3 block, cudaStream_t st, uint32_t seq, bool per_panel, uint32_t stream_hashed) {
  if (out_mode == 1) {
    if (per_panel) launch_pdl(encode_forward_panel_kernel<F, 1, TT>, grid, block, 0, st, lv, theta, ws, d_S, seq);
    else launch_pdl(encode_forward_kernel<F, 1, TT>, grid, block, 0, st, lv, theta, ws, d_S, seq, stream_hashed);
  } else {
    if (per_panel) launch_pdl(encode_forward_panel_kernel<F, 2, TT>, grid, block, 0, st, lv, theta, ws, d_S, seq);
    else launch_pdl(encode_forward_kernel<F, 2, TT>, grid, block, 0, st, lv, theta, ws, d_S, seq, stream_hashed);
  }
}

template <int F>
static void launch_encode_f(const LevelTable &lv, const float *theta, const Workspace &ws, const uint32_t *d_S, int out_mode,
                            dim3 grid, dim3 block, cudaStream_t st, uint32_t seq, bool per_panel, bool two_term,
                            uint32_t stream_hashed) {
  if (out_mode == 0) launch_pdl(encode_forward_kernel<F, 0>, grid, block, 0, st, lv, theta, ws, d_S, seq, stream_hashed);
  else if (two_term) launch_encode_ft<F, true>(lv, theta, ws, d_S, out_mode, grid, block, st, seq, per_panel, stream_hashed);
  else launch_encode_ft<F, false>(lv, theta, ws, d_S, out_mode, grid, block, st, seq, per_panel, stream_hashed);
}

int launch_encode(const LevelTable &lv, const float *theta, const Workspace &ws, const uint32_t *d_S, int out_mode,
                  int n_sms, cudaStream_t st, uint32_t seq, uint64_t max_samples, bool two_term) {
  dim3 grid(n_sms * 8), block(256);
  // Which mapping (measured on B200, profiles/r2g): a thread per (panel, sample) writes whole 16-byte rows of the operand
  // tile and wins when the tables fit the L2 and there is enough work to fill the chip with a quarter of the threads
  // (config 3: 175 -> 155 us, config 5: 12.4 -> 10.4 ms per two views); a thread per (level, sample) keeps the chip inside
  // one level's slice of tables beyond the L2 (config 4: 159 against 167 us) and has four times the threads when a step
  // has few samples (config 2, 22 K samples: 19.4 against 22.5 us).  S itself is only known on the device: the switch
  // uses the step's upper bound, rays x candidates.
  const bool l2_resident = lv.offset[lv.n_levels] * lv.n_features * sizeof(float) <= (96ull << 20);
  const bool per_panel = out_mode != 0 && l2_resident && max_samples >= (1ull << 20);
  const uint32_t stream_hashed = l2_resident ? 1u : 0u;   // the thread-per-(level, sample) kernel's hashed-level gather policy
  switch (lv.n_features) {
    case 1: launch_encode_f<1>(lv, theta, ws, d_S, out_mode, grid, block, st, seq, per_panel, two_term, stream_hashed); break;
    case 2: launch_encode_f<2>(lv, theta, ws, d_S, out_mode, grid, block, st, seq, per_panel, two_term, stream_hashed); break;
    case 4: launch_encode_f<4>(lv, theta, ws, d_S, out_mode, grid, block, st, seq, per_panel, two_term, stream_hashed); break;
    default: launch_encode_f<8>(lv, theta, ws, d_S, out_mode, grid, block, st, seq, per_panel, two_term, stream_hashed); break;
  }
  return 1;
}

int launch_set_grad(const FieldParams &fp, const float *src, const uint8_t *touched, cudaStream_t st) {
  set_grad_kernel<<<2048, 256, 0, st>>>(fp.grad, fp.F, fp.n_entries, fp.map, src, touched);
  return 1;
}

int launch_get_touched(const FieldParams &fp, uint8_t *dst, cudaStream_t st) {
  get_touched_kernel<<<2048, 256, 0, st>>>(fp.grad, fp.F, fp.n_canon, fp.map, dst);
  return 1;
}

int launch_scatter(const LevelTable &lv, float *grad, const Workspace &ws, const uint32_t *d_S, int n_sms, cudaStream_t st,
                   uint32_t seq) {
  // gradient array beyond what the L2 keeps (~64 MB, profiles/r1p): prefetch NSM_SCATTER_PF_CHUNKS chunks ahead
  const int prefetch = lv.offset[lv.n_levels] * lv.n_features * sizeof(float) > (96ull << 20) ? NSM_SCATTER_PF_CHUNKS : 0;
  dim3 grid(n_sms * 8), block(256);
  const uint32_t l0 = 0, l1 = lv.n_levels;
  switch (lv.n_features) {
    case 1: launch_pdl(scatter_backward_kernel<1>, grid, block, 0, st, lv, grad, ws, d_S, l0, l1, prefetch, seq); break;
    case 2: launch_pdl(scatter_backward_kernel<2>, grid, block, 0, st, lv, grad, ws, d_S, l0, l1, prefetch, seq); break;
    case 4: launch_pdl(scatter_backward_kernel<4>, grid, block, 0, st, lv, grad, ws, d_S, l0, l1, prefetch, seq); break;
    default: launch_pdl(scatter_backward_kernel<8>, grid, block, 0, st, lv, grad, ws, d_S, l0, l1, prefetch, seq); break;
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
