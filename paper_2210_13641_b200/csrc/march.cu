// march.cu — S1-S3 of DESIGN.md "Algorithm": candidate samples along each ray (PAPER.md:139,143:
// "sampling 3D positions along the pixel's ray", delta_i = d_{i+1} - d_i), the occupancy test,
// and prefix-sum compaction of the live samples in (ray, k) order.
//
// Index path: every fp32 operation below is an explicit round-to-nearest intrinsic so that the
// compiler cannot contract or reorder it; the integers it decides (live bits, counts) must be
// bit-exact against the oracle, and so must t, delta, x.
#include <cstdio>
#include <mutex>

#include "nsm_internal.cuh"

namespace {

__device__ __forceinline__ float jitter_u(uint32_t h_seed_step_ray, uint32_t k, uint32_t jitter) {
  if (!jitter) return 0.5f;
  uint32_t h = nsm_mix32(h_seed_step_ray ^ k);
  return __uint2float_rn(h >> 8) * 0x1p-24f;  // 24-bit integer, exact
}

// 2^e as a float, e in [-126, 127] (exact)
__device__ __forceinline__ float pow2f(int e) { return __int_as_float((127 + e) << 23); }

// S2 / F4 (reading R23): bit index of the occupancy cell that tests the normalised position x in [0,1)^3.
// C nested grids of G^3 cells share the cube's centre; cascade j (0 = finest) is the cube |x - 0.5|_max < 2^(j-C),
// cascade C-1 the whole cube; a point belongs to the finest cascade that contains it.  Index path: explicit fp32 ops.
__device__ __forceinline__ uint64_t occ_cell(uint32_t G, uint32_t C, const float x[3]) {
  uint32_t j = C - 1;
  float xp[3] = {x[0], x[1], x[2]};
  if (C > 1) {
    float q[3], m = 0.0f;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      q[a] = __fsub_rn(x[a], 0.5f);
      m = fmaxf(m, fabsf(q[a]));
    }
    for (j = 0; j + 1 < C; ++j)
      if (m < pow2f((int)j - (int)C)) break;
    if (j + 1 < C) {
      const float s = pow2f((int)(C - 1 - j));
#pragma unroll
      for (int a = 0; a < 3; ++a) xp[a] = __fmaf_rn(q[a], s, 0.5f);
    }
  }
  uint32_t g[3];
  const float Gf = __uint2float_rn(G);
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    int gi = __float2int_rd(__fmul_rn(xp[a], Gf));
    g[a] = (uint32_t)max(min(gi, (int)G - 1), 0);
  }
  return (uint64_t)j * G * G * G + (uint64_t)g[0] + (uint64_t)G * ((uint64_t)g[1] + (uint64_t)G * g[2]);
}

// the inverse: the point at offsets u in [0,1)^3 inside cell `cell` (u = 0.5: the centre, exact for power-of-two G)
__device__ __forceinline__ void occ_cell_point(uint32_t G, uint32_t C, uint64_t cell, const float u[3], float x[3]) {
  const uint64_t G3 = (uint64_t)G * G * G;
  const uint32_t j = (uint32_t)(cell / G3);
  const uint64_t loc = cell - (uint64_t)j * G3;
  const uint32_t g[3] = {(uint32_t)(loc % G), (uint32_t)((loc / G) % G), (uint32_t)(loc / ((uint64_t)G * G))};
  const float Gf = __uint2float_rn(G);
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    float xp = __fdiv_rn(__fadd_rn(__uint2float_rn(g[a]), u[a]), Gf);
    if (j + 1 < C) xp = __fmaf_rn(__fsub_rn(xp, 0.5f), pow2f((int)j - (int)(C - 1)), 0.5f);
    x[a] = xp;
  }
}

struct Candidate {
  float t, delta, x[3];
  bool live;
};

// S1.2-S1.4 and S2 for candidate k of one ray.
__device__ __forceinline__ Candidate make_candidate(const MarchParams &mp, const uint8_t *bits,
                                                    uint32_t hpre, const float o[3],
                                                    const float d[3], uint32_t k) {
  Candidate c;
  float u = jitter_u(hpre, k, mp.jitter);
  float ku = __fadd_rn(__uint2float_rn(k), u);
  c.t = __fmaf_rn(ku, mp.dt, mp.t_min);
  if (k + 1 < mp.K) {
    float u1 = jitter_u(hpre, k + 1, mp.jitter);
    c.delta = __fmul_rn(__fsub_rn(__fadd_rn(1.0f, u1), u), mp.dt);
  } else {
    c.delta = __fmul_rn(__fsub_rn(1.0f, u), mp.dt);
  }
  bool inside = true;
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    float p = __fmaf_rn(c.t, d[a], o[a]);
    c.x[a] = __fmul_rn(__fsub_rn(p, mp.aabb_min[a]), mp.inv_extent);
    inside = inside && (c.x[a] >= 0.0f) && (c.x[a] < 1.0f);  // NaN -> false
  }
  c.live = false;
  if (inside) {
    const uint64_t cell = occ_cell(mp.G, mp.C, c.x);
    c.live = bits ? ((__ldg(bits + (cell >> 3)) >> (cell & 7)) & 1u) : true;
  }
  return c;
}

// S1-S3 in ONE launch.  One warp per ray, MARCH_WARPS rays per block.  Pass 1: lanes stride over the
// K candidates, ballot gives the live-mask words (kept in shared memory) and the ray's count n_r.
// The exclusive scan over rays is a single-pass chained scan with decoupled look-back: blocks take a
// ticket (so block order = ray order whatever the hardware's dispatch order is), publish their
// aggregate, and sum their predecessors' aggregates back to the nearest published inclusive prefix.
// Pass 2: each live candidate is written at offsets[r] + its rank among the ray's live ones, so the
// compacted list is in (ray, k) order and bit-identical from run to run.  The last block to finish
// resets the scan state for the next launch.
constexpr uint32_t MARCH_WARPS = 16;
constexpr uint32_t MARCH_MAX_WORDS = 128;        // K <= 4096 (validate_config)
constexpr uint64_t SCAN_AGG = 1ull << 32, SCAN_INCL = 2ull << 32;

// Four blocks per SM (32 registers instead of 38, 16 bytes of spill): the kernel is issue- and barrier-bound, and a
// fourth block's warps fill the chained scan's waits (config 5: 1240 -> 1164 us per 816 000-ray view).
__global__ void __launch_bounds__(MARCH_WARPS * 32, 4) march_fused_kernel(MarchParams mp, const uint8_t *bits,
                                                                       const float *__restrict__ origins,
                                                                       const float *__restrict__ dirs, Workspace ws,
                                                                       int count_total, float *__restrict__ dirs_copy) {
  __shared__ uint32_t masks[MARCH_WARPS][MARCH_MAX_WORDS];
  __shared__ uint32_t warp_n[MARCH_WARPS];
  __shared__ uint32_t look_first[MARCH_WARPS], look_sum[MARCH_WARPS];
  __shared__ uint32_t ticket_s, block_base_s, total_s;
  const uint32_t tid = threadIdx.x, wid = tid >> 5, lane = tid & 31;
  uint32_t *ticket_ctr = ws.scan_ctr, *done_ctr = ws.scan_ctr + 1;
  volatile unsigned long long *state = ws.scan_state;
  pdl_wait();
  pdl_trigger();
  tl_mark(ws.timeline, K_MARCH, 0);
  if (tid == 0) ticket_s = atomicAdd(ticket_ctr, 1u);
  __syncthreads();
  const uint32_t ticket = ticket_s;
  const uint32_t r = ticket * MARCH_WARPS + wid, words = (mp.K + 31) >> 5;
  float o[3] = {0.f, 0.f, 0.f}, d[3] = {0.f, 0.f, 0.f};
  uint32_t hpre = 0, n = 0;
  if (r < mp.R) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      o[a] = __ldg(origins + 3 * (size_t)r + a);
      d[a] = __ldg(dirs + 3 * (size_t)r + a);
    }
    if (dirs_copy && lane < 3) dirs_copy[3 * (size_t)r + lane] = lane == 0 ? d[0] : (lane == 1 ? d[1] : d[2]);
    hpre = nsm_hash_prefix(mp.seed, mp.step, r);
    for (uint32_t wd0 = 0; wd0 < words; wd0 += 4) {   // four words at a time: their occupancy loads are independent
      bool live[4];
#pragma unroll
      for (uint32_t j = 0; j < 4; ++j) {
        const uint32_t k = (wd0 + j) * 32 + lane;
        live[j] = (k < mp.K) && make_candidate(mp, bits, hpre, o, d, k).live;
      }
#pragma unroll
      for (uint32_t j = 0; j < 4; ++j) {
        const uint32_t m = __ballot_sync(0xffffffffu, live[j]);
        if (lane == 0 && wd0 + j < words) masks[wid][wd0 + j] = m;
        n += __popc(m);
      }
    }
  }
  if (lane == 0) warp_n[wid] = n;
  __syncthreads();
  uint32_t total = 0;
  if (wid == 0) {
    // block-local exclusive scan of the MARCH_WARPS counts, then publish the block's aggregate
    const uint32_t v = lane < MARCH_WARPS ? warp_n[lane] : 0u;
    uint32_t incl = v;
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
      const uint32_t y = __shfl_up_sync(0xffffffffu, incl, s);
      if (lane >= (uint32_t)s) incl += y;
    }
    if (lane < MARCH_WARPS) warp_n[lane] = incl - v;
    total = __shfl_sync(0xffffffffu, incl, 31);
    if (lane == 0) {
      atomicExch((unsigned long long *)&state[ticket], (ticket == 0 ? SCAN_INCL : SCAN_AGG) | total);
      total_s = total;
    }
  }
  // look-back by the whole block: thread i reads predecessor ticket-1-i (spinning until it is
  // published); the sum runs back to the nearest inclusive prefix.  One L2 round trip covers
  // MARCH_WARPS*32 predecessors.
  uint32_t excl = 0;
  for (int64_t top = (int64_t)ticket - 1; top >= 0; top -= MARCH_WARPS * 32) {
    const int64_t idx = top - tid;
    unsigned long long st = SCAN_INCL;       // positions before ticket 0 count as "inclusive prefix 0"
    if (idx >= 0) do { st = state[idx]; } while ((st >> 32) == 0);
    const uint32_t incl_lanes = __ballot_sync(0xffffffffu, (st >> 32) == 2);
    if (lane == 0) look_first[wid] = incl_lanes ? (uint32_t)__ffs(incl_lanes) - 1 : 32u;
    __syncthreads();
    uint32_t first = MARCH_WARPS * 32;       // block-wide position of the nearest inclusive prefix
#pragma unroll
    for (uint32_t w = 0; w < MARCH_WARPS; ++w)
      if (first == MARCH_WARPS * 32 && look_first[w] < 32) first = w * 32 + look_first[w];
    uint32_t val = tid <= first ? (uint32_t)st : 0u;
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) val += __shfl_xor_sync(0xffffffffu, val, s);
    if (lane == 0) look_sum[wid] = val;
    __syncthreads();
#pragma unroll
    for (uint32_t w = 0; w < MARCH_WARPS; ++w) excl += look_sum[w];
    __syncthreads();
    if (first < MARCH_WARPS * 32) break;
  }
  if (tid == 0) {
    total = total_s;
    if (ticket != 0) atomicExch((unsigned long long *)&state[ticket], SCAN_INCL | (unsigned long long)(excl + total));
    block_base_s = excl;
    if (ticket == gridDim.x - 1) {
      ws.offsets[mp.R] = excl + total;
      ws.loss_acc[2] = (double)(excl + total);   // S beside the loss sums: the stats come back in one copy
      if (count_total) *ws.total_samples += excl + total;
    }
    if (ticket == 0) {
      ws.loss_acc[0] = 0.0; ws.loss_acc[1] = 0.0;
      *ws.grad_absmax = 0u;
    }
  }
  __syncthreads();
  if (r < mp.R) {
    uint32_t base = block_base_s + warp_n[wid];
    if (lane == 0) { ws.offsets[r] = base; ws.counts[r] = n; }
    for (uint32_t wd = 0; wd < words; ++wd) {
      const uint32_t m = masks[wid][wd];
      if ((m >> lane) & 1u) {
        const uint32_t k = wd * 32 + lane;
        const Candidate c = make_candidate(mp, nullptr, hpre, o, d, k);
        const uint64_t s = (uint64_t)base + __popc(m & ((1u << lane) - 1u));
        ws.s_ray[s] = r;
        ws.s_k[s] = k;
        ws.s_t[s] = c.t;
        ws.s_delta[s] = c.delta;
        ws.s_x[s] = c.x[0];
        ws.s_x[ws.cap + s] = c.x[1];
        ws.s_x[2 * ws.cap + s] = c.x[2];
      }
      base += __popc(m);
    }
  }
  // the last block to get here has seen every look-back finish: reset the scan state
  __syncthreads();
  if (tid == 0) {
    __threadfence();
    total_s = atomicAdd(done_ctr, 1u);
  }
  __syncthreads();
  if (total_s == gridDim.x - 1) {
    for (uint32_t i = tid; i < gridDim.x; i += MARCH_WARPS * 32) state[i] = 0ull;
    if (tid == 0) { *ticket_ctr = 0u; *done_ctr = 0u; }
  }
  tl_mark(ws.timeline, K_MARCH, 1);
}

// S14 FROM_FIELD / F4: the centres of the cells first_cell + i * stride (i < n_cells) of the occupancy structure (all
// cascades, global cell index) as "samples".
__global__ void occ_cells_kernel(uint32_t G, uint32_t C, uint64_t first_cell, uint32_t stride, uint64_t n_cells, Workspace ws,
                                 uint32_t *d_S) {
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) *d_S = (uint32_t)n_cells;
  if (i >= n_cells) return;
  const float half[3] = {0.5f, 0.5f, 0.5f};
  float x[3];
  occ_cell_point(G, C, first_cell + i * stride, half, x);
  ws.s_x[i] = x[0];
  ws.s_x[ws.cap + i] = x[1];
  ws.s_x[2 * ws.cap + i] = x[2];
  ws.s_ray[i] = 0;
}

// F4, stochastic refresh (reading R25): draw i of update `upd` picks cell (h(seed, upd, i, 0xffff0003) * n_total) >> 32 and
// the point at offsets u_a = (h(seed, upd, i, 0xffff0004 + a) >> 8) 2^-24 inside it; the cell index is kept in ws.s_k.
__global__ void occ_cells_stochastic_kernel(uint32_t G, uint32_t C, uint64_t seed, uint32_t upd, uint32_t first_draw,
                                            uint32_t n_draws, Workspace ws, uint32_t *d_S) {
  uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) *d_S = n_draws;
  if (i >= n_draws) return;
  const uint64_t n_total = (uint64_t)C * G * G * G;
  const uint32_t hpre = nsm_hash_prefix(seed, upd, first_draw + i);
  const uint64_t cell = ((uint64_t)nsm_mix32(hpre ^ 0xffff0003u) * n_total) >> 32;
  float u[3], x[3];
#pragma unroll
  for (uint32_t a = 0; a < 3; ++a) u[a] = __uint2float_rn(nsm_mix32(hpre ^ (0xffff0004u + a)) >> 8) * 0x1p-24f;
  occ_cell_point(G, C, cell, u, x);
  ws.s_x[i] = x[0];
  ws.s_x[ws.cap + i] = x[1];
  ws.s_x[2 * ws.cap + i] = x[2];
  ws.s_ray[i] = 0;
  ws.s_k[i] = (uint32_t)cell;
}

// grid[cell_i] <- max(grid[cell_i], sigma_i); a cell drawn twice keeps the larger density (order-free): densities and
// grid values are non-negative, so the integer maximum of their bit patterns is the float maximum
__global__ void occ_max_cells_kernel(float *__restrict__ grid, const uint32_t *__restrict__ cells, uint32_t n,
                                     const float *__restrict__ sigma) {
  uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  atomicMax(reinterpret_cast<int *>(grid + cells[i]), __float_as_int(fmaxf(sigma[i], 0.0f)));
}

// bit = sigma > thr; one warp packs 32 cells into one word (first_cell is a multiple of 32).  The densities also
// seed the running grid of the decayed refresh (F4).
__global__ void occ_threshold_kernel(uint64_t first_cell, uint64_t n_cells,
                                     const float *__restrict__ sigma, float thr, uint32_t *bits32, float *__restrict__ grid) {
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool on = i < n_cells && sigma[i] > thr;
  if (i < n_cells) grid[first_cell + i] = sigma[i];
  uint32_t m = __ballot_sync(0xffffffffu, on);
  if ((threadIdx.x & 31) == 0 && i < n_cells) bits32[(first_cell + i) >> 5] = m;
}

// ---- F4 (row f4; paper silent, after [17]): decayed running maximum of the density with a strided partial refresh ----
//   every cell: grid <- decay * grid;   cells c = c0 + j * n_sub (c0 = update index mod n_sub): grid <- max(grid, sigma(c));
//   bit = grid > thr.   n_sub consecutive updates visit every cell exactly once.
__global__ void occ_decay_kernel(float *__restrict__ grid, uint64_t n_cells, float decay) {
  for (uint64_t c = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; c < n_cells; c += (uint64_t)gridDim.x * blockDim.x)
    grid[c] *= decay;
}

__global__ void occ_max_visited_kernel(float *__restrict__ grid, uint64_t first_cell, uint32_t stride, uint64_t n_visited,
                                       const float *__restrict__ sigma) {
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_visited) return;
  float *g = grid + first_cell + i * stride;
  *g = fmaxf(*g, sigma[i]);
}

__global__ void occ_bits_from_grid_kernel(const float *__restrict__ grid, uint64_t n_cells, float thr, uint32_t *bits32) {
  uint64_t c = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool on = c < n_cells && grid[c] > thr;
  uint32_t m = __ballot_sync(0xffffffffu, on);
  if ((threadIdx.x & 31) == 0 && c < n_cells) bits32[c >> 5] = m;
}

}  // namespace

int launch_march(const MarchParams &mp, const uint8_t *bits, const float *origins, const float *dirs,
                 const Workspace &ws, int count_total, cudaStream_t st, float *dirs_copy) {
  dim3 grid((mp.R + MARCH_WARPS - 1) / MARCH_WARPS), block(MARCH_WARPS * 32);
  launch_pdl(march_fused_kernel, grid, block, 0, st, mp, bits, origins, dirs, ws, count_total, dirs_copy);
  return 1;
}

uint32_t march_scan_state_entries(uint32_t max_rays) { return (max_rays + MARCH_WARPS - 1) / MARCH_WARPS; }

int launch_occ_cells(uint32_t G, uint32_t C, uint64_t first_cell, uint32_t stride, uint64_t n_cells, const Workspace &ws,
                     uint32_t *d_S, cudaStream_t st) {
  occ_cells_kernel<<<(unsigned)((n_cells + 255) / 256), 256, 0, st>>>(G, C, first_cell, stride, n_cells, ws, d_S);
  return 1;
}

int launch_occ_cells_stochastic(uint32_t G, uint32_t C, uint64_t seed, uint32_t upd, uint32_t first_draw, uint32_t n_draws,
                                const Workspace &ws, uint32_t *d_S, cudaStream_t st) {
  occ_cells_stochastic_kernel<<<(n_draws + 255) / 256, 256, 0, st>>>(G, C, seed, upd, first_draw, n_draws, ws, d_S);
  return 1;
}

int launch_occ_max_cells(float *grid, const uint32_t *cells, uint32_t n, const float *sigma, cudaStream_t st) {
  occ_max_cells_kernel<<<(n + 255) / 256, 256, 0, st>>>(grid, cells, n, sigma);
  return 1;
}

int launch_occ_threshold(uint32_t G, uint64_t first_cell, uint64_t n_cells, const float *sigma,
                         float thr, uint8_t *bits, float *grid, cudaStream_t st) {
  (void)G;
  occ_threshold_kernel<<<(unsigned)((n_cells + 255) / 256), 256, 0, st>>>(first_cell, n_cells, sigma, thr,
                                                                         (uint32_t *)bits, grid);
  return 1;
}

int launch_occ_decay(float *grid, uint64_t n_cells, float decay, cudaStream_t st) {
  occ_decay_kernel<<<1184, 256, 0, st>>>(grid, n_cells, decay);
  return 1;
}

int launch_occ_max_visited(float *grid, uint64_t first_cell, uint32_t stride, uint64_t n_visited, const float *sigma, cudaStream_t st) {
  occ_max_visited_kernel<<<(unsigned)((n_visited + 255) / 256), 256, 0, st>>>(grid, first_cell, stride, n_visited, sigma);
  return 1;
}

int launch_occ_bits_from_grid(const float *grid, uint64_t n_cells, float thr, uint8_t *bits, cudaStream_t st) {
  occ_bits_from_grid_kernel<<<(unsigned)((n_cells + 255) / 256), 256, 0, st>>>(grid, n_cells, thr, (uint32_t *)bits);
  return 1;
}

// ---- nsm_march_static (include/nsm.h "S1-S3 alone, allocating nothing") ---------------------------------------------
// The scratch memory of march_fused_kernel -- the ticket / finished-block counters and the chained scan's per-block
// status words, plus the few words the kernel writes beside the loss sums for the field's step -- in a file-scope
// device array instead of the field's arena, so that the entry point below never allocates.  Layout (bytes):
//   [0, 8)     scan_ctr[2]          [8, 12)  grad_absmax        [16, 40)  loss_acc[3]        [40, 48)  total_samples
//   [256, ...) scan_state[NSM_MARCH_STATIC_MAX_RAYS / MARCH_WARPS]
// In HOST code the name below is a host-side stand-in, not a device address: the kernel gets the address that
// cudaGetSymbolAddress returns for the current device (looked up once per device, cached).
namespace {

constexpr uint32_t STATIC_ENTRIES = NSM_MARCH_STATIC_MAX_RAYS / MARCH_WARPS;
constexpr size_t STATIC_HEADER = 256, STATIC_BYTES = STATIC_HEADER + sizeof(unsigned long long) * STATIC_ENTRIES;
static_assert(NSM_MARCH_STATIC_MAX_RAYS % MARCH_WARPS == 0, "whole blocks");

static __device__ __align__(256) unsigned char march_static_scratch[STATIC_BYTES];

constexpr int STATIC_MAX_DEVICES = 64;
std::mutex g_static_mu;
unsigned char *g_static_ptr[STATIC_MAX_DEVICES] = {};

// device address of march_static_scratch on the CURRENT device
nsm_status static_scratch(unsigned char **out, int *dev_out) {
  char msg[256];
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) {
    snprintf(msg, sizeof msg, "cudaGetDevice: %s (there is no CPU fallback)", cudaGetErrorString(e));
    cudaGetLastError();
    return nsm_set_error(NSM_ERR_CUDA, msg);
  }
  if (dev < 0 || dev >= STATIC_MAX_DEVICES) return nsm_set_error(NSM_ERR_CUDA, "nsm_march_static: device ordinal out of range");
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_ptr[dev]) {
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, march_static_scratch);
    if (e != cudaSuccess || !p) {
      snprintf(msg, sizeof msg, "cudaGetSymbolAddress(march_static_scratch) on device %d: %s", dev, cudaGetErrorString(e));
      cudaGetLastError();
      return nsm_set_error(NSM_ERR_CUDA, msg);
    }
    g_static_ptr[dev] = (unsigned char *)p;
  }
  *out = g_static_ptr[dev];
  *dev_out = dev;
  return NSM_OK;
}

// a device pointer that belongs to another device than `dev`?  (host-mapped and unregistered pointers pass)
bool on_other_device(const void *p, int dev) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice && a.device != dev;
}

}  // namespace

extern "C" nsm_status nsm_march_static(const nsm_march_config *cfg, const nsm_ray_batch *rays, const uint8_t *d_occ_bits,
                                       const nsm_march_result *out, void *cuda_stream) {
  char msg[256];
  if (!cfg || !rays || !out) return nsm_set_error(NSM_ERR_INVALID_ARG, "nsm_march_static: cfg, rays or out is NULL");
  if (cfg->struct_size != sizeof(nsm_march_config)) {
    snprintf(msg, sizeof msg, "nsm_march_static: struct_size %u != %zu (ABI mismatch)", cfg->struct_size, sizeof(nsm_march_config));
    return nsm_set_error(NSM_ERR_INVALID_ARG, msg);
  }
  if (!(cfg->aabb_extent > 0.f) || !isfinite(cfg->aabb_extent)) return nsm_set_error(NSM_ERR_INVALID_ARG, "nsm_march_static: aabb_extent must be > 0");
  const uint32_t G = cfg->occ_res, C = cfg->occ_cascades ? cfg->occ_cascades : 1u;
  if (G < 1 || G > 1024 || (G & (G - 1))) return nsm_set_error(NSM_ERR_INVALID_ARG, "nsm_march_static: occ_res must be a power of two <= 1024");
  if (C > 8) return nsm_set_error(NSM_ERR_INVALID_ARG, "nsm_march_static: occ_cascades must be <= 8");
  if ((uint64_t)C * G * G * G > (1ull << 31)) return nsm_set_error(NSM_ERR_INVALID_ARG, "nsm_march_static: occ_cascades * occ_res^3 exceeds 2^31 cells");
  if (!rays->origins || !rays->dirs) return nsm_set_error(NSM_ERR_INVALID_ARG, "nsm_march_static: origins/dirs are NULL");
  const uint32_t R = rays->n_rays, K = rays->n_candidates;
  if (R == 0 || K == 0) return nsm_set_error(NSM_ERR_INVALID_ARG, "nsm_march_static: n_rays or n_candidates is 0");
  if (!(rays->t_min < rays->t_max) || !isfinite(rays->t_min) || !isfinite(rays->t_max))
    return nsm_set_error(NSM_ERR_INVALID_ARG, "nsm_march_static: need finite t_min < t_max");
  if (R > NSM_MARCH_STATIC_MAX_RAYS) {
    snprintf(msg, sizeof msg, "nsm_march_static: n_rays %u exceeds the static scratch array's maximum of %u rays per call", R,
             NSM_MARCH_STATIC_MAX_RAYS);
    return nsm_set_error(NSM_ERR_CAPACITY, msg);
  }
  if (K > MARCH_MAX_WORDS * 32) {
    snprintf(msg, sizeof msg, "nsm_march_static: n_candidates %u exceeds the maximum of %u", K, MARCH_MAX_WORDS * 32);
    return nsm_set_error(NSM_ERR_CAPACITY, msg);
  }
  if ((uint64_t)R * K > (1ull << 31)) return nsm_set_error(NSM_ERR_CAPACITY, "nsm_march_static: n_rays * n_candidates exceeds 2^31");
  if (!out->counts || !out->offsets || !out->s_ray || !out->s_k || !out->s_t || !out->s_delta || !out->s_x)
    return nsm_set_error(NSM_ERR_INVALID_ARG, "nsm_march_static: an output pointer is NULL");
  if (out->capacity < (uint64_t)R * K) {
    snprintf(msg, sizeof msg, "nsm_march_static: out->capacity %llu < n_rays * n_candidates = %llu", (unsigned long long)out->capacity,
             (unsigned long long)R * K);
    return nsm_set_error(NSM_ERR_CAPACITY, msg);
  }
  unsigned char *scratch = nullptr;
  int dev = -1;
  nsm_status st = static_scratch(&scratch, &dev);
  if (st != NSM_OK) return st;
  if (on_other_device(rays->origins, dev) || on_other_device(out->counts, dev) || on_other_device(out->s_x, dev)) {
    snprintf(msg, sizeof msg, "nsm_march_static: the pointers belong to another device than the current one (%d)", dev);
    return nsm_set_error(NSM_ERR_INVALID_ARG, msg);
  }
  cudaStream_t stream = (cudaStream_t)cuda_stream;

  MarchParams mp;
  for (int a = 0; a < 3; ++a) mp.aabb_min[a] = cfg->aabb_min[a];
  mp.inv_extent = 1.0f / cfg->aabb_extent;                        // as make_march (nsm_api.cu): one fp32 divide
  mp.t_min = rays->t_min;
  mp.dt = (rays->t_max - rays->t_min) / (float)K;                 // one fp32 subtract, one fp32 divide
  mp.K = K; mp.G = G; mp.C = C;
  mp.jitter = cfg->jitter ? 1u : 0u;
  mp.step = cfg->step;
  mp.seed = cfg->seed;
  mp.R = R;

  Workspace ws = {};                                              // everything the marcher does not touch stays NULL
  ws.cap = out->capacity;
  ws.max_rays = NSM_MARCH_STATIC_MAX_RAYS;
  ws.counts = out->counts; ws.offsets = out->offsets;
  ws.s_ray = out->s_ray; ws.s_k = out->s_k; ws.s_t = out->s_t; ws.s_delta = out->s_delta; ws.s_x = out->s_x;
  ws.scan_ctr = (uint32_t *)scratch;
  ws.grad_absmax = (uint32_t *)(scratch + 8);
  ws.loss_acc = (double *)(scratch + 16);
  ws.total_samples = (unsigned long long *)(scratch + 40);
  ws.scan_state = (unsigned long long *)(scratch + STATIC_HEADER);

  // The array keeps the last call's contents.  The kernel's last block zeroes the words it used, but a call that was
  // cut short (a fault, a reset stream) would leave them set: clear what this launch reads before it starts.
  const uint32_t n_blocks = (R + MARCH_WARPS - 1) / MARCH_WARPS;
  cudaError_t e = cudaMemsetAsync(scratch, 0, STATIC_HEADER + sizeof(unsigned long long) * n_blocks, stream);
  if (e == cudaSuccess) {
    march_fused_kernel<<<n_blocks, MARCH_WARPS * 32, 0, stream>>>(mp, d_occ_bits, rays->origins, rays->dirs, ws, 0, nullptr);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) {
    snprintf(msg, sizeof msg, "nsm_march_static: %s", cudaGetErrorString(e));
    return nsm_set_error(NSM_ERR_CUDA, msg);
  }
  return NSM_OK;
}
