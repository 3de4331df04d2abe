// march.cu — S1-S3 of DESIGN.md "Algorithm": candidate samples along each ray (PAPER.md:139,143:
// "sampling 3D positions along the pixel's ray", delta_i = d_{i+1} - d_i), the occupancy test,
// and prefix-sum compaction of the live samples in (ray, k) order.
//
// Index path: every fp32 operation below is an explicit round-to-nearest intrinsic so that the
// compiler cannot contract or reorder it; the integers it decides (live bits, counts) must be
// bit-exact against the oracle, and so must t, delta, x.
#include "nsm_internal.cuh"

namespace {

// DESIGN.md S1.1 — jitter hash (two-multiply xorshift finaliser absorbing seed, step, r, k).
__device__ __forceinline__ uint32_t mix32(uint32_t x) {
  x ^= x >> 16;
  x *= 0x7feb352du;
  x ^= x >> 15;
  x *= 0x846ca68bu;
  x ^= x >> 16;
  return x;
}

__device__ __forceinline__ float jitter_u(uint32_t h_seed_step_ray, uint32_t k, uint32_t jitter) {
  if (!jitter) return 0.5f;
  uint32_t h = mix32(h_seed_step_ray ^ k);
  return __uint2float_rn(h >> 8) * 0x1p-24f;  // 24-bit integer, exact
}

__device__ __forceinline__ uint32_t ray_hash_prefix(uint64_t seed, uint32_t step, uint32_t r) {
  uint32_t h = mix32((uint32_t)(seed & 0xffffffffu) ^ 0x9e3779b9u);
  h = mix32(h ^ (uint32_t)(seed >> 32));
  h = mix32(h ^ step);
  h = mix32(h ^ r);
  return h;
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
    uint32_t g[3];
    const float Gf = __uint2float_rn(mp.G);
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      int gi = __float2int_rd(__fmul_rn(c.x[a], Gf));
      g[a] = (uint32_t)min(gi, (int)mp.G - 1);
    }
    uint64_t cell = (uint64_t)g[0] + (uint64_t)mp.G * ((uint64_t)g[1] + (uint64_t)mp.G * g[2]);
    c.live = bits ? ((__ldg(bits + (cell >> 3)) >> (cell & 7)) & 1u) : true;
  }
  return c;
}

// One warp per ray: lanes stride over the K candidates; ballot gives the live mask words.
__global__ void __launch_bounds__(256) march_count_kernel(MarchParams mp, const uint8_t *bits,
                                                          const float *__restrict__ origins,
                                                          const float *__restrict__ dirs,
                                                          uint32_t *__restrict__ counts,
                                                          uint32_t *__restrict__ live_mask) {
  const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= mp.R) return;
  const uint32_t r = warp, words = (mp.K + 31) >> 5;
  float o[3], d[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    o[a] = __ldg(origins + 3 * (size_t)r + a);
    d[a] = __ldg(dirs + 3 * (size_t)r + a);
  }
  const uint32_t hpre = ray_hash_prefix(mp.seed, mp.step, r);
  uint32_t n = 0;
  for (uint32_t wd = 0; wd < words; ++wd) {
    uint32_t k = wd * 32 + lane;
    bool live = false;
    if (k < mp.K) live = make_candidate(mp, bits, hpre, o, d, k).live;
    uint32_t m = __ballot_sync(0xffffffffu, live);
    if (lane == 0) live_mask[(size_t)r * words + wd] = m;
    n += __popc(m);
  }
  if (lane == 0) counts[r] = n;
}

// Exclusive scan of counts[R] -> offsets[R+1] by one block (R <= a few 100 K per call), and
// reset of the loss accumulators.  Deterministic.
__global__ void __launch_bounds__(1024) scan_counts_kernel(const uint32_t *__restrict__ counts,
                                                           uint32_t *__restrict__ offsets, uint32_t R,
                                                           double *loss_acc, unsigned long long *total, uint32_t *absmax) {
  __shared__ uint32_t warp_sums[32];
  __shared__ uint32_t carry_s;
  const uint32_t tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  if (tid == 0) {
    carry_s = 0;
    if (loss_acc) { loss_acc[0] = 0.0; loss_acc[1] = 0.0; }
    if (absmax) *absmax = 0u;
  }
  __syncthreads();
  for (uint32_t base = 0; base < R; base += 1024) {
    uint32_t i = base + tid;
    uint32_t v = i < R ? counts[i] : 0u;
    uint32_t incl = v;
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
      uint32_t y = __shfl_up_sync(0xffffffffu, incl, s);
      if (lane >= s) incl += y;
    }
    if (lane == 31) warp_sums[wid] = incl;
    __syncthreads();
    if (wid == 0) {
      uint32_t ws = warp_sums[lane], wi = ws;
#pragma unroll
      for (int s = 1; s < 32; s <<= 1) {
        uint32_t y = __shfl_up_sync(0xffffffffu, wi, s);
        if (lane >= s) wi += y;
      }
      warp_sums[lane] = wi - ws;  // exclusive warp offsets
    }
    __syncthreads();
    uint32_t carry = carry_s;
    uint32_t excl = carry + warp_sums[wid] + incl - v;
    if (i < R) offsets[i] = excl;
    __syncthreads();
    if (tid == 1023) carry_s = excl + v;
    __syncthreads();
  }
  if (tid == 0) {
    offsets[R] = carry_s;
    if (total) *total += carry_s;
  }
}

// Second pass: each live candidate is written at offsets[r] + its rank among the ray's live ones.
__global__ void __launch_bounds__(256) march_write_kernel(MarchParams mp, const uint8_t *bits,
                                                          const float *__restrict__ origins,
                                                          const float *__restrict__ dirs,
                                                          const uint32_t *__restrict__ offsets,
                                                          const uint32_t *__restrict__ live_mask,
                                                          Workspace ws) {
  const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (warp >= mp.R) return;
  const uint32_t r = warp, words = (mp.K + 31) >> 5;
  float o[3], d[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    o[a] = __ldg(origins + 3 * (size_t)r + a);
    d[a] = __ldg(dirs + 3 * (size_t)r + a);
  }
  const uint32_t hpre = ray_hash_prefix(mp.seed, mp.step, r);
  uint32_t base = offsets[r];
  for (uint32_t wd = 0; wd < words; ++wd) {
    uint32_t m = live_mask[(size_t)r * words + wd];
    if ((m >> lane) & 1u) {
      uint32_t k = wd * 32 + lane;
      Candidate c = make_candidate(mp, nullptr, hpre, o, d, k);
      uint64_t s = (uint64_t)base + __popc(m & ((1u << lane) - 1u));
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

// S14 FROM_FIELD: the cell centres of a chunk of the occupancy grid as "samples".
__global__ void occ_cells_kernel(uint32_t G, uint64_t first_cell, uint64_t n_cells, Workspace ws,
                                 uint32_t *d_S) {
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) *d_S = (uint32_t)n_cells;
  if (i >= n_cells) return;
  uint64_t cell = first_cell + i;
  uint32_t gx = (uint32_t)(cell % G), gy = (uint32_t)((cell / G) % G), gz = (uint32_t)(cell / ((uint64_t)G * G));
  const float Gf = __uint2float_rn(G);
  ws.s_x[i] = __fdiv_rn(__fadd_rn(__uint2float_rn(gx), 0.5f), Gf);  // exact for power-of-two G
  ws.s_x[ws.cap + i] = __fdiv_rn(__fadd_rn(__uint2float_rn(gy), 0.5f), Gf);
  ws.s_x[2 * ws.cap + i] = __fdiv_rn(__fadd_rn(__uint2float_rn(gz), 0.5f), Gf);
  ws.s_ray[i] = 0;
}

// bit = sigma > thr; one warp packs 32 cells into one word (first_cell is a multiple of 32).
__global__ void occ_threshold_kernel(uint64_t first_cell, uint64_t n_cells,
                                     const float *__restrict__ sigma, float thr, uint32_t *bits32) {
  uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool on = i < n_cells && sigma[i] > thr;
  uint32_t m = __ballot_sync(0xffffffffu, on);
  if ((threadIdx.x & 31) == 0 && i < n_cells) bits32[(first_cell + i) >> 5] = m;
}

}  // namespace

int launch_march_count(const MarchParams &mp, const uint8_t *bits, const float *origins, const float *dirs,
                       const Workspace &ws, cudaStream_t st) {
  dim3 grid((mp.R + 7) / 8), block(256);
  march_count_kernel<<<grid, block, 0, st>>>(mp, bits, origins, dirs, ws.counts, ws.live_mask);
  return 1;
}

int launch_scan(const MarchParams &mp, const Workspace &ws, int count_total, cudaStream_t st) {
  scan_counts_kernel<<<1, 1024, 0, st>>>(ws.counts, ws.offsets, mp.R, ws.loss_acc,
                                         count_total ? ws.total_samples : nullptr, ws.grad_absmax);
  return 1;
}

int launch_march_write(const MarchParams &mp, const float *origins, const float *dirs, const Workspace &ws,
                       cudaStream_t st) {
  dim3 grid((mp.R + 7) / 8), block(256);
  march_write_kernel<<<grid, block, 0, st>>>(mp, nullptr, origins, dirs, ws.offsets, ws.live_mask, ws);
  return 1;
}

int launch_occ_cells(uint32_t G, uint64_t first_cell, uint64_t n_cells, const Workspace &ws,
                     uint32_t *d_S, cudaStream_t st) {
  occ_cells_kernel<<<(unsigned)((n_cells + 255) / 256), 256, 0, st>>>(G, first_cell, n_cells, ws, d_S);
  return 1;
}

int launch_occ_threshold(uint32_t G, uint64_t first_cell, uint64_t n_cells, const float *sigma,
                         float thr, uint8_t *bits, cudaStream_t st) {
  (void)G;
  occ_threshold_kernel<<<(unsigned)((n_cells + 255) / 256), 256, 0, st>>>(first_cell, n_cells, sigma, thr,
                                                                         (uint32_t *)bits);
  return 1;
}
