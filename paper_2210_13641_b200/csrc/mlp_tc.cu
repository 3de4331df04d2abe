// mlp_tc.cu — S5/S6/S7 (and S11) on the 5th-generation tensor cores: the density and colour MLPs
// of PAPER.md:143,151 as 128-sample tcgen05.mma tiles (M = 128 samples, N = layer width, K = input
// width; 16-bit operands in shared memory, fp32 accumulators in TMEM).
//
// One CTA (4 warps) owns a 128-sample tile; thread r owns sample row r: it builds its row of the
// layer input in shared memory (UMMA canonical no-swizzle K-major layout, 16-byte chunks at a 16 B
// stride across threads: conflict-free), ONE thread issues the layer's tcgen05.mma k-steps and a
// tcgen05.commit onto an mbarrier, everyone waits on it, reads its accumulator row back with
// tcgen05.ld (TMEM lane = sample row), applies the activation and writes the next layer's input.
// Weights are converted fp32 -> 16-bit and staged in shared memory once per CTA (persistent over
// tiles).  Activations never leave the SM between layers.
#include "nsm_internal.cuh"
#include "tc_common.cuh"

namespace {

using namespace tc;

constexpr uint32_t H = 64;      // hidden width of both MLPs on this path
constexpr uint32_t DO = 16;     // density MLP outputs
constexpr uint32_t CIP = 32;    // colour-MLP input width padded to a k-step multiple
constexpr uint32_t ROWS = NSM_TILE;
constexpr uint32_t PANEL = ROWS * 16;  // bytes of one 8-column panel of a 128-row tile

// TMEM column map (fp32 accumulators, 128 lanes = sample rows)
constexpr uint32_t COL_D1 = 0, COL_D2 = 64, COL_C1 = 96, COL_C2 = 160, COL_C3 = 224, FWD_COLS = 256;

struct FwdSmem {
  static constexpr uint32_t wd1 = 0;                         // [64][LF<=64]
  static constexpr uint32_t wd2 = wd1 + H * 64 * 2;          // [16][64]
  static constexpr uint32_t wc1 = wd2 + DO * H * 2;          // [64][32]
  static constexpr uint32_t wc2 = wc1 + H * CIP * 2;         // [64][64]
  static constexpr uint32_t wc3 = wc2 + H * H * 2;           // [16][64]
  static constexpr uint32_t bufA = wc3 + 16 * H * 2;         // [128][64]
  static constexpr uint32_t bufB = bufA + ROWS * H * 2;      // [128][64]
  static constexpr uint32_t bar = bufB + ROWS * H * 2;       // mbarrier
  static constexpr uint32_t tmem = bar + 8;
  static constexpr uint32_t total = tmem + 8;
};

// fp32 canonical W[n_out][n_in] (global) -> 16-bit operand tile [NP][KP] in shared memory, zero padded
template <typename T>
__device__ void stage_weight(uint8_t *tile, const float *__restrict__ W, uint32_t n_out, uint32_t n_in, uint32_t NP,
                             uint32_t KP) {
  for (uint32_t i = threadIdx.x; i < NP * KP; i += blockDim.x) {
    const uint32_t n = i / KP, k = i - n * KP;
    const float v = (n < n_out && k < n_in) ? __ldg(W + n * n_in + k) : 0.f;
    *reinterpret_cast<T *>(tile + tile_off(NP, n, k)) = T(v);
  }
}

// issue the k-steps of one layer: D[128 x N] = A[128 x K] * B[N x K]^T, both K-major
__device__ __forceinline__ void issue_layer(uint32_t tmem_d, uint32_t a_saddr, uint32_t b_saddr, uint32_t K, uint32_t N,
                                            uint32_t NP, uint32_t fmt, uint32_t bar_saddr) {
  const uint32_t idesc = make_idesc(fmt, 128, N, 0, 0);
  for (uint32_t k = 0; k < K / 16; ++k) {
    const uint64_t da = make_desc(a_saddr + k * 2 * PANEL, PANEL, 128);
    const uint64_t db = make_desc(b_saddr + k * 2 * NP * 16, NP * 16, 128);
    mma_ss(tmem_d, da, db, idesc, k > 0);
  }
  mma_commit(bar_saddr);
}

__device__ __forceinline__ void sh_row(uint32_t n, float x, float y, float z, float *Y) {
  // DESIGN.md S6, polynomial form, n <= 4
  Y[0] = 0.28209479177387814f;
  if (n < 2) return;
  Y[1] = 0.4886025119029199f * y; Y[2] = 0.4886025119029199f * z; Y[3] = 0.4886025119029199f * x;
  if (n < 3) return;
  const float xx = x * x, yy = y * y, zz = z * z;
  Y[4] = 1.0925484305920792f * x * y; Y[5] = 1.0925484305920792f * y * z;
  Y[6] = 0.31539156525252005f * (3.f * zz - 1.f); Y[7] = 1.0925484305920792f * x * z;
  Y[8] = 0.5462742152960396f * (xx - yy);
  if (n < 4) return;
  Y[9] = 0.5900435899266435f * y * (3.f * xx - yy); Y[10] = 2.890611442640554f * x * y * z;
  Y[11] = 0.4570457994644658f * y * (5.f * zz - 1.f); Y[12] = 0.3731763325901154f * z * (5.f * zz - 3.f);
  Y[13] = 0.4570457994644658f * x * (5.f * zz - 1.f); Y[14] = 1.445305721320277f * z * (xx - yy);
  Y[15] = 0.5900435899266435f * x * (xx - 3.f * yy);
}

template <typename T>
__global__ void __launch_bounds__(128) mlp_forward_tc_kernel(MlpShape ms, const float *__restrict__ Wm,
                                                             const float *__restrict__ dirs, Workspace ws,
                                                             const uint32_t *__restrict__ d_S, int density_only,
                                                             int write_planes) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t tid = threadIdx.x, warp = tid >> 5;
  const uint32_t sbase = smem_u32(smem);
  const uint32_t bar = sbase + FwdSmem::bar;
  const uint32_t LF = ms.LF;

  stage_weight<T>(smem + FwdSmem::wd1, Wm + ms.o_d1, H, LF, H, LF);
  stage_weight<T>(smem + FwdSmem::wd2, Wm + ms.o_d2, DO, H, DO, H);
  if (!density_only) {
    stage_weight<T>(smem + FwdSmem::wc1, Wm + ms.o_c1, H, ms.Ci, H, CIP);
    if (ms.n_color_layers == 2) stage_weight<T>(smem + FwdSmem::wc2, Wm + ms.o_c2, H, H, H, H);
    stage_weight<T>(smem + FwdSmem::wc3, Wm + ms.o_c3, 3, H, 16, H);
  }
  if (tid == 0) mbar_init(bar, 1);
  if (warp == 0) tmem_alloc<FWD_COLS>(sbase + FwdSmem::tmem);
  fence_async_smem();
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t *>(smem + FwdSmem::tmem);
  const uint32_t tlane = tmem_base + ((warp * 32u) << 16);
  uint32_t phase = 0;
  const uint32_t fmt = Fmt<T>::id;
  uint8_t *bufA = smem + FwdSmem::bufA, *bufB = smem + FwdSmem::bufB;
  const uint32_t sA = sbase + FwdSmem::bufA, sB = sbase + FwdSmem::bufB;

  const uint64_t S = *d_S;
  for (uint64_t base = (uint64_t)blockIdx.x * ROWS; base < S; base += (uint64_t)gridDim.x * ROWS) {
    const uint64_t s = base + tid;
    const bool valid = s < S;
    float v[16];
    // ---- layer input: e row -> bufA
    for (uint32_t c0 = 0; c0 < LF; c0 += 8) {
#pragma unroll
      for (int j = 0; j < 8; ++j) v[j] = valid ? ws.e[(size_t)(c0 + j) * ws.cap + s] : 0.f;
      store8<T>(bufA, ROWS, tid, c0, v);
    }
    fence_async_smem(); fence_before(); __syncthreads();
    if (tid == 0) { fence_after(); issue_layer(tmem_base + COL_D1, sA, sbase + FwdSmem::wd1, LF, H, H, fmt, bar); }
    mbar_wait(bar, phase); phase ^= 1; fence_after();
    // ---- h = ReLU(.) -> bufB
#pragma unroll
    for (uint32_t c0 = 0; c0 < H; c0 += 16) {
      tmem_ld16(tlane + COL_D1 + c0, v);
      tmem_ld_wait();
#pragma unroll
      for (int j = 0; j < 16; ++j) v[j] = fmaxf(v[j], 0.f);
      store8<T>(bufB, ROWS, tid, c0, v);
      store8<T>(bufB, ROWS, tid, c0 + 8, v + 8);
      if (write_planes && valid && !density_only)
#pragma unroll
        for (int j = 0; j < 16; ++j) ws.hd[(size_t)(c0 + j) * ws.cap + s] = v[j];
    }
    fence_async_smem(); fence_before(); __syncthreads();
    if (tid == 0) { fence_after(); issue_layer(tmem_base + COL_D2, sB, sbase + FwdSmem::wd2, H, DO, DO, fmt, bar); }
    mbar_wait(bar, phase); phase ^= 1; fence_after();
    float g[16];
    tmem_ld16(tlane + COL_D2, g);
    tmem_ld_wait();
    if (valid) ws.sigma[s] = expf(fminf(fmaxf(g[0], -15.f), 15.f));
    if (density_only) { fence_before(); __syncthreads(); continue; }
    if (write_planes && valid)
#pragma unroll
      for (int j = 0; j < 16; ++j) ws.g[(size_t)j * ws.cap + s] = g[j];
    // ---- colour input [g slice, Y(d), 0 pad] -> bufA (K = 32)
    {
      float ci[CIP];
#pragma unroll
      for (int j = 0; j < (int)CIP; ++j) ci[j] = 0.f;
      for (uint32_t j = 0; j < ms.geo_cnt; ++j) ci[j] = g[ms.geo_off + j];
      float dx = 0.f, dy = 0.f, dz = 1.f;
      if (valid) {
        const uint32_t ray = ws.s_ray[s];
        dx = __ldg(dirs + 3 * (size_t)ray); dy = __ldg(dirs + 3 * (size_t)ray + 1); dz = __ldg(dirs + 3 * (size_t)ray + 2);
      }
      float Y[16];
      sh_row(ms.sh_degree, dx, dy, dz, Y);
      for (uint32_t j = 0; j < ms.n_sh; ++j) ci[ms.geo_cnt + j] = Y[j];
#pragma unroll
      for (uint32_t c0 = 0; c0 < CIP; c0 += 8) store8<T>(bufA, ROWS, tid, c0, ci + c0);
    }
    fence_async_smem(); fence_before(); __syncthreads();
    if (tid == 0) { fence_after(); issue_layer(tmem_base + COL_C1, sA, sbase + FwdSmem::wc1, CIP, H, H, fmt, bar); }
    mbar_wait(bar, phase); phase ^= 1; fence_after();
#pragma unroll
    for (uint32_t c0 = 0; c0 < H; c0 += 16) {
      tmem_ld16(tlane + COL_C1 + c0, v);
      tmem_ld_wait();
#pragma unroll
      for (int j = 0; j < 16; ++j) v[j] = fmaxf(v[j], 0.f);
      store8<T>(bufB, ROWS, tid, c0, v);
      store8<T>(bufB, ROWS, tid, c0 + 8, v + 8);
      if (write_planes && valid)
#pragma unroll
        for (int j = 0; j < 16; ++j) ws.h1[(size_t)(c0 + j) * ws.cap + s] = v[j];
    }
    uint32_t sLast = sB;
    if (ms.n_color_layers == 2) {
      fence_async_smem(); fence_before(); __syncthreads();
      if (tid == 0) { fence_after(); issue_layer(tmem_base + COL_C2, sB, sbase + FwdSmem::wc2, H, H, H, fmt, bar); }
      mbar_wait(bar, phase); phase ^= 1; fence_after();
#pragma unroll
      for (uint32_t c0 = 0; c0 < H; c0 += 16) {
        tmem_ld16(tlane + COL_C2 + c0, v);
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 16; ++j) v[j] = fmaxf(v[j], 0.f);
        store8<T>(bufA, ROWS, tid, c0, v);
        store8<T>(bufA, ROWS, tid, c0 + 8, v + 8);
        if (write_planes && valid)
#pragma unroll
          for (int j = 0; j < 16; ++j) ws.h2[(size_t)(c0 + j) * ws.cap + s] = v[j];
      }
      sLast = sA;
    }
    fence_async_smem(); fence_before(); __syncthreads();
    if (tid == 0) { fence_after(); issue_layer(tmem_base + COL_C3, sLast, sbase + FwdSmem::wc3, H, 16, 16, fmt, bar); }
    mbar_wait(bar, phase); phase ^= 1; fence_after();
    tmem_ld16(tlane + COL_C3, v);
    tmem_ld_wait();
    if (valid) {
#pragma unroll
      for (int c = 0; c < 3; ++c) ws.rgb[3 * s + c] = 1.f / (1.f + expf(-v[c]));
    }
    fence_before();
    __syncthreads();
  }
  fence_before();
  __syncthreads();
  if (warp == 0) tmem_free<FWD_COLS>(tmem_base);
}


// ------------------------------------------------------------------------------------- backward
// S11 on tcgen05.  Per layer and tile, two kinds of MMA read the same two shared-memory tiles:
//   dgrad  dX[128 x n_in]   = dY[128 x n_out] * W          A = dY (K-major), B = W^T tile (K-major)
//   wgrad  G [n_in x n_out] += X^T * dY over the 128 samples  A = X, B = dY, both viewed MN-major
// The wgrad accumulators stay in TMEM across ALL tiles of the persistent CTA (one flush of ~11 K
// atomics per CTA at the end); thread r owns sample row r for dgrad and feature row r for wgrad.
constexpr uint32_t COL_G = 0;                                   // dgrad result, reused per layer (<= 64 cols)
constexpr uint32_t GW_C3 = 64, GW_C2 = 80, GW_C1 = 144, GW_D2 = 208, GW_D1 = 224, BWD_COLS = 512;

struct BwdSmem {
  static constexpr uint32_t wt_c3 = 0;                          // [N=64][K=16]
  static constexpr uint32_t wt_c2 = wt_c3 + H * 16 * 2;         // [64][64]
  static constexpr uint32_t wt_c1 = wt_c2 + H * H * 2;          // [32][64]
  static constexpr uint32_t wt_d2 = wt_c1 + CIP * H * 2;        // [64][16]
  static constexpr uint32_t wt_d1 = wt_d2 + H * 16 * 2;         // [LF<=64][64]
  static constexpr uint32_t bufX = wt_d1 + 64 * H * 2;          // [128][128] (features >= 64 stay zero)
  static constexpr uint32_t bufY = bufX + ROWS * 128 * 2;       // [128][64]
  static constexpr uint32_t bar = bufY + ROWS * H * 2;
  static constexpr uint32_t tmem = bar + 8;
  static constexpr uint32_t total = tmem + 8;
};

// transposed operand tile for dgrad: element (i, o) = W[o][i], tile [NP = n_in pad][KP = n_out pad]
template <typename T>
__device__ void stage_weight_t(uint8_t *tile, const float *__restrict__ W, uint32_t n_out, uint32_t n_in, uint32_t NP,
                               uint32_t KP) {
  for (uint32_t idx = threadIdx.x; idx < NP * KP; idx += blockDim.x) {
    const uint32_t i = idx / KP, o = idx - i * KP;
    const float v = (i < n_in && o < n_out) ? __ldg(W + o * n_in + i) : 0.f;
    *reinterpret_cast<T *>(tile + tile_off(NP, i, o)) = T(v);
  }
}

// wgrad k-steps over the 128 samples: G[128 (feature i) x N (output o)] (+)= X^T dY
__device__ __forceinline__ void issue_wgrad(uint32_t tmem_d, uint32_t x_saddr, uint32_t y_saddr, uint32_t N, uint32_t fmt,
                                            uint32_t accumulate) {
  const uint32_t idesc = make_idesc(fmt, 128, N, 1, 1);
  for (uint32_t k = 0; k < ROWS / 16; ++k) {
    const uint64_t da = make_desc(x_saddr + k * 256, 128, PANEL);   // MN-major: LBO = next 8 samples, SBO = next 8 features
    const uint64_t db = make_desc(y_saddr + k * 256, 128, PANEL);
    mma_ss(tmem_d, da, db, idesc, accumulate | (k > 0));
  }
}

// this thread's sample row of a [n_cols][cap] fp32 plane array -> 16-bit row of `buf`; returns the
// ReLU mask (bit c set iff x_c > 0)
template <typename T>
__device__ __forceinline__ uint64_t row_from_planes(uint8_t *buf, const float *__restrict__ planes, uint64_t cap,
                                                    uint32_t n_cols, uint64_t s, bool valid) {
  uint64_t mask = 0;
  float v[8];
  for (uint32_t c0 = 0; c0 < n_cols; c0 += 8) {
#pragma unroll
    for (int j = 0; j < 8; ++j) {
      v[j] = valid ? planes[(size_t)(c0 + j) * cap + s] : 0.f;
      if (v[j] > 0.f) mask |= 1ull << (c0 + j);
    }
    store8<T>(buf, ROWS, threadIdx.x, c0, v);
  }
  return mask;
}

template <typename T>
__global__ void __launch_bounds__(128, 1) mlp_backward_tc_kernel(MlpShape ms, const float *__restrict__ Wm,
                                                                 float *__restrict__ gradW, const float *__restrict__ dirs,
                                                                 Workspace ws, const uint32_t *__restrict__ d_S) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t tid = threadIdx.x, warp = tid >> 5;
  const uint32_t sbase = smem_u32(smem);
  const uint32_t bar = sbase + BwdSmem::bar;
  const uint32_t LF = ms.LF;
  const uint64_t S = *d_S;
  if ((uint64_t)blockIdx.x * ROWS >= S) return;   // CTA without tiles: nothing allocated yet

  stage_weight_t<T>(smem + BwdSmem::wt_c3, Wm + ms.o_c3, 3, H, H, 16);
  if (ms.n_color_layers == 2) stage_weight_t<T>(smem + BwdSmem::wt_c2, Wm + ms.o_c2, H, H, H, H);
  stage_weight_t<T>(smem + BwdSmem::wt_c1, Wm + ms.o_c1, H, ms.Ci, CIP, H);
  stage_weight_t<T>(smem + BwdSmem::wt_d2, Wm + ms.o_d2, DO, H, H, 16);
  stage_weight_t<T>(smem + BwdSmem::wt_d1, Wm + ms.o_d1, H, LF, LF, H);
  for (uint32_t i = tid; i < ROWS * 128 * 2 / 16; i += blockDim.x) reinterpret_cast<uint4 *>(smem + BwdSmem::bufX)[i] = make_uint4(0, 0, 0, 0);
  if (tid == 0) mbar_init(bar, 1);
  if (warp == 0) tmem_alloc<BWD_COLS>(sbase + BwdSmem::tmem);
  fence_async_smem();
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t *>(smem + BwdSmem::tmem);
  const uint32_t tlane = tmem_base + ((warp * 32u) << 16);
  uint32_t phase = 0;
  const uint32_t fmt = Fmt<T>::id;
  uint8_t *bufX = smem + BwdSmem::bufX, *bufY = smem + BwdSmem::bufY;
  const uint32_t sX = sbase + BwdSmem::bufX, sY = sbase + BwdSmem::bufY;

  // loss scale (fp16 only): one power of two per step from the largest input gradient magnitude
  float scale = 1.f;
  if (Fmt<T>::id == 0) {
    const float mx = __uint_as_float(*ws.grad_absmax);
    if (mx > 0.f && isfinite(mx)) scale = exp2f(fminf(fmaxf(floorf(8.f - log2f(mx)), -24.f), 30.f));
  }
  const float inv_scale = 1.f / scale;
  uint32_t acc = 0;   // wgrad accumulate flag (0 on the CTA's first tile)

  for (uint64_t base = (uint64_t)blockIdx.x * ROWS; base < S; base += (uint64_t)gridDim.x * ROWS) {
    const uint64_t s = base + tid;
    const bool valid = s < S;
    float v[16];
    // ---- colour output layer: dY = dL/dc * c (1 - c)
#pragma unroll
    for (int j = 0; j < 16; ++j) v[j] = 0.f;
    if (valid) {
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        const float col = ws.rgb[3 * s + c];
        v[c] = ws.drgb[3 * s + c] * col * (1.f - col) * scale;
      }
    }
    store8<T>(bufY, ROWS, tid, 0, v);
    store8<T>(bufY, ROWS, tid, 8, v + 8);
    uint64_t mask = row_from_planes<T>(bufX, ms.n_color_layers == 2 ? ws.h2 : ws.h1, ws.cap, H, s, valid);
    fence_async_smem(); fence_before(); __syncthreads();
    if (tid == 0) {
      fence_after();
      issue_wgrad(tmem_base + GW_C3, sX, sY, 16, fmt, acc);
      issue_layer(tmem_base + COL_G, sY, sbase + BwdSmem::wt_c3, 16, H, H, fmt, bar);
    }
    mbar_wait(bar, phase); phase ^= 1; fence_after();
    // ---- second colour hidden layer
    if (ms.n_color_layers == 2) {
#pragma unroll
      for (uint32_t c0 = 0; c0 < H; c0 += 16) {
        tmem_ld16(tlane + COL_G + c0, v);
        tmem_ld_wait();
#pragma unroll
        for (int j = 0; j < 16; ++j) v[j] = ((mask >> (c0 + j)) & 1ull) ? v[j] : 0.f;
        store8<T>(bufY, ROWS, tid, c0, v);
        store8<T>(bufY, ROWS, tid, c0 + 8, v + 8);
      }
      fence_before(); __syncthreads();          // everyone has read its accumulator row; bufX may be replaced
      mask = row_from_planes<T>(bufX, ws.h1, ws.cap, H, s, valid);
      fence_async_smem(); fence_before(); __syncthreads();
      if (tid == 0) {
        fence_after();
        issue_wgrad(tmem_base + GW_C2, sX, sY, H, fmt, acc);
        issue_layer(tmem_base + COL_G, sY, sbase + BwdSmem::wt_c2, H, H, H, fmt, bar);
      }
      mbar_wait(bar, phase); phase ^= 1; fence_after();
    }
    // ---- first colour layer: dY = d h1 (masked); X = [g slice, Y(d), 0]
#pragma unroll
    for (uint32_t c0 = 0; c0 < H; c0 += 16) {
      tmem_ld16(tlane + COL_G + c0, v);
      tmem_ld_wait();
#pragma unroll
      for (int j = 0; j < 16; ++j) v[j] = ((mask >> (c0 + j)) & 1ull) ? v[j] : 0.f;
      store8<T>(bufY, ROWS, tid, c0, v);
      store8<T>(bufY, ROWS, tid, c0 + 8, v + 8);
    }
    fence_before(); __syncthreads();
    float g0 = 0.f;
    {
      float ci[CIP];
#pragma unroll
      for (int j = 0; j < (int)CIP; ++j) ci[j] = 0.f;
      float dx = 0.f, dy = 0.f, dz = 1.f;
      if (valid) {
        g0 = ws.g[s];
        for (uint32_t j = 0; j < ms.geo_cnt; ++j) ci[j] = ws.g[(size_t)(ms.geo_off + j) * ws.cap + s];
        const uint32_t ray = ws.s_ray[s];
        dx = __ldg(dirs + 3 * (size_t)ray); dy = __ldg(dirs + 3 * (size_t)ray + 1); dz = __ldg(dirs + 3 * (size_t)ray + 2);
        float Y[16];
        sh_row(ms.sh_degree, dx, dy, dz, Y);
        for (uint32_t j = 0; j < ms.n_sh; ++j) ci[ms.geo_cnt + j] = Y[j];
      }
#pragma unroll
      for (uint32_t c0 = 0; c0 < CIP; c0 += 8) store8<T>(bufX, ROWS, tid, c0, ci + c0);
    }
    fence_async_smem(); fence_before(); __syncthreads();
    if (tid == 0) {
      fence_after();
      issue_wgrad(tmem_base + GW_C1, sX, sY, H, fmt, acc);
      issue_layer(tmem_base + COL_G, sY, sbase + BwdSmem::wt_c1, H, CIP, CIP, fmt, bar);
    }
    mbar_wait(bar, phase); phase ^= 1; fence_after();
    // ---- density output layer: dg = [geo slice of d ci] + e_0 * dL/dsigma * sigma (0 where clamped)
    {
      float dci[CIP], dg[16];
      tmem_ld16(tlane + COL_G, dci);
      tmem_ld16(tlane + COL_G + 16, dci + 16);
      tmem_ld_wait();
#pragma unroll
      for (int j = 0; j < 16; ++j) dg[j] = 0.f;
      for (uint32_t j = 0; j < ms.geo_cnt; ++j) dg[ms.geo_off + j] = dci[j];
      if (valid && g0 > -15.f && g0 < 15.f) dg[0] += ws.dsigma[s] * ws.sigma[s] * scale;
      store8<T>(bufY, ROWS, tid, 0, dg);
      store8<T>(bufY, ROWS, tid, 8, dg + 8);
    }
    fence_before(); __syncthreads();
    mask = row_from_planes<T>(bufX, ws.hd, ws.cap, H, s, valid);
    fence_async_smem(); fence_before(); __syncthreads();
    if (tid == 0) {
      fence_after();
      issue_wgrad(tmem_base + GW_D2, sX, sY, 16, fmt, acc);
      issue_layer(tmem_base + COL_G, sY, sbase + BwdSmem::wt_d2, 16, H, H, fmt, bar);
    }
    mbar_wait(bar, phase); phase ^= 1; fence_after();
    // ---- density hidden layer: dY = d hd (masked); X = e
#pragma unroll
    for (uint32_t c0 = 0; c0 < H; c0 += 16) {
      tmem_ld16(tlane + COL_G + c0, v);
      tmem_ld_wait();
#pragma unroll
      for (int j = 0; j < 16; ++j) v[j] = ((mask >> (c0 + j)) & 1ull) ? v[j] : 0.f;
      store8<T>(bufY, ROWS, tid, c0, v);
      store8<T>(bufY, ROWS, tid, c0 + 8, v + 8);
    }
    fence_before(); __syncthreads();
    row_from_planes<T>(bufX, ws.e, ws.cap, LF, s, valid);
    fence_async_smem(); fence_before(); __syncthreads();
    if (tid == 0) {
      fence_after();
      issue_wgrad(tmem_base + GW_D1, sX, sY, H, fmt, acc);
      issue_layer(tmem_base + COL_G, sY, sbase + BwdSmem::wt_d1, H, LF, LF, fmt, bar);
    }
    mbar_wait(bar, phase); phase ^= 1; fence_after();
    // ---- dL/de -> planes
    for (uint32_t c0 = 0; c0 < LF; c0 += 16) {
      tmem_ld16(tlane + COL_G + c0, v);
      tmem_ld_wait();
      if (valid)
#pragma unroll
        for (int j = 0; j < 16; ++j) ws.de[(size_t)(c0 + j) * ws.cap + s] = v[j] * inv_scale;
    }
    fence_before(); __syncthreads();
    acc = 1;
  }
  // ---- flush the CTA's weight gradients: thread i holds feature row i of every G = X^T dY
  fence_after();
  auto flush = [&](uint32_t col, uint32_t g_off, uint32_t n_out, uint32_t n_in, uint32_t ncols) {
    float v[16];
    for (uint32_t c0 = 0; c0 < ncols; c0 += 16) {
      tmem_ld16(tlane + col + c0, v);
      tmem_ld_wait();
      if (tid < n_in)
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const uint32_t o = c0 + j;
          if (o < n_out && v[j] != 0.f) atomicAdd(gradW + g_off + o * n_in + tid, v[j] * inv_scale);
        }
    }
  };
  flush(GW_C3, ms.o_c3, 3, H, 16);
  if (ms.n_color_layers == 2) flush(GW_C2, ms.o_c2, H, H, H);
  flush(GW_C1, ms.o_c1, H, ms.Ci, H);
  flush(GW_D2, ms.o_d2, DO, H, 16);
  flush(GW_D1, ms.o_d1, H, LF, H);
  fence_before();
  __syncthreads();
  if (warp == 0) tmem_free<BWD_COLS>(tmem_base);
}

}  // namespace

bool mlp_tc_supported(const MlpShape &ms) {
  return ms.Hd == H && ms.Hc == H && ms.Do == DO && ms.LF % 16 == 0 && ms.LF >= 16 && ms.LF <= 64 && ms.Ci <= CIP &&
         ms.n_sh <= 16 && ms.geo_off + ms.geo_cnt <= DO;
}

int launch_mlp_forward_tc(const MlpShape &ms, int bf16, const float *theta_mlp, const float *dirs, const Workspace &ws,
                          const uint32_t *d_S, int density_only, int write_planes, int n_sms, cudaStream_t st) {
  const size_t smem = FwdSmem::total;
  if (bf16) {
    cudaFuncSetAttribute(mlp_forward_tc_kernel<__nv_bfloat16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    mlp_forward_tc_kernel<__nv_bfloat16><<<2 * n_sms, 128, smem, st>>>(ms, theta_mlp, dirs, ws, d_S, density_only, write_planes);
  } else {
    cudaFuncSetAttribute(mlp_forward_tc_kernel<__half>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    mlp_forward_tc_kernel<__half><<<2 * n_sms, 128, smem, st>>>(ms, theta_mlp, dirs, ws, d_S, density_only, write_planes);
  }
  return 1;
}

int launch_mlp_backward_tc(const MlpShape &ms, int bf16, const float *theta_mlp, float *grad_mlp, const float *dirs,
                           const Workspace &ws, const uint32_t *d_S, int n_sms, cudaStream_t st) {
  const size_t smem = BwdSmem::total;
  if (bf16) {
    cudaFuncSetAttribute(mlp_backward_tc_kernel<__nv_bfloat16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    mlp_backward_tc_kernel<__nv_bfloat16><<<n_sms, 128, smem, st>>>(ms, theta_mlp, grad_mlp, dirs, ws, d_S);
  } else {
    cudaFuncSetAttribute(mlp_backward_tc_kernel<__half>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    mlp_backward_tc_kernel<__half><<<n_sms, 128, smem, st>>>(ms, theta_mlp, grad_mlp, dirs, ws, d_S);
  }
  return 1;
}
