// mlp_tc.cu — S5/S6/S7 and S11 on the 5th-generation tensor cores: the density and colour MLPs of
// PAPER.md:143,151 as 128-sample tcgen05.mma tiles (M = 128 samples, N = layer width, K = input
// width; 16-bit operands, fp32 accumulators in TMEM).
//
// A group of 4 warps owns a 128-sample tile; thread r owns sample row r (TMEM lane = sample row): it
// reads its accumulator row back with tcgen05.ld, applies the activation and writes its row of the
// next layer's A operand; ONE elected thread issues the layer's tcgen05.mma k-steps and a
// tcgen05.commit onto an mbarrier the group waits on.  Activations never leave the SM between layers.
//
// Forward (mlp_forward_tc_kernel): one persistent CTA per SM holding FWD_GROUPS = 4 such groups,
// each a pipeline of its own (own tiles, own 128 TMEM columns, own mbarriers, bar.sync on a named
// barrier of 128 threads), so four dependent layer chains hide each other's MMA issue-to-commit
// latency.  On the two-term training path the next layer's A operand goes straight into tensor
// memory (tcgen05.st by the thread that owns the row: hi at +64, lo at +96 of the group's columns)
// and the MMAs take A from TMEM (.ts form); only the first layer's A (the encoder's blob, by TMA)
// and the weights sit in shared memory.  The plain 16-bit forward (render, occupancy refresh) keeps
// its A operand in shared memory (UMMA canonical no-swizzle layout: 16-byte chunks at a 16 B stride
// across threads, conflict-free), which measured faster there.
//
// Backward (mlp_backward_tc_kernel): 2 CTAs per SM (TMEM bounds it) of 8 epilogue warps, one MMA-
// issuing warp and one TMA warp; a three-slot ring of TMA-loaded saved activations X and two buffers
// for the gradients Y; per layer the data gradient's MMAs are issued and committed BEFORE the weight
// gradient's, so the next layer's epilogue starts while the weight-gradient MMAs still run.
//
// Everything that crosses HBM is stored as the exact byte image of the shared-memory operand tile
// ("blob": [tile][8-column panel][128 rows][8 x 16 bit]), so it comes back with ONE TMA bulk copy
// (cp.async.bulk, no tensor map needed) straight into the MMA operand buffer: the encoder's output
// e, the activations saved for the backward pass, and the 16-bit weight images (packed once per
// step by pack_weights_kernel, not converted per CTA).
//
// Forward precision: every forward operand is carried as a two-term 16-bit expansion x = hi + lo
// (hi = round16(x), lo = round16(x - hi)) and each layer issues three MMA groups into the same fp32
// accumulator, hi*hi + lo*hi + hi*lo.  The tensor-core time is negligible here, and the forward
// pre-activations become accurate to ~2^-16 or better, so the ReLU masks the backward pass uses agree with the
// float64 oracle (a plain 16-bit forward flips masks of near-zero pre-activations, which alone
// costs 1-3 % of relative L2 error on the fine-level table gradients).
#include "nsm_internal.cuh"
#include "tc_common.cuh"

namespace {

using namespace tc;

constexpr uint32_t H = 64;      // hidden width of both MLPs on this path
constexpr uint32_t DO = 16;     // density MLP outputs
constexpr uint32_t CIP = 32;    // colour-MLP input width padded to a k-step multiple
constexpr uint32_t ROWS = NSM_TILE;
constexpr uint32_t PANEL = ROWS * 16;  // bytes of one 8-column panel of a 128-row tile

// ---- weight images (byte images of the shared-memory weight regions) ---------------------------
// forward: B tiles [N = n_out pad][K = n_in pad] (K-major);  backward: transposed tiles [n_in pad][n_out pad]
struct WImg {
  // forward region
  static constexpr uint32_t f_d1 = 0;                       // [64][64 max]  (LF <= 64 columns used)
  static constexpr uint32_t f_d2 = f_d1 + H * 64 * 2;       // [16][64]
  static constexpr uint32_t f_c1 = f_d2 + DO * H * 2;       // [64][32]
  static constexpr uint32_t f_c2 = f_c1 + H * CIP * 2;      // [64][64]
  static constexpr uint32_t f_c3 = f_c2 + H * H * 2;        // [16][64]
  static constexpr uint32_t f_total = f_c3 + 16 * H * 2;    // 24576
  // backward region
  static constexpr uint32_t b_c3 = 0;                       // [64][16]
  static constexpr uint32_t b_c2 = b_c3 + H * 16 * 2;       // [64][64]
  static constexpr uint32_t b_c1 = b_c2 + H * H * 2;        // [32][64]
  static constexpr uint32_t b_d2 = b_c1 + CIP * H * 2;      // [64][16]
  static constexpr uint32_t b_d1 = b_d2 + H * 16 * 2;       // [64 max][64]
  static constexpr uint32_t b_total = b_d1 + 64 * H * 2;    // 24576
};

// where the five weight matrices live in the canonical fp32 block and in the two images
struct MatImg { uint32_t off, n_out, n_in, f_off, f_NP, f_KP, b_off, b_NP, b_KP; };
__device__ __forceinline__ MatImg mat_img(const MlpShape &ms, uint32_t i) {
  switch (i) {
    case 0: return {ms.o_d1, H, ms.LF, WImg::f_d1, H, ms.LF, WImg::b_d1, ms.LF, H};
    case 1: return {ms.o_d2, DO, H, WImg::f_d2, DO, H, WImg::b_d2, H, 16};
    case 2: return {ms.o_c1, H, ms.Ci, WImg::f_c1, H, CIP, WImg::b_c1, CIP, H};
    case 3: return {ms.o_c2, ms.n_color_layers == 2 ? H : 0, H, WImg::f_c2, H, H, WImg::b_c2, H, H};
    default: return {ms.o_c3, 3, H, WImg::f_c3, 16, H, WImg::b_c3, H, 16};
  }
}

// one weight W[n][k] = v -> forward image (hi and lo terms, element (n, k)) and backward image (element (k, n))
template <typename T>
__device__ __forceinline__ void put_weight(const MatImg &m, uint32_t n, uint32_t k, float v, uint8_t *img_f, uint8_t *img_b) {
  const T hi = T(v);
  *reinterpret_cast<T *>(img_f + m.f_off + tile_off(m.f_NP, n, k)) = hi;
  *reinterpret_cast<T *>(img_f + WImg::f_total + m.f_off + tile_off(m.f_NP, n, k)) = T(v - (float)hi);
  *reinterpret_cast<T *>(img_b + m.b_off + tile_off(m.b_NP, k, n)) = T(v);
}

// fp32 master weights -> both 16-bit images, padding included (after nsm_set_params / at creation).
template <typename T>
__global__ void pack_weights_kernel(MlpShape ms, const float *__restrict__ Wm, uint8_t *__restrict__ img_f,
                                    uint8_t *__restrict__ img_b) {
  const MatImg m = mat_img(ms, blockIdx.x);
  // forward tile: element (n, k) = W[n][k];  backward tile: element (i, o) = W[o][i]
  for (uint32_t idx = threadIdx.x; idx < m.f_NP * m.f_KP; idx += blockDim.x) {
    const uint32_t n = idx / m.f_KP, k = idx - n * m.f_KP;
    const float v = (n < m.n_out && k < m.n_in) ? Wm[m.off + n * m.n_in + k] : 0.f;
    const T hi = T(v);
    *reinterpret_cast<T *>(img_f + m.f_off + tile_off(m.f_NP, n, k)) = hi;
    *reinterpret_cast<T *>(img_f + WImg::f_total + m.f_off + tile_off(m.f_NP, n, k)) = T(v - (float)hi);   // lo image
  }
  for (uint32_t idx = threadIdx.x; idx < m.b_NP * m.b_KP; idx += blockDim.x) {
    const uint32_t i = idx / m.b_KP, o = idx - i * m.b_KP;
    const float v = (i < m.n_in && o < m.n_out) ? Wm[m.off + o * m.n_in + i] : 0.f;
    *reinterpret_cast<T *>(img_b + m.b_off + tile_off(m.b_NP, i, o)) = T(v);
  }
}

// Sum of the per-CTA weight-gradient slices written by mlp_backward_tc_kernel: CTA c wrote a slice iff it had a
// tile, i.e. c < min(n_ctas, ceil(S / 128)).  Four warps per 32 weights: warp q adds slices q, q+4, ... (each load
// is a coalesced 128 B row segment, eight in flight), then the four partial sums meet in shared memory.
__device__ __forceinline__ float sum_wgrad_parts(const float *__restrict__ parts, uint32_t n_mlp, uint32_t n_parts, uint32_t p,
                                                 uint32_t q, float *red /* [4][32] */) {
  float acc = 0.f;
  if (p < n_mlp) {
    uint32_t c = q;
    for (; c + 28 < n_parts; c += 32) {
      float t[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) t[u] = parts[(size_t)(c + 4 * u) * n_mlp + p];
#pragma unroll
      for (int u = 0; u < 8; ++u) acc += t[u];
    }
    for (; c < n_parts; c += 4) acc += parts[(size_t)c * n_mlp + p];
  }
  red[q * 32 + (threadIdx.x & 31)] = acc;
  __syncthreads();
  return red[threadIdx.x & 31] + red[32 + (threadIdx.x & 31)] + red[64 + (threadIdx.x & 31)] + red[96 + (threadIdx.x & 31)];
}

// slices -> mlp_grad (nsm_backward: the gradient is left in place for the debug getter / nsm_apply_adam)
__global__ void __launch_bounds__(128) reduce_wgrad_kernel(const float *__restrict__ parts, uint32_t n_mlp, uint32_t n_ctas,
                                                           const uint32_t *__restrict__ d_S, float *__restrict__ grad) {
  __shared__ float red[128];
  const uint32_t tiles = (*d_S + ROWS - 1) / ROWS, n_parts = tiles < n_ctas ? tiles : n_ctas;
  const uint32_t p = blockIdx.x * 32 + (threadIdx.x & 31), q = threadIdx.x >> 5;
  const float g = sum_wgrad_parts(parts, n_mlp, n_parts, p, q, red);
  if (q == 0 && p < n_mlp) grad[p] += g;
}

// S13 on the MLP weights (all of them, every step) fused with the reduction of the weight-gradient slices and the
// image refresh: the thread of weight p (warp 0 of its block) updates theta, m, v, clears the gradient and writes the
// weight's three 16-bit image elements.  Padding elements of the images stay zero from pack_weights_kernel.
// n_ctas = 0: the gradient is already complete in grad[] (after nsm_backward or nsm_debug_set_grad).
template <typename T>
__global__ void __launch_bounds__(128) adam_pack_kernel(MlpShape ms, float *__restrict__ theta, float *__restrict__ m_,
                                                        float *__restrict__ v_, float *__restrict__ grad, uint8_t *__restrict__ img_f,
                                                        uint8_t *__restrict__ img_b, AdamConst c, const float *__restrict__ parts,
                                                        uint32_t n_ctas, const uint32_t *__restrict__ d_S, unsigned long long *tl) {
  __shared__ float red[128];
  pdl_wait();
  pdl_trigger();
  tl_mark(tl, K_ADAM_MLP, 0);
  const uint32_t p = blockIdx.x * 32 + (threadIdx.x & 31), q = threadIdx.x >> 5;
  float g = 0.f;
  if (n_ctas) {
    const uint32_t tiles = (*d_S + ROWS - 1) / ROWS;
    g = sum_wgrad_parts(parts, ms.n_mlp, tiles < n_ctas ? tiles : n_ctas, p, q, red);
  }
  if (q != 0 || p >= ms.n_mlp) return;
  g += grad[p];
  float th = theta[p], mm = m_[p], vv = v_[p];
  adam_one(th, mm, vv, g, c);
  theta[p] = th; m_[p] = mm; v_[p] = vv; grad[p] = 0.f;
  const uint32_t mi = p >= ms.o_c3 ? 4u : (p >= ms.o_c2 && ms.n_color_layers == 2) ? 3u : p >= ms.o_c1 ? 2u : p >= ms.o_d2 ? 1u : 0u;
  const MatImg mt = mat_img(ms, mi);
  const uint32_t k0 = p - mt.off, n = k0 / mt.n_in, k = k0 - n * mt.n_in;
  put_weight<T>(mt, n, k, th, img_f, img_b);
  tl_mark(tl, K_ADAM_MLP, 1);
}

// issue the k-steps of one layer: D[128 x N] = A[128 x K] * B[N x K]^T, both K-major.  The descriptors of consecutive
// k-steps differ in their 14-bit address field only (two 8-column panels further): one add per operand and MMA.
__device__ __forceinline__ void issue_layer(uint32_t tmem_d, uint32_t a_saddr, uint32_t b_saddr, uint32_t K, uint32_t N,
                                            uint32_t NP, uint32_t fmt, uint32_t bar_saddr) {
  const uint32_t idesc = make_idesc(fmt, 128, N, 0, 0);
  uint64_t da = make_desc(a_saddr, PANEL, 128), db = make_desc(b_saddr, NP * 16, 128);
  const uint64_t sa = (2 * PANEL) >> 4, sb = (2 * NP * 16) >> 4;
  for (uint32_t k = 0; k < K / 16; ++k) {
    mma_ss(tmem_d, da, db, idesc, k > 0);
    da += sa; db += sb;
  }
  mma_commit(bar_saddr);
}

// the same with two-term operands: D = A_hi B_hi + A_lo B_hi + A_hi B_lo (lo tiles sit a_lo / b_lo bytes behind)
__device__ __forceinline__ void issue_layer_split(uint32_t tmem_d, uint32_t a_saddr, uint32_t a_lo, uint32_t b_saddr,
                                                  uint32_t b_lo, uint32_t K, uint32_t N, uint32_t NP, uint32_t fmt,
                                                  uint32_t bar_saddr) {
  const uint32_t idesc = make_idesc(fmt, 128, N, 0, 0);
  const uint64_t da0 = make_desc(a_saddr, PANEL, 128), db0 = make_desc(b_saddr, NP * 16, 128);
  const uint64_t sa = (2 * PANEL) >> 4, sb = (2 * NP * 16) >> 4;
#pragma unroll
  for (uint32_t term = 0; term < 3; ++term) {
    uint64_t da = da0 + (term == 1 ? (uint64_t)(a_lo >> 4) : 0ull), db = db0 + (term == 2 ? (uint64_t)(b_lo >> 4) : 0ull);
    for (uint32_t k = 0; k < K / 16; ++k) {
      mma_ss(tmem_d, da, db, idesc, (term | k) > 0);
      da += sa; db += sb;
    }
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

// 16 accumulator columns -> (optional ReLU) -> this thread's row of a shared tile and of a global blob tile
template <typename T, bool RELU>
__device__ __forceinline__ void emit16(float *v, uint8_t *smem_tile, uint8_t *blob_tile, uint32_t row, uint32_t c0, bool valid) {
  if (RELU) {
#pragma unroll
    for (int j = 0; j < 16; ++j) v[j] = fmaxf(v[j], 0.f);
  }
  uint4 q0, q1;
  q0.x = pack2<T>(v[0], v[1]); q0.y = pack2<T>(v[2], v[3]); q0.z = pack2<T>(v[4], v[5]); q0.w = pack2<T>(v[6], v[7]);
  q1.x = pack2<T>(v[8], v[9]); q1.y = pack2<T>(v[10], v[11]); q1.z = pack2<T>(v[12], v[13]); q1.w = pack2<T>(v[14], v[15]);
  const uint32_t o0 = tile_off(ROWS, row, c0), o1 = tile_off(ROWS, row, c0 + 8);
  *reinterpret_cast<uint4 *>(smem_tile + o0) = q0;
  *reinterpret_cast<uint4 *>(smem_tile + o1) = q1;
  if (blob_tile) {   // rows of invalid samples are stored as zeros so the backward wgrad never sees garbage
    const uint4 z = make_uint4(0, 0, 0, 0);
    *reinterpret_cast<uint4 *>(blob_tile + o0) = valid ? q0 : z;
    *reinterpret_cast<uint4 *>(blob_tile + o1) = valid ? q1 : z;
  }
}

// two-term version: hi -> smem_tile and blob, lo -> smem_tile + lo_off
template <typename T, bool RELU>
__device__ __forceinline__ void emit16s(float *v, uint8_t *smem_tile, uint32_t lo_off, uint8_t *blob_tile, uint32_t row,
                                        uint32_t c0, bool valid) {
  if (RELU) {
    // fp16 rounds 0 < h < 2^-25 to zero; the backward pass reads its ReLU mask off the stored value (h > 0), so a positive
    // activation is raised to at least the smallest fp16 subnormal, 2^-24: the mask is then exactly [pre-activation > 0]
    constexpr float tiny = Fmt<T>::id == 0 ? 5.9604644775390625e-08f : 0.f;
#pragma unroll
    for (int j = 0; j < 16; ++j) v[j] = v[j] > 0.f ? fmaxf(v[j], tiny) : 0.f;
  }
  uint32_t hi[8], lo[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    hi[j] = pack2<T>(v[2 * j], v[2 * j + 1]);
    const float2 h = unpack2<T>(hi[j]);
    lo[j] = pack2<T>(v[2 * j] - h.x, v[2 * j + 1] - h.y);
  }
  const uint32_t o0 = tile_off(ROWS, row, c0), o1 = tile_off(ROWS, row, c0 + 8);
  *reinterpret_cast<uint4 *>(smem_tile + o0) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
  *reinterpret_cast<uint4 *>(smem_tile + o1) = make_uint4(hi[4], hi[5], hi[6], hi[7]);
  *reinterpret_cast<uint4 *>(smem_tile + lo_off + o0) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
  *reinterpret_cast<uint4 *>(smem_tile + lo_off + o1) = make_uint4(lo[4], lo[5], lo[6], lo[7]);
  if (blob_tile) {
    const uint4 z = make_uint4(0, 0, 0, 0);
    *reinterpret_cast<uint4 *>(blob_tile + o0) = valid ? make_uint4(hi[0], hi[1], hi[2], hi[3]) : z;
    *reinterpret_cast<uint4 *>(blob_tile + o1) = valid ? make_uint4(hi[4], hi[5], hi[6], hi[7]) : z;
  }
}

// ------------------------------------------------------------------------------------- forward
constexpr uint32_t TILE_BYTES = ROWS * H * 2;   // one [128][64] 16-bit tile

// One CTA per SM runs FOUR independent tile pipelines ("groups" of 128 threads = 4 warps, one TMEM lane quarter each) that
// share one copy of the weight images.  Per tile a group walks the five layers as a chain  MMA -> accumulator read-back ->
// activation -> next layer's A operand -> next MMA; each link waits on the tensor core, so what keeps the SM busy is the
// number of chains in flight (round 1 ran two per SM, one per CTA, each CTA with its own 48 KB of weights: tensor pipe
// 12 % active, a third of all warp samples waiting on the MMA barrier, profiles/r2d).
//  - Two-term (training) forward: the activations never touch shared memory: thread r owns sample row r = TMEM lane r, and a K-major A operand in tensor
//    memory is exactly "lane = row, two 16-bit K elements per 32-bit column" -- so the thread that read its accumulator row
//    back writes its row of the next layer's A operand (hi and lo terms) straight into TMEM with tcgen05.st, and the
//    next layer's MMAs take A from TMEM (no st.shared, no proxy fence, no shared-memory read of A by the tensor core).
//    Only the first layer's A, the encoder tile, comes from shared memory, where TMA puts it.  (Config 3: 66.7 -> 54.3 us.)
//    The plain forward keeps one in-place shared-memory buffer per group (see emit32).
//  - 128 TMEM columns per group: a 64-column accumulator reused by every layer (read back before the next layer's MMAs are
//    issued), 32 columns of A_hi and 32 of A_lo: 4 x 128 = 512 columns per CTA.
//  - groups synchronise on their own named barrier and mbarriers and drift apart, so one group's read-back and packing
//    overlap another's MMAs and TMA fetch.
constexpr uint32_t FWD_GROUPS = 4, FWD_GROUP_THREADS = 128, FWD_THREADS = FWD_GROUPS * FWD_GROUP_THREADS;
constexpr uint32_t FWD_COLS = 128 * FWD_GROUPS, FWD_COL_AHI = 64, FWD_COL_ALO = 96;
template <bool SPLIT>
struct FwdSmem {
  static constexpr uint32_t w = 0;                                          // weight images: hi (WImg forward region), then lo
  static constexpr uint32_t w_bytes = SPLIT ? 2 * WImg::f_total : WImg::f_total;
  static constexpr uint32_t buf_bytes = SPLIT ? 2 * TILE_BYTES : TILE_BYTES; // the TMA destination of the encoder tile (hi | lo)
  static constexpr uint32_t buf = w + w_bytes;
  static constexpr uint32_t bar_w = buf + FWD_GROUPS * buf_bytes;
  static constexpr uint32_t bar_mma = bar_w + 8;                            // [FWD_GROUPS]
  static constexpr uint32_t bar_e = bar_mma + 8 * FWD_GROUPS;               // [FWD_GROUPS]
  static constexpr uint32_t tmem = bar_e + 8 * FWD_GROUPS;
  static constexpr uint32_t total = tmem + 8;
};

// SPLIT = true: two-term (hi + lo) operands, three MMA groups per layer -- the training forward, whose ReLU masks the
// backward pass reuses and must agree with the float64 oracle.  SPLIT = false: plain 16-bit operands (one MMA group, half
// the read-back work and half the operand bytes) for the forward-only uses: render (S15) and the occupancy refresh.
template <bool SPLIT>
__device__ __forceinline__ void issue_fwd(uint32_t tmem_d, uint32_t a, uint32_t a_lo, uint32_t b, uint32_t b_lo, uint32_t K, uint32_t N,
                                          uint32_t NP, uint32_t fmt, uint32_t bar) {
  if constexpr (SPLIT) issue_layer_split(tmem_d, a, a_lo, b, b_lo, K, N, NP, fmt, bar);
  else issue_layer(tmem_d, a, b, K, N, NP, fmt, bar);
}
// the same with A in tensor memory: D[128 x N] = A[128 x K] * B[N x K]^T, A_hi at ta_hi, A_lo at ta_lo (8 columns per k-step)
template <bool SPLIT>
__device__ __forceinline__ void issue_fwd_ts(uint32_t tmem_d, uint32_t ta_hi, uint32_t ta_lo, uint32_t b_saddr, uint32_t b_lo, uint32_t K,
                                             uint32_t N, uint32_t NP, uint32_t fmt, uint32_t bar) {
  const uint32_t idesc = make_idesc(fmt, 128, N, 0, 0);
  const uint64_t db0 = make_desc(b_saddr, NP * 16, 128), sb = (2 * NP * 16) >> 4;
#pragma unroll
  for (uint32_t term = 0; term < (SPLIT ? 3u : 1u); ++term) {
    uint32_t ta = term == 1 ? ta_lo : ta_hi;
    uint64_t db = db0 + (term == 2 ? (uint64_t)(b_lo >> 4) : 0ull);
    for (uint32_t k = 0; k < K / 16; ++k) {
      mma_ts(tmem_d, ta, db, idesc, (term | k) > 0);
      ta += 8; db += sb;
    }
  }
  mma_commit(bar);
}
// barrier of one 128-thread group (barrier 0 is __syncthreads)
__device__ __forceinline__ void group_bar(uint32_t grp) { asm volatile("bar.sync %0, 128;" ::"r"(grp + 1u) : "memory"); }

// 32 values of this thread's row (columns c0 .. c0+31 of a layer's output) -> (optional ReLU) -> the next layer's A operand in
// tensor memory (16 packed columns of A_hi, and of A_lo when SPLIT) and, when saved, the global blob tile (hi term)
template <typename T, bool RELU, bool SPLIT>
__device__ __forceinline__ void emit32_tmem(float *v, uint32_t ta_hi, uint32_t ta_lo, uint8_t *blob_tile, uint32_t row, uint32_t c0,
                                            bool valid) {
  if (RELU) {
    // fp16 rounds 0 < h < 2^-25 to zero; the backward pass reads its ReLU mask off the stored value (h > 0), so a positive
    // activation is raised to at least the smallest fp16 subnormal, 2^-24: the mask is then exactly [pre-activation > 0]
    constexpr float tiny = (SPLIT && Fmt<T>::id == 0) ? 5.9604644775390625e-08f : 0.f;
#pragma unroll
    for (int j = 0; j < 32; ++j) v[j] = v[j] > 0.f ? fmaxf(v[j], tiny) : 0.f;
  }
  uint32_t hi[16];
#pragma unroll
  for (int j = 0; j < 16; ++j) hi[j] = pack2<T>(v[2 * j], v[2 * j + 1]);
  tmem_st16(ta_hi + c0 / 2, hi);
  if constexpr (SPLIT) {
    uint32_t lo[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const float2 h = unpack2<T>(hi[j]);
      lo[j] = pack2<T>(v[2 * j] - h.x, v[2 * j + 1] - h.y);
    }
    tmem_st16(ta_lo + c0 / 2, lo);
  }
  if (blob_tile) {   // rows of invalid samples are stored as zeros so the backward wgrad never sees garbage
    const uint4 z = make_uint4(0, 0, 0, 0);
#pragma unroll
    for (int p = 0; p < 4; ++p)
      *reinterpret_cast<uint4 *>(blob_tile + tile_off(ROWS, row, c0 + 8 * p)) =
          valid ? make_uint4(hi[4 * p], hi[4 * p + 1], hi[4 * p + 2], hi[4 * p + 3]) : z;
  }
}

// the plain 16-bit forward keeps its operands in shared memory (one in-place buffer per group): with one MMA group per
// layer the chain is short and the A-from-TMEM MMAs' longer latency costs more than the shared-memory traffic they save
// (render: 2.39 ms against 2.81 ms per two views with A in TMEM)
template <typename T, bool RELU, bool SPLIT>
__device__ __forceinline__ void emit32(float *v, uint32_t tlane, uint8_t *buf, uint8_t *blob_tile, uint32_t row, uint32_t c0, bool valid) {
  if constexpr (SPLIT) emit32_tmem<T, RELU, true>(v, tlane + FWD_COL_AHI, tlane + FWD_COL_ALO, blob_tile, row, c0, valid);
  else {
    emit16<T, RELU>(v, buf, blob_tile, row, c0, valid);
    emit16<T, RELU>(v + 16, buf, blob_tile, row, c0 + 16, valid);
  }
}
// what a group does between writing an operand and the barrier before its MMAs
template <bool SPLIT>
__device__ __forceinline__ void operand_written() {
  if constexpr (SPLIT) tmem_st_wait(); else fence_async_smem();
}

// a 64-wide hidden layer's accumulator -> ReLU -> the next layer's A operand (TMEM) and, when saved, its blob tile
template <typename T, bool SPLIT>
__device__ __forceinline__ void hidden_epilogue(uint32_t tlane, uint8_t *buf, uint8_t *blob, uint32_t row, bool valid) {
  float v[32];
#pragma unroll
  for (uint32_t c0 = 0; c0 < H; c0 += 32) {   // two accumulator loads in flight
    tmem_ld16(tlane + c0, v);
    tmem_ld16(tlane + c0 + 16, v + 16);
    tmem_ld_wait();
    emit32<T, true, SPLIT>(v, tlane, buf, blob, row, c0, valid);
  }
  operand_written<SPLIT>();
}

// a layer after the first: A from tensor memory (two-term forward) or from the group's shared-memory buffer (plain forward)
template <bool SPLIT>
__device__ __forceinline__ void issue_next(uint32_t tcol, uint32_t sBuf, uint32_t b_saddr, uint32_t K, uint32_t N, uint32_t NP,
                                           uint32_t fmt, uint32_t bar) {
  if constexpr (SPLIT) issue_fwd_ts<true>(tcol, tcol + FWD_COL_AHI, tcol + FWD_COL_ALO, b_saddr, WImg::f_total, K, N, NP, fmt, bar);
  else issue_layer(tcol, sBuf, b_saddr, K, N, NP, fmt, bar);
}

template <typename T, bool SPLIT>
__global__ void __launch_bounds__(FWD_THREADS, 1) mlp_forward_tc_kernel(MlpShape ms, const float *__restrict__ dirs, Workspace ws,
                                                                       const uint32_t *__restrict__ d_S, int density_only,
                                                                       int save_blobs) {
  using SM = FwdSmem<SPLIT>;
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t tid = threadIdx.x, warp = tid >> 5;
  const uint32_t grp = tid >> 7, row = tid & 127u;          // warp & 3 = the TMEM lane quarter of rows 32 (warp & 3) .. +31
  const bool lead_warp = row < 32;                          // the group's first warp: one lane of it issues the MMAs and the TMA
  const uint32_t sbase = smem_u32(smem);
  const uint32_t bar_w = sbase + SM::bar_w, bar_mma = sbase + SM::bar_mma + 8 * grp, bar_e = sbase + SM::bar_e + 8 * grp;
  const uint32_t LF = ms.LF;
  const uint32_t e_half = LF * ROWS * 2, e_stride = 2 * e_half;   // the encoder writes hi | lo per tile
  const uint32_t e_bytes = SPLIT ? e_stride : e_half;
  // Before pdl_wait(): only data produced at least two kernels back (S from the marcher, the weight images).
  const uint64_t S = *d_S;
  const uint64_t n_tiles = (S + ROWS - 1) / ROWS;
  const bool has_tiles = blockIdx.x < n_tiles;
  if (has_tiles) {
    if (tid == 0) {
      mbar_init(bar_w, 1);
#pragma unroll
      for (uint32_t g = 0; g < FWD_GROUPS; ++g) { mbar_init(sbase + SM::bar_mma + 8 * g, 1); mbar_init(sbase + SM::bar_e + 8 * g, 1); }
      fence_async_smem();
      mbar_expect_tx(bar_w, SM::w_bytes);
      bulk_g2s(sbase + SM::w, ws.wimg_fwd, SM::w_bytes, bar_w);
    }
    if (warp == 0) tmem_alloc<FWD_COLS>(sbase + SM::tmem);
  }
  pdl_wait();
  pdl_trigger();
  if (!has_tiles) return;
  tl_mark(ws.timeline, K_MLP_FWD, 0);
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t *>(smem + SM::tmem);
  const uint32_t tcol = tmem_base + 128u * grp;                       // the group's columns: accumulator | A_hi | A_lo
  const uint32_t tlane = tcol + (((warp & 3u) * 32u) << 16);
  uint32_t ph_mma = 0, ph_e = 0;
  const uint32_t fmt = Fmt<T>::id;
  uint8_t *buf = smem + SM::buf + grp * SM::buf_bytes;
  const uint32_t sBuf = sbase + SM::buf + grp * SM::buf_bytes, sW = sbase + SM::w;
  // group g of CTA b takes tiles b + g * gridDim.x, then every 4 * gridDim.x: with few tiles every SM gets one first
  const uint64_t first_tile = blockIdx.x + (uint64_t)grp * gridDim.x, tile_stride = (uint64_t)FWD_GROUPS * gridDim.x;
  if (lead_warp) {
    if (first_tile < n_tiles && elect_one()) {   // the encoder's output: after the wait
      mbar_expect_tx(bar_e, e_bytes);
      bulk_g2s(sBuf, ws.blob_e + (size_t)first_tile * e_stride, e_bytes, bar_e);
    }
    mbar_wait(bar_w, 0);
  }

  for (uint64_t tile = first_tile; tile < n_tiles; tile += tile_stride) {
    const uint64_t s = tile * ROWS + row;
    const bool valid = s < S;
    // ---- density hidden layer: A = encoder tile (in shared memory via TMA)
    if (lead_warp) {
      mbar_wait(bar_e, ph_e);
      fence_after();
      if (elect_one()) issue_fwd<SPLIT>(tcol, sBuf, e_half, sW + WImg::f_d1, WImg::f_total, LF, H, H, fmt, bar_mma);
    }
    ph_e ^= 1;
    // the ray direction of this row's sample (two dependent global loads): in flight under the first MMAs
    float dx = 0.f, dy = 0.f, dz = 1.f;
    if (!density_only && valid) {
      const uint32_t ray = ws.s_ray[s];
      dx = __ldg(dirs + 3 * (size_t)ray); dy = __ldg(dirs + 3 * (size_t)ray + 1); dz = __ldg(dirs + 3 * (size_t)ray + 2);
    }
    mbar_wait(bar_mma, ph_mma); ph_mma ^= 1; fence_after();
    auto fetch_next_e = [&]() {   // the group's next encoder tile
      const uint64_t nxt = tile + tile_stride;
      if (lead_warp && nxt < n_tiles && elect_one()) { mbar_expect_tx(bar_e, e_bytes); bulk_g2s(sBuf, ws.blob_e + (size_t)nxt * e_stride, e_bytes, bar_e); }
    };
    if constexpr (SPLIT) fetch_next_e();   // only the first layer reads the buffer: it is free as soon as that layer's MMAs are done
    hidden_epilogue<T, SPLIT>(tlane, buf, (save_blobs && !density_only) ? ws.blob_hd + (size_t)tile * (H * ROWS * 2) : nullptr, row, valid);
    fence_before(); group_bar(grp);
    if (lead_warp) { fence_after(); if (elect_one()) issue_next<SPLIT>(tcol, sBuf, sW + WImg::f_d2, H, DO, DO, fmt, bar_mma); }
    mbar_wait(bar_mma, ph_mma); ph_mma ^= 1; fence_after();
    float g[16];
    tmem_ld16(tlane, g);
    tmem_ld_wait();
    if (valid) ws.sigma[s] = expf(fminf(fmaxf(g[0], -15.f), 15.f));
    if (density_only) {
      if constexpr (!SPLIT) fetch_next_e();   // (plain forward: the buffer held the hidden activations until now)
      fence_before(); group_bar(grp);   // every read of the accumulator is done before the next tile's MMAs
      continue;
    }
    // ---- colour input [g slice, Y(d), 0 pad] -> A operand (K = 32)
    {
      float ci[CIP];
      // mlp_tc_supported() admits only the slice (geo_offset, geo_count) = (1, 15) with 16 SH terms (configs 2-5):
      // static register indexing, no local memory
#pragma unroll
      for (int j = 0; j < 15; ++j) ci[j] = g[1 + j];
      float Y[16];
      sh_row(4, dx, dy, dz, Y);
#pragma unroll
      for (int j = 0; j < 16; ++j) ci[15 + j] = Y[j];
      ci[31] = 0.f;
      emit32<T, false, SPLIT>(ci, tlane, buf, save_blobs ? ws.blob_ci + (size_t)tile * (CIP * ROWS * 2) : nullptr, row, 0, valid);
      operand_written<SPLIT>();
    }
    fence_before(); group_bar(grp);
    if (lead_warp) { fence_after(); if (elect_one()) issue_next<SPLIT>(tcol, sBuf, sW + WImg::f_c1, CIP, H, H, fmt, bar_mma); }
    mbar_wait(bar_mma, ph_mma); ph_mma ^= 1; fence_after();
    hidden_epilogue<T, SPLIT>(tlane, buf, save_blobs ? ws.blob_h1 + (size_t)tile * (H * ROWS * 2) : nullptr, row, valid);
    if (ms.n_color_layers == 2) {
      fence_before(); group_bar(grp);
      if (lead_warp) { fence_after(); if (elect_one()) issue_next<SPLIT>(tcol, sBuf, sW + WImg::f_c2, H, H, H, fmt, bar_mma); }
      mbar_wait(bar_mma, ph_mma); ph_mma ^= 1; fence_after();
      hidden_epilogue<T, SPLIT>(tlane, buf, save_blobs ? ws.blob_h2 + (size_t)tile * (H * ROWS * 2) : nullptr, row, valid);
    }
    fence_before(); group_bar(grp);
    if (lead_warp) { fence_after(); if (elect_one()) issue_next<SPLIT>(tcol, sBuf, sW + WImg::f_c3, H, 16, 16, fmt, bar_mma); }
    mbar_wait(bar_mma, ph_mma); ph_mma ^= 1; fence_after();
    if constexpr (!SPLIT) fetch_next_e();
    {
      float v[16];
      tmem_ld16(tlane, v);
      tmem_ld_wait();
      if (valid) {
#pragma unroll
        for (int c = 0; c < 3; ++c) ws.rgb[3 * s + c] = 1.f / (1.f + expf(-v[c]));
      }
    }
    fence_before();
    group_bar(grp);   // nobody of the group may still be reading the accumulator when the next tile's first MMA is issued
  }
  fence_before();
  __syncthreads();
  if (warp == 0) tmem_free<FWD_COLS>(tmem_base);
  tl_mark(ws.timeline, K_MLP_FWD, 1);
}

// ------------------------------------------------------------------------------------- backward
// Per layer and tile, two kinds of MMA read the same two shared-memory tiles:
//   dgrad  dX[128 x n_in]   = dY[128 x n_out] * W           A = dY (K-major), B = W^T tile (K-major)
//   wgrad  G [n_in x n_out] += X^T * dY over the 128 samples   A = X, B = dY, both viewed MN-major
// The wgrad accumulators stay in TMEM across ALL tiles of the persistent CTA (one flush per CTA at
// the end); thread r owns sample row r for dgrad and feature row r for wgrad.  The saved
// activations X of the five layers arrive by TMA into two ping-pong buffers, one layer ahead.
constexpr uint32_t COL_G = 0;                                   // dgrad result, reused per layer (<= 64 cols)
// wgrad accumulators.  The first colour layer's is kept TRANSPOSED (rows = 64 outputs, 32 input columns), which
// brings the total to 256 columns: two CTAs per SM.
constexpr uint32_t GW_C3 = 64, GW_C2 = 80, GW_C1T = 144, GW_D2 = 176, GW_D1 = 192, BWD_COLS = 256;
// 8 epilogue warps (TMEM lane quarter x column half) + one warp whose elected lane issues every MMA of the CTA + one warp
// whose elected lane issues every TMA load of the saved activations
constexpr uint32_t BWD_EPI_WARPS = 8, BWD_MMA_WARP = 8, BWD_TMA_WARP = 9, BWD_THREADS = 32 * (BWD_EPI_WARPS + 2);

struct BwdSmem {
  // [X0][X1][X2][Y0][Y1][W], 16 KB tiles.  An M = 128 MMA that reads a 64-column tile MN-major also reads the 16 KB behind
  // it (rows 64..127 of its result are never used): behind every tile sits another tile, behind Y1 the weight image.
  static constexpr uint32_t tile = ROWS * H * 2;
  static constexpr uint32_t bufX = 0;                              // ring of three saved-activation tiles (TMA destinations)
  static constexpr uint32_t bufY = bufX + 3 * tile;                // two dY tiles, alternating per layer
  static constexpr uint32_t w = bufY + 2 * tile;                   // weight image (WImg backward region)
  static constexpr uint32_t bar_mma = w + WImg::b_total;
  static constexpr uint32_t bar_w = bar_mma + 8;
  static constexpr uint32_t bar_x = bar_w + 8;                     // [3]
  static constexpr uint32_t bar_y = bar_x + 24;                    // dY of the next item written (one arrival per epilogue warp)
  static constexpr uint32_t bar_fin = bar_y + 8;                   // every MMA of the CTA done
  static constexpr uint32_t bar_free = bar_fin + 8;                // [3] ring slot released (its item's wgrad done, its mask read)
  static constexpr uint32_t tmem = bar_free + 24;
  static constexpr uint32_t total = tmem + 8;
};
static_assert(WImg::b_total >= BwdSmem::tile, "the slack behind Y1 must be covered by the weight image");

// wgrad k-steps over the 128 samples: G[128 (columns of tile A) x N (columns of tile B)] (+)= A^T B
__device__ __forceinline__ void issue_wgrad(uint32_t tmem_d, uint32_t x_saddr, uint32_t y_saddr, uint32_t N, uint32_t fmt,
                                            uint32_t accumulate) {
  const uint32_t idesc = make_idesc(fmt, 128, N, 1, 1);
  uint64_t da = make_desc(x_saddr, 128, PANEL), db = make_desc(y_saddr, 128, PANEL);   // MN-major: LBO = next 8 samples, SBO = next 8 features
#pragma unroll
  for (uint32_t k = 0; k < ROWS / 16; ++k) {
    mma_ss(tmem_d, da, db, idesc, accumulate | (k > 0));
    da += 256 >> 4; db += 256 >> 4;
  }
}

// ReLU mask of columns [cb, cb+32) of this thread's row of a [128][64] activation tile in shared memory
template <typename T>
__device__ __forceinline__ uint32_t row_mask32(const uint8_t *tile, uint32_t row, uint32_t cb) {
  uint32_t mask = 0;
#pragma unroll
  for (uint32_t p = 0; p < 4; ++p) {
    const uint4 q = *reinterpret_cast<const uint4 *>(tile + (cb / 8 + p) * PANEL + row * 16);
    const uint32_t w[4] = {q.x, q.y, q.z, q.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const float2 f = unpack2<T>(w[j]);
      if (f.x > 0.f) mask |= 1u << (p * 8 + 2 * j);
      if (f.y > 0.f) mask |= 1u << (p * 8 + 2 * j + 1);
    }
  }
  return mask;
}

// dgrad columns [cb, cb+32) of this thread's row -> ReLU-masked -> bufY
template <typename T>
__device__ __forceinline__ void masked_to_Y(uint32_t tlane, uint32_t mask, uint8_t *bufY, uint32_t row, uint32_t cb) {
  float v[16];
#pragma unroll
  for (uint32_t c0 = 0; c0 < 32; c0 += 16) {
    tmem_ld16(tlane + COL_G + cb + c0, v);
    tmem_ld_wait();
#pragma unroll
    for (int j = 0; j < 16; ++j) v[j] = ((mask >> (c0 + j)) & 1u) ? v[j] : 0.f;
    emit16<T, false>(v, bufY, nullptr, row, cb + c0, true);
  }
}

// 8 epilogue warps per tile: warp w owns sample rows 32 (w & 3) .. +31 (TMEM lane quarter) and the column half (w >> 2) of
// every 64-wide dgrad; a ninth warp does nothing but issue the CTA's MMAs, a tenth nothing but the TMA loads of the saved
// activations.  Two CTAs per SM.
//
// The layers of the CTA's tiles form one sequence of items n = 0, 1, 2, ...  Item n reads its saved activation from
// X[n % 3] and its dY from Y[n % 2].  Only the item's dgrad is on the critical path (the next item's dY is computed from
// it): the MMA warp's elected lane issues the dgrad MMAs, commits them onto the barrier the epilogue warps wait on, and
// THEN issues the item's wgrad MMAs, which run under the read-back and packing of the next item.  A tcgen05.commit
// covers every MMA the thread issued before it, so when item n+1's dgrad has completed, item n's wgrad has too and
// Y[n % 2] is free for item n+2.  The ring slot X[n % 3] is released to the TMA warp (bar_free) by a commit the MMA warp
// issues once the epilogue warps have handed over item n+1, i.e. have read item n's ReLU mask; the TMA warp then
// fetches item n+3 into it.
//
// Why a warp of its own: a tcgen05.mma takes ~50 cycles to issue and an item has ~12 of them, so the issuing thread is
// busy for ~600 cycles per item; while it also owned a sample row, its share of the read-back started that much later
// than everyone else's and the whole CTA waited for it at the next barrier (measured with clock64 per phase: 2100
// cycles per item of which the issuing thread spent 600 issuing, 500 on its row mask behind the queued MMAs and 460
// on the TMA request; the request alone still cost the warp that issued it ~500 cycles per item, hence the TMA warp).
// The epilogue warps hand an item over with one mbarrier arrival per warp (bar_y) and never __syncthreads inside the
// tile loop.
template <typename T>
__global__ void __launch_bounds__(BWD_THREADS, 2) mlp_backward_tc_kernel(MlpShape ms, Workspace ws,
                                                                        const uint32_t *__restrict__ d_S) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const uint32_t tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t row = (warp & 3u) * 32u + lane, half = warp >> 2, cb = half * 32u;   // epilogue warps (half < 2)
  const bool mma_warp = warp == BWD_MMA_WARP, tma_warp = warp == BWD_TMA_WARP;
  const uint32_t sbase = smem_u32(smem);
  const uint32_t bar_mma = sbase + BwdSmem::bar_mma, bar_w = sbase + BwdSmem::bar_w;
  const uint32_t bar_y = sbase + BwdSmem::bar_y, bar_fin = sbase + BwdSmem::bar_fin;
  const uint32_t sW = sbase + BwdSmem::w;
  const uint32_t LF = ms.LF;
  const uint64_t S = *d_S;                         // from the marcher, several kernels back: safe before pdl_wait()
  const bool has_tiles = (uint64_t)blockIdx.x * ROWS < S;
  const bool two = ms.n_color_layers == 2;
  const uint32_t hbytes = H * ROWS * 2, cbytes = CIP * ROWS * 2, ebytes = LF * ROWS * 2;

  // ---- the X ring.  Loader state (identical in every lane of warp 0; the elected lane issues): the next item to fetch.
  uint64_t ld_tile = blockIdx.x;
  uint32_t ld_layer = 0, ld_slot = 0;              // layer 0..4 (1 is skipped with one hidden colour layer); ring slot
  auto load_next = [&]() {                         // the TMA warp, converged
    if (ld_tile * ROWS < S && elect_one()) {
      const uint8_t *src; uint32_t bytes;
      switch (ld_layer) {                          // the activation the layer's wgrad needs
        case 0: src = (two ? ws.blob_h2 : ws.blob_h1) + ld_tile * hbytes; bytes = hbytes; break;
        case 1: src = ws.blob_h1 + ld_tile * hbytes; bytes = hbytes; break;
        case 2: src = ws.blob_ci + ld_tile * cbytes; bytes = cbytes; break;
        case 3: src = ws.blob_hd + ld_tile * hbytes; bytes = hbytes; break;
        default: src = ws.blob_e + ld_tile * (2 * (size_t)ebytes); bytes = ebytes; break;   // the hi half of the two-term tile
      }
      const uint32_t bar = sbase + BwdSmem::bar_x + 8 * ld_slot;
      mbar_expect_tx(bar, bytes);
      bulk_g2s(sbase + BwdSmem::bufX + ld_slot * BwdSmem::tile, src, bytes, bar);
    }
    ld_layer = ld_layer == 4 ? 0u : (ld_layer == 0 && !two ? 2u : ld_layer + 1u);
    if (ld_layer == 0) ld_tile += gridDim.x;
    ld_slot = ld_slot == 2 ? 0u : ld_slot + 1u;
  };
  // consumer state: ring slot and dY buffer of the current item, barrier phases of the three slots (bit i = slot i)
  uint32_t xs = 0, ys = 0, ph_x = 0, items = 0;
  auto wait_x = [&]() { mbar_wait(sbase + BwdSmem::bar_x + 8 * xs, (ph_x >> xs) & 1u); ph_x ^= 1u << xs; };
  auto bufX = [&]() { return smem + BwdSmem::bufX + xs * BwdSmem::tile; };
  auto sX = [&]() { return sbase + BwdSmem::bufX + xs * BwdSmem::tile; };
  auto bufY = [&]() { return smem + BwdSmem::bufY + ys * BwdSmem::tile; };
  auto sY = [&]() { return sbase + BwdSmem::bufY + ys * BwdSmem::tile; };

  if (has_tiles) {   // prologue on data that is at least two kernels old (weight image, the forward pass's saved activations)
    if (tid == 0) {
      mbar_init(bar_mma, 1); mbar_init(bar_w, 1);
      mbar_init(bar_y, BWD_EPI_WARPS); mbar_init(bar_fin, 1);
      fence_async_smem();
      mbar_expect_tx(bar_w, WImg::b_total);
      bulk_g2s(sW, ws.wimg_bwd, WImg::b_total, bar_w);
    }
    if (warp == 0) {
      __syncwarp();
      tmem_alloc<BWD_COLS>(sbase + BwdSmem::tmem);
    }
    if (tma_warp) {   // the ring's barriers are this warp's own: initialise them and request the first three items
      if (lane == 0) {
        for (uint32_t i = 0; i < 3; ++i) { mbar_init(sbase + BwdSmem::bar_x + 8 * i, 1); mbar_init(sbase + BwdSmem::bar_free + 8 * i, 1); }
        fence_async_smem();
      }
      __syncwarp();
      load_next(); load_next(); load_next();
    }
  }
  pdl_wait();     // the compositor's dL/dsigma, dL/dc and gradient maximum
  pdl_trigger();
  if (!has_tiles) return;
  tl_mark(ws.timeline, K_MLP_BWD, 0);
  fence_async_smem();
  fence_before();
  __syncthreads();
  fence_after();
  const uint32_t tmem_base = *reinterpret_cast<volatile uint32_t *>(smem + BwdSmem::tmem);
  const uint32_t tlane = tmem_base + (((warp & 3u) * 32u) << 16);
  uint32_t ph_mma = 0;
  const uint32_t fmt = Fmt<T>::id;

  // loss scale (fp16 only): one power of two per step from the largest gradient entering S11
  float scale = 1.f;
  if (Fmt<T>::id == 0) {
    const float mx = __uint_as_float(*ws.grad_absmax);
    if (mx > 0.f && isfinite(mx)) scale = exp2f(fminf(fmaxf(floorf(8.f - log2f(mx)), -24.f), 30.f));
  }
  const float inv_scale = 1.f / scale;
  if (mma_warp) {
    // ---- the MMA warp: per item, wait for the item's dY (bar_y) and saved activation (its ring slot), issue
    // Behind bar_y of item n+1 the epilogue warps have read item n's ring slot for the last time (its ReLU mask), so a
    // commit issued there -- it also covers item n's wgrad MMAs -- releases the slot to the TMA warp.
    uint32_t ph_y = 0, acc = 0, issued = 0;   // acc: wgrad accumulate flag (0 on the CTA's first tile)
    mbar_wait(bar_w, 0);
#define BWD_ISSUE(WGRAD_STMT, DGRAD_STMT)                                                    \
  do {                                                                                       \
    mbar_wait(bar_y, ph_y); ph_y ^= 1;                                                       \
    if (issued && elect_one()) mma_commit(sbase + BwdSmem::bar_free + 8 * (xs == 0 ? 2u : xs - 1u)); \
    __syncwarp();                                                                            \
    wait_x();                                                                                \
    fence_after();                                                                           \
    if (elect_one()) { DGRAD_STMT; WGRAD_STMT; }                                             \
    __syncwarp();                                                                            \
    issued = 1;                                                                              \
    xs = xs == 2 ? 0u : xs + 1u; ys ^= 1u;                                                   \
  } while (0)
    for (uint64_t tile = blockIdx.x; tile * ROWS < S; tile += gridDim.x) {
      BWD_ISSUE(issue_wgrad(tmem_base + GW_C3, sX(), sY(), 16, fmt, acc),
                issue_layer(tmem_base + COL_G, sY(), sW + WImg::b_c3, 16, H, H, fmt, bar_mma));
      if (two)
        BWD_ISSUE(issue_wgrad(tmem_base + GW_C2, sX(), sY(), H, fmt, acc),
                  issue_layer(tmem_base + COL_G, sY(), sW + WImg::b_c2, H, H, H, fmt, bar_mma));
      BWD_ISSUE(issue_wgrad(tmem_base + GW_C1T, sY(), sX(), CIP, fmt, acc),                 // transposed: G^T = dY^T X
                issue_layer(tmem_base + COL_G, sY(), sW + WImg::b_c1, H, CIP, CIP, fmt, bar_mma));
      BWD_ISSUE(issue_wgrad(tmem_base + GW_D2, sX(), sY(), 16, fmt, acc),
                issue_layer(tmem_base + COL_G, sY(), sW + WImg::b_d2, 16, H, H, fmt, bar_mma));
      BWD_ISSUE(issue_wgrad(tmem_base + GW_D1, sX(), sY(), H, fmt, acc),
                issue_layer(tmem_base + COL_G, sY(), sW + WImg::b_d1, H, LF, LF, fmt, bar_mma));
      acc = 1;
    }
#undef BWD_ISSUE
    if (elect_one()) mma_commit(bar_fin);   // the last item's wgrad is still in flight
    __syncwarp();
  } else if (tma_warp) {
    // ---- the TMA warp: item j goes into ring slot j % 3 once item j - 3 has released it
    uint32_t ph_f = 0;
    while (ld_tile * ROWS < S) {
      mbar_wait(sbase + BwdSmem::bar_free + 8 * ld_slot, (ph_f >> ld_slot) & 1u);
      ph_f ^= 1u << ld_slot;
      load_next();
    }
  } else {
  // ---- the epilogue warps.  One item: this thread's part of dY is in Y[ys]; hand the item to the MMA warp, do what does
  // not need the dgrad under the MMAs' latency, wait for the dgrad, advance.
#define BWD_ITEM(UNDER_MMA_STMT)                                                             \
  do {                                                                                       \
    fence_async_smem(); fence_before(); __syncwarp();                                        \
    if (lane == 0) mbar_arrive(bar_y);                                                       \
    wait_x();                                                                                \
    UNDER_MMA_STMT;                                                                          \
    mbar_wait(bar_mma, ph_mma); ph_mma ^= 1; fence_after();                                  \
    items += 1;                                                                              \
    xs = xs == 2 ? 0u : xs + 1u; ys ^= 1u;                                                   \
  } while (0)

  // the first item's inputs (dL/dc * c (1 - c), sigma, dL/dsigma of this thread's sample): global loads, fetched for the
  // NEXT tile under the last item's MMAs
  // (raw values only: the arithmetic on them waits until the top of that tile, so nothing here stalls on the loads)
  float in_col[3] = {0.f, 0.f, 0.f}, in_dc[3] = {0.f, 0.f, 0.f}, in_sig = 0.f, in_dsig = 0.f;
  auto fetch_inputs = [&](uint64_t tile) {
    const uint64_t s = tile * ROWS + row;
    in_col[0] = in_col[1] = in_col[2] = 0.f; in_dc[0] = in_dc[1] = in_dc[2] = 0.f; in_sig = 0.f; in_dsig = 0.f;
    if (half == 0 && s < S) {
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        in_col[c] = ws.rgb[3 * s + c];
        in_dc[c] = ws.drgb[3 * s + c];
      }
      in_sig = ws.sigma[s];
      in_dsig = ws.dsigma[s];
    }
  };
  fetch_inputs(blockIdx.x);

  for (uint64_t tile = blockIdx.x; tile * ROWS < S; tile += gridDim.x) {
    const uint64_t s = tile * ROWS + row;
    const bool valid = s < S;
    float v[16];
    // ---- colour output layer: dY = dL/dc * c (1 - c); X = last hidden activations
    const float sig = in_sig, dsig = in_dsig;
    if (half == 0) {
#pragma unroll
      for (int j = 0; j < 16; ++j) v[j] = 0.f;
#pragma unroll
      for (int c = 0; c < 3; ++c) v[c] = in_dc[c] * in_col[c] * (1.f - in_col[c]) * scale;
      emit16<T, false>(v, bufY(), nullptr, row, 0, true);
    }
    uint32_t mask = 0;   // ReLU mask of the item's saved activation: needed by the NEXT item's dY, read under this item's MMAs
    BWD_ITEM(mask = row_mask32<T>(bufX(), row, cb));
    // ---- second colour hidden layer
    if (two) {
      masked_to_Y<T>(tlane, mask, bufY(), row, cb);
      BWD_ITEM(mask = row_mask32<T>(bufX(), row, cb));
    }
    // ---- first colour layer: dY = d h1 (masked); X = [g slice, Y(d), 0]
    masked_to_Y<T>(tlane, mask, bufY(), row, cb);
    BWD_ITEM((void)0);
    // ---- density output layer: dg = [geo slice of d ci] + e_0 * dL/dsigma * sigma (0 where clamped)
    if (half == 0) {
      float dci[CIP], dg[16];
      tmem_ld16(tlane + COL_G, dci);
      tmem_ld16(tlane + COL_G + 16, dci + 16);
      tmem_ld_wait();
#pragma unroll
      for (int j = 0; j < 16; ++j) dg[j] = 0.f;
#pragma unroll
      for (int j = 0; j < 15; ++j) dg[1 + j] = dci[j];   // geo slice (1, 15), see mlp_tc_supported()
      if (ws.dY && valid) {                              // row f2: dL/dY, the 16 SH slots of the colour input
#pragma unroll
        for (int j = 0; j < 16; ++j) ws.dY[(size_t)j * ws.cap + s] = dci[15 + j] * inv_scale;
      }
      // sigma = exp(clamp(g0, -15, 15)): the clamp is active iff sigma sits on a bound
      if (valid && sig > 3.0590232e-07f * 1.0001f && sig < 3269017.4f * 0.9999f) dg[0] += dsig * sig * scale;
      emit16<T, false>(dg, bufY(), nullptr, row, 0, true);
    }
    BWD_ITEM(mask = row_mask32<T>(bufX(), row, cb));
    // ---- density hidden layer: dY = d hd (masked); X = e
    masked_to_Y<T>(tlane, mask, bufY(), row, cb);
    BWD_ITEM(fetch_inputs(tile + gridDim.x));
    // ---- dL/de -> planes; the two column halves take the 16-column chunks of the LF columns alternately
    for (uint32_t c0 = half * 16; c0 < LF; c0 += 32) {
      tmem_ld16(tlane + COL_G + c0, v);
      tmem_ld_wait();
      if (valid)
#pragma unroll
        for (int j = 0; j < 16; ++j) ws.de[(size_t)(c0 + j) * ws.cap + s] = v[j] * inv_scale;
    }
    // (the next item's arrival on bar_y follows these reads of COL_G, before the MMA warp's next dgrad overwrites it)
  }
#undef BWD_ITEM
  }
  // ---- every MMA of the CTA done (the MMA warp's last commit), then flush the CTA's weight gradients
  mbar_wait(bar_fin, 0);
  fence_after();
  // Each CTA stores its sums into its own slice of ws.wgrad_part with plain, lane-coalesced stores; the slices are
  // summed by the consumer (the MLP Adam kernel, or reduce_wgrad_kernel).  Atomics onto the 9-11 K shared addresses
  // from every CTA serialise in L2 and kept the CTAs draining at exit for 40 % of the kernel (profiles/r1h).
  float *part = ws.wgrad_part + (size_t)blockIdx.x * ms.n_mlp;
  // G[i][o] = dW[o][i]: rows = input features, ncols output columns
  auto flush = [&](uint32_t col, uint32_t g_off, uint32_t n_out, uint32_t n_in, uint32_t ncols) {
    float v[16];
    for (uint32_t c0 = half * 16; c0 < ncols; c0 += 32) {
      tmem_ld16(tlane + col + c0, v);
      tmem_ld_wait();
      if (row < n_in)
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const uint32_t o = c0 + j;
          if (o < n_out) part[g_off + o * n_in + row] = v[j] * inv_scale;
        }
    }
  };
  if (!mma_warp) {
  flush(GW_C3, ms.o_c3, 3, H, 16);
  if (two) flush(GW_C2, ms.o_c2, H, H, H);
  {   // transposed accumulator: rows = outputs, columns = inputs
    float v[16];
    tmem_ld16(tlane + GW_C1T + half * 16, v);
    tmem_ld_wait();
    if (row < H)
#pragma unroll
      for (int j = 0; j < 16; ++j) {
        const uint32_t i = half * 16 + j;
        if (i < ms.Ci) part[ms.o_c1 + row * ms.Ci + i] = v[j] * inv_scale;
      }
  }
  flush(GW_D2, ms.o_d2, DO, H, 16);
  flush(GW_D1, ms.o_d1, H, LF, H);
  }
  fence_before();
  __syncthreads();
  if (warp == 0) tmem_free<BWD_COLS>(tmem_base);
  tl_mark(ws.timeline, K_MLP_BWD, 1);
}

// blob tile image -> fp32 rows [S][n_cols] (debug getter)
template <typename T>
__global__ void blob_to_rows_kernel(const uint8_t *__restrict__ blob, uint32_t n_cols, int two_term,
                                    const uint32_t *__restrict__ d_S, float *__restrict__ rows) {
  const uint64_t S = *d_S, total = S * n_cols;
  for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (uint64_t)gridDim.x * blockDim.x) {
    const uint64_t s = i / n_cols;
    const uint32_t c = (uint32_t)(i - s * n_cols);
    const size_t half = (size_t)n_cols * ROWS * 2;
    const uint8_t *p = blob + (s >> 7) * (two_term ? 2 * half : half) + tile_off(ROWS, (uint32_t)(s & 127), c);
    float v = (float)(*reinterpret_cast<const T *>(p));
    if (two_term == 1) v += (float)(*reinterpret_cast<const T *>(p + half));   // 2: hi | lo layout whose lo tile was not written
    rows[i] = v;
  }
}

}  // namespace

bool mlp_tc_supported(const MlpShape &ms) {
  // the widths of configs 2-5; other shapes run on the fp32 CUDA-core kernels (mlp_simt.cu)
  return ms.Hd == H && ms.Hc == H && ms.Do == DO && ms.LF % 16 == 0 && ms.LF >= 16 && ms.LF <= 64 && ms.n_sh == 16 &&
         ms.geo_off == 1 && ms.geo_cnt == 15;
}

size_t mlp_tc_wimg_bytes(int backward) { return backward ? WImg::b_total : 2 * WImg::f_total; }

int launch_pack_weights(const MlpShape &ms, int bf16, const float *theta_mlp, const Workspace &ws, cudaStream_t st) {
  if (bf16) pack_weights_kernel<__nv_bfloat16><<<5, 256, 0, st>>>(ms, theta_mlp, ws.wimg_fwd, ws.wimg_bwd);
  else pack_weights_kernel<__half><<<5, 256, 0, st>>>(ms, theta_mlp, ws.wimg_fwd, ws.wimg_bwd);
  return 1;
}

int launch_adam_mlp_pack(const MlpShape &ms, int bf16, const FieldParams &fp, const Workspace &ws, const AdamConst &c,
                         uint32_t n_ctas, const uint32_t *d_S, cudaStream_t st) {
  const unsigned grid = (ms.n_mlp + 31) / 32;
  if (bf16) launch_pdl(adam_pack_kernel<__nv_bfloat16>, dim3(grid), dim3(128), 0, st, ms, fp.mlp_theta, fp.mlp_m, fp.mlp_v, fp.mlp_grad, ws.wimg_fwd, ws.wimg_bwd, c, ws.wgrad_part, n_ctas, d_S, ws.timeline);
  else launch_pdl(adam_pack_kernel<__half>, dim3(grid), dim3(128), 0, st, ms, fp.mlp_theta, fp.mlp_m, fp.mlp_v, fp.mlp_grad, ws.wimg_fwd, ws.wimg_bwd, c, ws.wgrad_part, n_ctas, d_S, ws.timeline);
  return 1;
}

int launch_reduce_wgrad(const MlpShape &ms, const Workspace &ws, float *grad_mlp, uint32_t n_ctas, const uint32_t *d_S, cudaStream_t st) {
  reduce_wgrad_kernel<<<(ms.n_mlp + 31) / 32, 128, 0, st>>>(ws.wgrad_part, ms.n_mlp, n_ctas, d_S, grad_mlp);
  return 1;
}

uint32_t mlp_tc_backward_ctas(int n_sms) { return 2u * (uint32_t)n_sms; }

// The kernels need more than 48 KB of dynamic shared memory: an opt-in that CUDA keeps per device.
cudaError_t mlp_tc_prepare_device() {
  const auto attr = cudaFuncAttributeMaxDynamicSharedMemorySize;
  cudaError_t e = cudaFuncSetAttribute(mlp_forward_tc_kernel<__half, true>, attr, (int)FwdSmem<true>::total);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(mlp_forward_tc_kernel<__half, false>, attr, (int)FwdSmem<false>::total);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(mlp_forward_tc_kernel<__nv_bfloat16, true>, attr, (int)FwdSmem<true>::total);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(mlp_forward_tc_kernel<__nv_bfloat16, false>, attr, (int)FwdSmem<false>::total);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(mlp_backward_tc_kernel<__half>, attr, (int)BwdSmem::total);
  if (e == cudaSuccess) e = cudaFuncSetAttribute(mlp_backward_tc_kernel<__nv_bfloat16>, attr, (int)BwdSmem::total);
  return e;
}

template <typename T, bool SPLIT>
static void launch_fwd_variant(const MlpShape &ms, const float *dirs, const Workspace &ws, const uint32_t *d_S, int density_only,
                               int save_blobs, int n_sms, cudaStream_t st) {
  launch_pdl(mlp_forward_tc_kernel<T, SPLIT>, dim3(n_sms), dim3(FWD_THREADS), (size_t)FwdSmem<SPLIT>::total, st, ms, dirs, ws, d_S,
             density_only, save_blobs);
}

int launch_mlp_forward_tc(const MlpShape &ms, int bf16, const float *dirs, const Workspace &ws, const uint32_t *d_S,
                          int density_only, int save_blobs, int n_sms, cudaStream_t st) {
  // the training forward (save_blobs) runs two-term operands; render and occupancy refresh run plain 16-bit operands
  if (bf16) {
    if (save_blobs) launch_fwd_variant<__nv_bfloat16, true>(ms, dirs, ws, d_S, density_only, save_blobs, n_sms, st);
    else launch_fwd_variant<__nv_bfloat16, false>(ms, dirs, ws, d_S, density_only, save_blobs, n_sms, st);
  } else {
    if (save_blobs) launch_fwd_variant<__half, true>(ms, dirs, ws, d_S, density_only, save_blobs, n_sms, st);
    else launch_fwd_variant<__half, false>(ms, dirs, ws, d_S, density_only, save_blobs, n_sms, st);
  }
  return 1;
}

int launch_mlp_backward_tc(const MlpShape &ms, int bf16, const Workspace &ws, const uint32_t *d_S,
                           int n_sms, cudaStream_t st) {
  const size_t smem = BwdSmem::total;
  if (bf16) {
    launch_pdl(mlp_backward_tc_kernel<__nv_bfloat16>, dim3(2 * n_sms), dim3(BWD_THREADS), smem, st, ms, ws, d_S);
  } else {
    launch_pdl(mlp_backward_tc_kernel<__half>, dim3(2 * n_sms), dim3(BWD_THREADS), smem, st, ms, ws, d_S);
  }
  return 1;
}

int launch_blob_to_rows(int bf16, const uint8_t *blob, uint32_t n_cols, int two_term, const uint32_t *d_S, float *rows,
                        cudaStream_t st) {
  if (bf16) blob_to_rows_kernel<__nv_bfloat16><<<1024, 256, 0, st>>>(blob, n_cols, two_term, d_S, rows);
  else blob_to_rows_kernel<__half><<<1024, 256, 0, st>>>(blob, n_cols, two_term, d_S, rows);
  return 1;
}
