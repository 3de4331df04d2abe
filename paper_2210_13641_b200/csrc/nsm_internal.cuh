// nsm_internal.cuh — device-side data layout and kernel launchers shared by the .cu files of
// the CUDA path.  Nothing here is shared with oracle/.  See DESIGN.md "Data layout in HBM".
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "nsm.h"

#define NSM_MAX_LEVELS 32
#define NSM_TILE 128          // samples per MLP tile
#define NSM_LD 132            // smem row stride (floats) of a [feature][sample] activation buffer

// Per-level constants (S0), passed by value to kernels.
struct LevelTable {
  uint32_t n_levels, n_features, t_mask;
  uint32_t res[NSM_MAX_LEVELS];
  uint32_t dense[NSM_MAX_LEVELS];      // 1: slot = vx + (N+1)(vy + (N+1) vz); 0: hashed
  uint64_t offset[NSM_MAX_LEVELS + 1]; // in entries, of the STORAGE arrays (theta, m|v, grad): every level starts on a 64-byte
                                       // boundary (see EntryMap); the canonical offsets of include/nsm.h are EntryMap::canon
};

// Canonical entry index (include/nsm.h: levels back to back) <-> storage entry index.  A level's slice of the storage
// arrays starts at a multiple of 64 bytes of theta (16 / F entries), so that the x-neighbour corners (x, x + 1) of an even
// cell x -- adjacent slots on a dense level and, the hash XORing x in unmultiplied, on a hashed level too -- form an
// ALIGNED pair whatever the sizes of the levels before: one 16-byte load / reduction at F = 2, one 32-byte sector at
// F = 4 (configs 2 and 4: the dense levels hold an odd number of entries, which left every hashed level's pairs
// straddling a boundary).  The padding entries are never referenced: theta 0, gradient "untouched" for ever.  Used by
// the boundary kernels only (pack / unpack / debug).
struct EntryMap {
  uint32_t n_levels;
  uint64_t canon[NSM_MAX_LEVELS + 1], storage[NSM_MAX_LEVELS + 1];
};

// Offsets (floats) of the MLP matrices inside the MLP block (canonical order) and their shapes.
struct MlpShape {
  uint32_t LF, Hd, Do, Ci, Hc, n_color_layers, n_sh, sh_degree, geo_off, geo_cnt;
  uint32_t o_d1, o_d2, o_c1, o_c2, o_c3, n_mlp;
};

// Candidate lattice + field cube, by value to the march kernels.
struct MarchParams {
  float aabb_min[3], inv_extent;
  float t_min, dt;
  uint32_t K, G, C, jitter, step;   // C: occupancy cascades (F4)
  uint64_t seed;
  uint32_t R;
};

// Per-step device workspace.  All per-sample arrays are planes of `cap` floats (cap = capacity,
// a multiple of NSM_TILE), feature-major, so a warp reading 32 consecutive samples is coalesced.
struct Workspace {
  uint64_t cap;          // samples
  uint32_t max_rays;
  // rays
  uint32_t *counts;      // [R]
  uint32_t *offsets;     // [R+1]; offsets[R] = S
  unsigned long long *scan_state;  // chained-scan status words of the fused marcher, one per block; zero between launches
  uint32_t *scan_ctr;    // [0] ticket counter, [1] finished-block counter; zero between launches
  uint32_t *work_ctr;    // [8] ring of chunk counters of the table kernels (ChunkQueue)
  float *C, *D_hat, *O;  // [R,3], [R], [R]
  // samples
  uint32_t *s_ray, *s_k; // [cap]
  float *s_t, *s_delta;  // [cap]
  float *s_x;            // [3][cap] planes
  float *e;              // [LF][cap]
  float *hd;             // [Hd][cap]
  float *g;              // [Do][cap]
  float *h1, *h2;        // [Hc][cap]
  float *sigma;          // [cap]
  float *rgb;            // [cap,3]
  float *T_excl;         // [cap] transmittance before the sample (T_i of Eq. 6)
  float *dsigma;         // [cap]
  float *drgb;           // [cap,3]
  float *de;             // [LF][cap]
  // row f2 (pose gradients; allocated when NSM_OPT_POSE_GRADIENTS is set, else NULL and nothing below is written)
  float *dY;             // [16][cap] dL/dY of every sample (the SH slots of the colour MLP's input gradient)
  float *dx;             // [3][cap]  dL/dx of every sample
  // loss accumulators: [0]=sum rgb, [1]=sum depth, [2]=S of the step (doubles); device
  double *loss_acc;
  unsigned long long *total_samples;  // running sum of S over training steps (device)
  // tensor-core path: 16-bit operand-tile images ("blobs", see mlp_tc.cu) instead of the fp32 planes e/hd/g/h1/h2
  uint8_t *blob_e, *blob_hd, *blob_ci, *blob_h1, *blob_h2;
  uint8_t *wimg_fwd, *wimg_bwd;       // 16-bit weight images, repacked whenever the MLP weights change
  unsigned long long *timeline;       // debug (NSM_TIMELINE=1): [2][K_COUNT] first-block start / last-block end, globaltimer ns
  float *wgrad_part;                  // [mlp_tc_backward_ctas][n_mlp] per-CTA weight-gradient slices of the tensor-core backward
  uint32_t *grad_absmax;              // bits of max |dL/d(pre-activation)| entering S11 this step (loss scale)
};

// Kernel classes, for launch counting and the optional per-kernel event timing.
enum KernelId {
  K_MARCH = 0, K_ENCODE, K_MLP_FWD, K_COMPOSITE, K_MLP_BWD, K_SCATTER,
  K_ADAM_TABLE, K_ADAM_MLP, K_OCC, K_DEBUG, K_SAMPLE, K_POSE, K_COUNT
};

// DESIGN.md S1.1 -- the counter-based hash behind the jitter stream (S1) and the batch sampler (F1):
// two-multiply xorshift finaliser absorbing seed, step, ray, k.  32-bit wrap-around arithmetic.
__device__ __forceinline__ uint32_t nsm_mix32(uint32_t x) {
  x ^= x >> 16;
  x *= 0x7feb352du;
  x ^= x >> 15;
  x *= 0x846ca68bu;
  x ^= x >> 16;
  return x;
}
__device__ __forceinline__ uint32_t nsm_hash_prefix(uint64_t seed, uint32_t step, uint32_t r) {
  uint32_t h = nsm_mix32((uint32_t)(seed & 0xffffffffu) ^ 0x9e3779b9u);
  h = nsm_mix32(h ^ (uint32_t)(seed >> 32));
  h = nsm_mix32(h ^ step);
  h = nsm_mix32(h ^ r);
  return h;
}

// F1: one keyframe of the device-side store (pinhole view; R rotates camera to world, row-major; t = camera centre;
// rgb [H,W,3], z-depth [H,W] and its variance [H,W] are library-owned device copies)
struct KeyframeDev {
  uint32_t W, H;
  float fx, fy, cx, cy;
  float R[9];
  float t[3];
  const float *rgb, *depth, *var;
};
#define NSM_MAX_KEYFRAMES 1024
#define NSM_KF_GRAD_STRIDE 8   /* per keyframe: dL/dt (3), dL/d(omega) (3), number of rays in the batch, pad */

// Debug timeline: when ws.timeline is set, thread 0 of every block stamps the kernel class's earliest start
// and latest end with %globaltimer.  Unlike CUDA events between launches this does not disturb PDL or the
// two-stream overlap, so it shows the step as it really runs.
__device__ __forceinline__ void tl_mark(unsigned long long *tl, int id, int end) {
  if (tl && threadIdx.x == 0) {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    if (end) atomicMax(tl + K_COUNT + id, t);
    else atomicMin(tl + id, t);
  }
}

// Parameters.  Three arrays over the table entries, each sized for what reads it:
//   theta[e*F + f]          the values the encoder gathers: compact (48.8 MB at config 2), so a 64-byte DRAM fetch
//                           brings 8 entries (F = 2) and the x-neighbour corner pairs of a cell share a 16-byte word;
//   mv[e*2F + 0..F) = m,    Adam moments, one 4F-byte record per entry (16 B for F = 2): only the table Adam touches
//   mv[e*2F + F..2F) = v    them, for the random ~25 % of entries a step references;
//   grad[e*F + f]           the gradient, compact like theta (L2-sized): the scatter's vector reductions land in a
//                           table that fits the cache, and Adam reads it as a dense coalesced stream.
// (Measured on B200, profiles/r1h: with theta inside 32-byte per-entry records the encoder moved 120 MB of DRAM
// for 12 MB of useful theta and ran at 81 % of the HBM peak; DRAM fetches are 64 bytes.)
//
// Touched set without flags: between steps every gradient word holds -0.0f (bits 0x80000000).
// The scatter never adds -0.0 or a magnitude below 2^-96 (those addends become +0.0), and under
// round-to-nearest a sum of such addends is +0.0, or a multiple of 2^-119 >= FLT_MIN in magnitude;
// it is never -0.0 (x + (-x) = +0.0) and never a subnormal that the reduction unit could flush to
// -0.0.  Hence "entry e was referenced this step"  <=>  bits(grad[e*F]) != 0x80000000, whatever the
// gradient's value (the touched set is structural, S12); Adam writes -0.0f back.
// (Round 2 measured the alternative -- a one-bit-per-entry touched bitmap set by atomicOr in the scatter or in the
// training forward's encoder, walked by Adam instead of the dense gradient scan: the marking costs as much as the scan
// saves, profiles/r2a_touched_bitmap.md.)
// The canonical flat layout of include/nsm.h exists only at the boundary (pack/unpack kernels).
#define NSM_GRAD_UNTOUCHED 0x80000000u
#define NSM_GRAD_MIN_ADDEND 1.262177448e-29f   /* 2^-96 */
struct FieldParams {
  float *theta;                                     // [n_entries][F]
  float *mv;                                        // [n_entries][2F]
  float *grad;                                      // [n_entries][F]
  float *mlp_theta, *mlp_m, *mlp_v, *mlp_grad;      // [n_mlp] each, canonical order
  uint8_t *occ_bits;                                // [G^3/8]
  float *occ_grid;                                  // [G^3] running density of the decayed refresh (F4); seeded by FROM_FIELD
  uint64_t n_entries;                               // STORAGE entries (padding included): array sizes, the table Adam's range
  uint64_t n_canon, n_table, n_mlp;                 // canonical entries, n_table = n_canon * F parameters (the boundary's count)
  uint32_t F;
  EntryMap map;
};

// ---- programmatic dependent launch (PDL) ---------------------------------------------------------
// Every hot-path kernel is launched with the programmatic-stream-serialization attribute and starts
// with pdl_wait(); pdl_trigger():  the wait returns once the preceding kernel in the stream has
// completed and its writes are visible; the trigger (issued by every block right after its wait)
// lets the NEXT kernel's blocks be scheduled and run their own prologue while this one computes.
// Because a block triggers only after its own wait, "kernel A has triggered" implies that
// everything before A is complete: code placed before pdl_wait() may read data produced two or
// more kernels back (the MLP weight images), never the immediate predecessor's output.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// Which kernel classes (bit = KernelId) are launched with the PDL attribute (swept on the GPU, profiles/r1g).
nsm_status nsm_set_error(nsm_status st, const char *msg);   // nsm_api.cu: sets nsm_last_error()'s message, returns st

extern const uint32_t g_pdl_mask;
extern thread_local int g_cur_kernel;

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = ((g_pdl_mask >> g_cur_kernel) & 1u) ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ---- L2 residency control (PTX createpolicy + .L2::cache_hint) -------------------------------------
// The compact gradient array is the one structure every step touches three times (scatter RMW, Adam
// read, Adam reset) and that fits the 126 MB L2; the table records and the per-sample workspace are
// streams several times its size.  Gradient accesses carry evict_last, record traffic of the hashed
// levels evict_first, so the streams do not push the gradient array out between its uses.
__device__ __forceinline__ uint64_t l2_evict_first() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ uint64_t l2_evict_normal() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_normal.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ uint64_t l2_evict_last() {
  uint64_t p;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
  return p;
}
__device__ __forceinline__ float4 ld_hint_f4(const float *p, uint64_t pol) {
  float4 v;
  asm volatile("ld.global.L2::cache_hint.v4.f32 {%0, %1, %2, %3}, [%4], %5;"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p), "l"(pol) : "memory");
  return v;
}
__device__ __forceinline__ float2 ld_hint_f2(const float *p, uint64_t pol) {
  float2 v;
  asm volatile("ld.global.L2::cache_hint.v2.f32 {%0, %1}, [%2], %3;" : "=f"(v.x), "=f"(v.y) : "l"(p), "l"(pol) : "memory");
  return v;
}
__device__ __forceinline__ float ld_hint_f1(const float *p, uint64_t pol) {
  float v;
  asm volatile("ld.global.L2::cache_hint.f32 %0, [%1], %2;" : "=f"(v) : "l"(p), "l"(pol) : "memory");
  return v;
}
__device__ __forceinline__ void st_hint_f4(float *p, float4 v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_hint_f2(float *p, float2 v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(p), "f"(v.x), "f"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_hint_f1(float *p, float v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(p), "f"(v), "l"(pol) : "memory");
}
// vectorised no-return reductions (red.global.add.v2/v4.f32, sm_90+) with an L2 policy
__device__ __forceinline__ void red_hint_f4(float *p, float4 v, uint64_t pol) {
  asm volatile("red.global.add.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(pol) : "memory");
}
__device__ __forceinline__ void red_hint_f2(float *p, float2 v, uint64_t pol) {
  asm volatile("red.global.add.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(p), "f"(v.x), "f"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ void red_hint_f1(float *p, float v, uint64_t pol) {
  asm volatile("red.global.add.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(p), "f"(v), "l"(pol) : "memory");
}

// S13: one Adam update with bias correction (inv_bc = 1 / (1 - beta^t), computed on the host in float64)
struct AdamConst {
  float lr, b1, b2, eps, inv_bc1, inv_bc2;
};

__device__ __forceinline__ void adam_one(float &th, float &m, float &v, float g, const AdamConst &c) {
  m = c.b1 * m + (1.f - c.b1) * g;
  v = c.b2 * v + (1.f - c.b2) * g * g;
  float mhat = m * c.inv_bc1, vhat = v * c.inv_bc2;
  th = th - c.lr * mhat / (sqrtf(vhat) + c.eps);
}

// Work distribution of the table kernels (encoder, scatter): the (level, sample) items are level-major, and a block takes
// them 256 at a time from a counter, in increasing order -- so at any moment the whole chip works inside a window of
// ~0.25 M consecutive items, i.e. on ONE level's slice of the tables (67 MB at config 4, where the tables are 719 MB):
// that slice is what the TLBs and the L2 have to cover, not the whole table.  A static grid-stride loop lets the blocks
// drift across ten levels (measured at config 4: scatter 343 -> 239 us, encoder 208 -> 172 us with in-order chunks).
// The counters form a ring indexed by the launch sequence number: launch n counts in slot n % 8 and zeroes slot
// (n + 4) % 8, which no kernel in flight can be using (launches on one stream are ordered).
#ifndef NSM_SCATTER_PF_CHUNKS
#define NSM_SCATTER_PF_CHUNKS 96
#endif
struct ChunkQueue {
  uint32_t *ctr;
  __device__ __forceinline__ ChunkQueue(uint32_t *ring, uint32_t seq) : ctr(ring + (seq & 7u)) {
    if (blockIdx.x == 0 && threadIdx.x == 0) ring[(seq + 4u) & 7u] = 0u;
  }
  // first item of the block's next chunk of blockDim.x items; every thread of the block must call it
  __device__ __forceinline__ uint64_t next(uint32_t *slot) {
    __syncthreads();   // the previous value has been read by everyone
    if (threadIdx.x == 0) *slot = atomicAdd(ctr, 1u);
    __syncthreads();
    return (uint64_t)*slot * blockDim.x;
  }
};

// ---- launchers (each enqueues on `st`, returns the number of kernels launched) ----
// S1-S3 in one launch; also resets the loss accumulators and (count_total) adds S to the running sample count
// dirs_copy (optional): [R,3] device buffer that receives the directions (host entry points: origins / dirs may be
// device-mapped pinned HOST memory, read once here; the later kernels use the copy)
int launch_march(const MarchParams &mp, const uint8_t *bits, const float *origins, const float *dirs,
                 const Workspace &ws, int count_total, cudaStream_t st, float *dirs_copy = nullptr);
uint32_t march_scan_state_entries(uint32_t max_rays);
// out_mode: 0 = fp32 planes ws.e, 1 = fp16 blob ws.blob_e, 2 = bf16 blob ws.blob_e
// seq: launch sequence number of the field's table kernels (selects the ChunkQueue counter)
// max_samples: an upper bound on S known to the host (rays x candidates, cells of a refresh chunk): picks the work mapping
// two_term: blob modes only -- write the hi AND the lo tile (training: the two-term forward) or the hi tile alone
// (forward-only uses, whose MLP kernel reads nothing else)
int launch_encode(const LevelTable &lv, const float *theta, const Workspace &ws,
                  const uint32_t *d_S, int out_mode, int n_sms, cudaStream_t st, uint32_t seq, uint64_t max_samples, bool two_term);
// S12 over all levels: vector reductions into grad
int launch_scatter(const LevelTable &lv, float *grad, const Workspace &ws, const uint32_t *d_S, int n_sms, cudaStream_t st,
                   uint32_t seq);
// gradient array <- canonical gradient + touched flags (NULL: every entry touched); src == nullptr: all untouched
int launch_set_grad(const FieldParams &fp, const float *src, const uint8_t *touched, cudaStream_t st);
int launch_get_touched(const FieldParams &fp, uint8_t *dst, cudaStream_t st);
// canonical [n_canon][F] <-> `which` (0 theta, 1 gradient (unpack only), 2 m, 3 v) of the internal arrays; src == nullptr packs zeros
int launch_pack_records(const FieldParams &fp, int which, const float *src, cudaStream_t st);
int launch_unpack_records(const FieldParams &fp, int which, float *dst, cudaStream_t st);
int launch_mlp_forward_simt(const MlpShape &ms, const float *theta_mlp, const float *dirs,
                            const Workspace &ws, const uint32_t *d_S, int density_only, int n_sms,
                            cudaStream_t st);
int launch_mlp_backward_simt(const MlpShape &ms, const float *theta_mlp, float *grad_mlp,
                             const float *dirs, const Workspace &ws, const uint32_t *d_S, int n_sms,
                             cudaStream_t st);
size_t mlp_simt_smem_bytes(const MlpShape &ms, int backward);

bool mlp_tc_supported(const MlpShape &ms);
size_t mlp_tc_wimg_bytes(int backward);
// opt-in shared-memory size of the tcgen05 kernels on the CURRENT device (a per-device attribute): once per field
cudaError_t mlp_tc_prepare_device();
int launch_pack_weights(const MlpShape &ms, int bf16, const float *theta_mlp, const Workspace &ws, cudaStream_t st);
int launch_mlp_forward_tc(const MlpShape &ms, int bf16, const float *dirs, const Workspace &ws, const uint32_t *d_S,
                          int density_only, int save_blobs, int n_sms, cudaStream_t st);
// weight gradients: one slice of ws.wgrad_part per CTA (mlp_tc_backward_ctas of them), summed by the consumer
int launch_mlp_backward_tc(const MlpShape &ms, int bf16, const Workspace &ws, const uint32_t *d_S,
                           int n_sms, cudaStream_t st);
uint32_t mlp_tc_backward_ctas(int n_sms);
int launch_reduce_wgrad(const MlpShape &ms, const Workspace &ws, float *grad_mlp, uint32_t n_ctas, const uint32_t *d_S, cudaStream_t st);
int launch_blob_to_rows(int bf16, const uint8_t *blob, uint32_t n_cols, int two_term, const uint32_t *d_S, float *rows,
                        cudaStream_t st);
int launch_composite_train(const Workspace &ws, uint32_t R, const float *rgb, const float *depth,
                           const float *depth_var, float lambda_d, const float bg[3],
                           cudaStream_t st);
int launch_composite_render(const Workspace &ws, uint32_t R, float cut, const float bg[3],
                            float *out_rgb, float *out_depth, float *out_opacity, cudaStream_t st);
// S13 on the touched table entries (sparse) or on all of them; consumes the gradients (every word back to "untouched")
int launch_adam_table(const FieldParams &fp, uint32_t F, int sparse, float lr, float beta1, float beta2,
                      float eps, float inv_bc1, float inv_bc2, cudaStream_t st, unsigned long long *tl, uint64_t max_samples);
int launch_adam_mlp(const FieldParams &fp, float lr, float beta1, float beta2, float eps, float inv_bc1,
                    float inv_bc2, cudaStream_t st);
// tensor-core path: Adam on the MLP weights and, in the same launch, the refreshed 16-bit weight images
// n_ctas > 0: the gradient is the sum of the backward kernel's slices (+ fp.mlp_grad); 0: fp.mlp_grad alone
int launch_adam_mlp_pack(const MlpShape &ms, int bf16, const FieldParams &fp, const Workspace &ws, const AdamConst &c,
                         uint32_t n_ctas, const uint32_t *d_S, cudaStream_t st);
// F1: n_rays rays drawn uniformly over (keyframe, pixel) for draw number `draw`; outputs are a ray batch
// ray_kf (optional): [n_rays] keyframe index of every ray
int launch_sample_batch(const KeyframeDev *kfs, uint32_t n_kf, uint64_t seed, uint32_t draw, uint32_t n_rays, float *origins,
                        float *dirs, float *rgb, float *depth, float *depth_var, uint32_t *ray_kf, cudaStream_t st);
// f2: per-ray dL/do and rotation gradient from ws.de / ws.dY (after the MLP backward, before Adam); ray_kf + kf_grad
// (optional): the per-keyframe vectors [n_kf][NSM_KF_GRAD_STRIDE], written (not accumulated) by a block per keyframe
int launch_pose_gradients(const LevelTable &lv, const float *theta, const Workspace &ws, const uint32_t *d_S, uint32_t R,
                          const float *dirs, float inv_extent, uint32_t sh_degree, float *g_o, float *tau, const uint32_t *ray_kf,
                          float *kf_grad, uint32_t n_kf, int n_sms, cudaStream_t st, uint32_t pose_levels = 0);
// f2, the update: Adam + exponential map on the keyframes that received rays (kf_grad: [n_kf][NSM_KF_GRAD_STRIDE])
int launch_pose_step(KeyframeDev *kfs, uint32_t n_kf, const float *kf_grad, float *pm, float *pv, uint32_t *pcnt, float lr_t,
                     float lr_r, float beta1, float beta2, float eps, cudaStream_t st);
// the centres of cells first_cell + i * stride, i < n_cells (global cell index over the C cascades), as samples
int launch_occ_cells(uint32_t G, uint32_t C, uint64_t first_cell, uint32_t stride, uint64_t n_cells, const Workspace &ws,
                     uint32_t *d_S, cudaStream_t st);
// F4 stochastic refresh: draws first_draw .. first_draw + n_draws of update `upd` as samples; their cells in ws.s_k
int launch_occ_cells_stochastic(uint32_t G, uint32_t C, uint64_t seed, uint32_t upd, uint32_t first_draw, uint32_t n_draws,
                                const Workspace &ws, uint32_t *d_S, cudaStream_t st);
int launch_occ_max_cells(float *grid, const uint32_t *cells, uint32_t n, const float *sigma, cudaStream_t st);
int launch_occ_threshold(uint32_t G, uint64_t first_cell, uint64_t n_cells, const float *sigma,
                         float thr, uint8_t *bits, float *grid, cudaStream_t st);
// F4: decayed running-maximum density grid with a strided partial refresh
int launch_occ_decay(float *grid, uint64_t n_cells, float decay, cudaStream_t st);
int launch_occ_max_visited(float *grid, uint64_t first_cell, uint32_t stride, uint64_t n_visited, const float *sigma, cudaStream_t st);
int launch_occ_bits_from_grid(const float *grid, uint64_t n_cells, float thr, uint8_t *bits, cudaStream_t st);
int launch_debug_slots(const LevelTable &lv, const Workspace &ws, const uint32_t *d_S,
                       uint32_t *slots, float *w, cudaStream_t st);
int launch_planes_to_rows(const float *planes, uint64_t cap, uint32_t n_planes, const uint32_t *d_S,
                          float *rows, cudaStream_t st);
