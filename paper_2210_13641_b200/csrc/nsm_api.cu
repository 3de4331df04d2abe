// nsm_api.cu — the C-ABI boundary (include/nsm.h): argument validation, the field object
// (parameters, Adam state, occupancy bits, workspace arena) and the host-side step scheduler
// that enqueues the kernels of S1..S15 on the field's stream.  No arithmetic of the method is
// done on the host except S0's integer level table and Adam's scalar bias corrections.
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "nsm_internal.cuh"

namespace {

thread_local std::string g_err;

nsm_status fail(nsm_status st, const char *fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return st;
}

#define CUDA_TRY(expr)                                                                         \
  do {                                                                                         \
    cudaError_t e_ = (expr);                                                                   \
    if (e_ != cudaSuccess)                                                                     \
      return fail(e_ == cudaErrorMemoryAllocation ? NSM_ERR_OOM : NSM_ERR_CUDA, "%s: %s", #expr, \
                  cudaGetErrorString(e_));                                                     \
  } while (0)

}  // namespace

// the thread-local message behind nsm_last_error(), for entry points defined in other files (march.cu)
nsm_status nsm_set_error(nsm_status st, const char *msg) {
  g_err = msg;
  return st;
}

// Default: every hot-path kernel except the marcher (bit 0) and the scatter (bit 5).  Measured on B200 at
// config 2 (profiles/r1g_pdl_sweep.md): 148.7 us/step without PDL, 135.5 us with this mask; letting the
// table Adam's blocks become resident under the scatter, or the marcher's under the MLP Adam, costs
// more than the launch gap it hides (149 us / 184 us).
const uint32_t g_pdl_mask = 0xdeu;
thread_local int g_cur_kernel = 0;   // kernel class of the launch in progress on this host thread (RUN macro)

static const char *kKernelNames[K_COUNT] = {"march", "encode", "mlp_fwd", "composite",
                                            "mlp_bwd", "scatter", "adam_table", "adam_mlp", "occupancy", "debug", "sample", "pose"};

// Optional per-kernel CUDA-event timing (bench.py's roofline leg).  When enabled every launch is
// bracketed by two events on the field's stream and each step ends with a synchronise.
struct Profiler {
  bool on = false;
  bool failed = false;   // an event of the timing pass could not be recorded or read: its numbers are not to be trusted
  double ms[K_COUNT] = {0};
  uint64_t n[K_COUNT] = {0};
  struct Rec { int id; cudaEvent_t a, b; };
  std::vector<Rec> pending;
  std::vector<cudaEvent_t> pool;
  cudaEvent_t get() {
    if (!pool.empty()) { cudaEvent_t e = pool.back(); pool.pop_back(); return e; }
    cudaEvent_t e; cudaEventCreate(&e); return e;
  }
  void collect() {
    for (auto &r : pending) {
      float t = 0.f;
      if (cudaEventSynchronize(r.b) != cudaSuccess || cudaEventElapsedTime(&t, r.a, r.b) != cudaSuccess) failed = true;
      ms[r.id] += t; n[r.id] += 1;
      pool.push_back(r.a); pool.push_back(r.b);
    }
    pending.clear();
  }
  void destroy() { collect(); for (auto e : pool) cudaEventDestroy(e); pool.clear(); }
};

struct nsm_field {
  nsm_field_config cfg;
  Profiler prof;
  uint64_t launches_by[K_COUNT] = {0};
  cudaStream_t stream = nullptr;
  int device = 0;             // the CUDA device the field lives on (current at creation); every entry point runs there
  int n_sms = 148;
  LevelTable lv;
  MlpShape ms;
  FieldParams fp;
  Workspace ws;
  std::vector<void *> allocs;
  uint32_t step = 0;
  uint64_t launches = 0;
  uint32_t work_seq = 0;      // launch sequence number of the table kernels (ChunkQueue counter ring)
  bool occ_full = true;
  uint32_t occ_updates = 0;   // F4: decayed partial refreshes since the last full one
  uint32_t occ_draws = 0;     // F4: stochastic refreshes since creation (keys their draws; never reset)
  bool grid_seeded = false;   // F4: the running density grid holds a full FROM_FIELD pass (SET / FULL invalidate it)
  bool grads_dirty = false;
  // state of the last step, for the debug getter
  uint32_t last_R = 0, last_K = 0;
  bool last_was_render = false;
  // staging for the *_host entry points
  float *stage_dev = nullptr;     // [max_rays * 12]: a training batch (11 floats per ray) or two render buffers (origins | dirs)
  float *stage_out = nullptr;     // render outputs, two buffers of [max_rays * 5]
  struct HostStats { double acc[3]; uint32_t S; } *pinned = nullptr;   // acc[2] = S of the step, as a double
  // Side stream: work that does not depend on the table Adam runs beside it (it is DRAM-bound, the others
  // are latency-bound): the MLP Adam of the same step and, when the caller has declared its batches ready
  // (NSM_OPT_BATCH_READY), the marcher of the NEXT step.  ev_pre_adam marks "scatter of the last step done".
  cudaStream_t side = nullptr;
  cudaEvent_t ev_pre_adam = nullptr, ev_side = nullptr, ev_main = nullptr;
  // the step's statistics (loss sums, S) are final after the compositor: they are copied out on the side stream right
  // behind it, and a call that wants them waits for that copy only, not for the backward pass and Adam
  cudaEvent_t ev_comp = nullptr, ev_stats = nullptr;
  // nsm_render_host: two staging buffers each way; [j] "rays of buffer j are on the device", "the kernels of buffer j's
  // chunk are done" (its rays consumed, its image complete), "buffer j's image has been copied out"
  cudaEvent_t ev_in[2] = {nullptr, nullptr}, ev_done[2] = {nullptr, nullptr}, ev_outfree[2] = {nullptr, nullptr};
  // F1: the keyframe store (library-owned device copies) and its device-side directory
  std::vector<KeyframeDev> kf_host;
  KeyframeDev *kf_dev = nullptr;
  // row f2: pose gradients (NSM_OPT_POSE_GRADIENTS)
  bool pose_grads = false, last_sampled = false;
  uint32_t pose_levels = 0;   // row f2, reading R26: encoding levels that carry the pose gradient (0 = all)
  float *pose_go = nullptr, *pose_tau = nullptr, *kf_grad = nullptr;   // [max_rays,3] x2, [NSM_MAX_KEYFRAMES,NSM_KF_GRAD_STRIDE]
  float *kf_pose_m = nullptr, *kf_pose_v = nullptr;                    // Adam moments of the keyframe poses [NSM_MAX_KEYFRAMES,6]
  uint32_t *kf_pose_cnt = nullptr;                                     // updates received per keyframe
  uint32_t *ray_kf = nullptr;                                           // [max_rays] keyframe of every sampled ray
  bool stats_pending = false;
  bool join_pending = false;   // ev_side (recorded behind the MLP Adam) has not been waited for on the main stream yet
  unsigned long long *timeline_base = nullptr;   // NSM_OPT_DEBUG_TIMELINE: ring of 64 steps x [2][K_COUNT] globaltimer stamps
  bool timeline_on = false;
  bool scatter_pending = false;   // the backward pass stopped before S12: enqueue_adam issues the scatter right before the table Adam
  uint32_t wgrad_parts = 0;   // > 0: the MLP weight gradient of the last backward is still in that many per-CTA slices
  bool batch_ready = false;   // NSM_OPT_BATCH_READY
  bool e_two_term = true;     // the last encoder launch wrote hi + lo operand tiles (training) or hi alone (forward-only uses)
  bool side_ok = false;       // nothing but a train step's Adam has been enqueued on `stream` since ev_pre_adam
  const char *mlp_path = "simt_fp32";
  bool use_tc = false;   // tcgen05 MLP kernels (16-bit configurations with supported shapes)

  template <typename T>
  cudaError_t alloc(T **p, size_t n, bool zero = true) {
    void *q = nullptr;
    size_t bytes = (n * sizeof(T) + 255) & ~size_t(255);
    cudaError_t e = cudaMalloc(&q, bytes ? bytes : 256);
    if (e != cudaSuccess) return e;
    allocs.push_back(q);
    *p = (T *)q;
    if (zero) return cudaMemsetAsync(q, 0, bytes ? bytes : 256, stream);
    return cudaSuccess;
  }
};

namespace {

// S0 — integer level table: N_l = floor(N_min * exp(l ln(N_max/N_min)/(L-1)) + 1e-6) in float64,
// ends forced; E_l = min((N_l+1)^3, T); dense iff (N_l+1)^3 <= T.
// lv.offset: storage offsets, each level on a 64-byte boundary; map: canonical <-> storage (EntryMap, nsm_internal.cuh)
nsm_status build_levels(const nsm_field_config &c, LevelTable &lv, EntryMap &map) {
  const uint32_t L = c.n_levels;
  const uint64_t T = 1ull << c.log2_table_size;
  // entries per 64 bytes: the x-neighbour pair (slot, slot ^ 1) of an even cell x then shares one 16-byte (F = 2) or one
  // 32-byte sector (F = 4) in theta, in the gradient array and in the moment records' neighbourhood
  const uint64_t align = c.n_features >= 16 ? 1 : 16 / c.n_features;
  lv.n_levels = L;
  lv.n_features = c.n_features;
  lv.t_mask = (uint32_t)(T - 1);
  lv.offset[0] = 0;
  map.n_levels = L;
  map.canon[0] = map.storage[0] = 0;
  for (uint32_t l = 0; l < L; ++l) {
    uint32_t N;
    if (l == 0) N = c.n_min;
    else if (l == L - 1) N = c.n_max;
    else {
      double step = std::log((double)c.n_max / (double)c.n_min) / (double)(L - 1);
      N = (uint32_t)std::floor((double)c.n_min * std::exp(step * (double)l) + 1e-6);
    }
    lv.res[l] = N;
    const uint64_t side = (uint64_t)N + 1, cube = side * side * side;
    lv.dense[l] = cube <= T;
    const uint64_t n_l = cube <= T ? cube : T;
    map.canon[l + 1] = map.canon[l] + n_l;
    lv.offset[l + 1] = (lv.offset[l] + n_l + align - 1) / align * align;
    map.storage[l + 1] = lv.offset[l + 1];
  }
  return NSM_OK;
}

nsm_status validate_config(const nsm_field_config *c) {
  if (!c) return fail(NSM_ERR_INVALID_ARG, "config is NULL");
  if (c->struct_size != sizeof(nsm_field_config))
    return fail(NSM_ERR_INVALID_ARG, "struct_size %u != %zu (ABI mismatch)", c->struct_size, sizeof(nsm_field_config));
  if (!(c->aabb_extent > 0.f) || !std::isfinite(c->aabb_extent)) return fail(NSM_ERR_INVALID_ARG, "aabb_extent must be > 0");
  if (c->n_levels < 1 || c->n_levels > NSM_MAX_LEVELS) return fail(NSM_ERR_INVALID_ARG, "n_levels out of [1,32]");
  if (c->n_features != 1 && c->n_features != 2 && c->n_features != 4 && c->n_features != 8)
    return fail(NSM_ERR_INVALID_ARG, "n_features must be 1, 2, 4 or 8");
  if (c->log2_table_size < 4 || c->log2_table_size > 28) return fail(NSM_ERR_INVALID_ARG, "log2_table_size out of [4,28]");
  if (c->n_min < 1 || c->n_max < c->n_min || c->n_max > (1u << 20)) return fail(NSM_ERR_INVALID_ARG, "bad n_min/n_max");
  if (c->occ_res < 1 || (c->occ_res & (c->occ_res - 1)) || c->occ_res > 1024)
    return fail(NSM_ERR_INVALID_ARG, "occ_res must be a power of two <= 1024");
  if (c->occ_cascades > 8) return fail(NSM_ERR_INVALID_ARG, "occ_cascades must be <= 8");
  if ((uint64_t)(c->occ_cascades ? c->occ_cascades : 1) * c->occ_res * c->occ_res * c->occ_res > (1ull << 31))
    return fail(NSM_ERR_INVALID_ARG, "occ_cascades * occ_res^3 exceeds 2^31 cells");
  if (c->density_hidden < 1 || c->density_hidden > 128 || c->density_out < 1 || c->density_out > 16)
    return fail(NSM_ERR_INVALID_ARG, "density MLP widths out of range");
  if (c->geo_offset + c->geo_count > c->density_out) return fail(NSM_ERR_INVALID_ARG, "geo slice exceeds density_out");
  if (c->sh_degree < 1 || c->sh_degree > 4) return fail(NSM_ERR_UNIMPLEMENTED, "sh_degree must be in [1,4]");
  if (c->color_hidden < 1 || c->color_hidden > 128) return fail(NSM_ERR_INVALID_ARG, "color_hidden out of range");
  if (c->color_hidden_layers < 1 || c->color_hidden_layers > 2) return fail(NSM_ERR_INVALID_ARG, "color_hidden_layers must be 1 or 2");
  if (c->n_levels * c->n_features > 128) return fail(NSM_ERR_UNIMPLEMENTED, "L*F > 128 not supported");
  if (c->mlp_precision > NSM_MLP_BF16) return fail(NSM_ERR_INVALID_ARG, "bad mlp_precision");
  if (!(c->lr > 0.f) || !(c->beta1 >= 0.f && c->beta1 < 1.f) || !(c->beta2 >= 0.f && c->beta2 < 1.f) || !(c->eps >= 0.f))
    return fail(NSM_ERR_INVALID_ARG, "bad Adam hyper-parameters");
  if (c->max_rays < 1 || c->max_candidates < 1 || c->max_candidates > 4096)
    return fail(NSM_ERR_INVALID_ARG, "bad workspace capacity");
  if ((uint64_t)c->max_rays * c->max_candidates > (1ull << 31))
    return fail(NSM_ERR_INVALID_ARG, "max_rays * max_candidates exceeds 2^31");
  return NSM_OK;
}

nsm_status validate_batch(const nsm_field *f, const nsm_ray_batch *b, bool train, bool chunked) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  if (!b) return fail(NSM_ERR_INVALID_ARG, "batch is NULL");
  if (!b->origins || !b->dirs) return fail(NSM_ERR_INVALID_ARG, "origins/dirs are NULL");
  if (train && (!b->rgb || !b->depth || !b->depth_var)) return fail(NSM_ERR_INVALID_ARG, "rgb/depth/depth_var are NULL");
  if (b->n_rays == 0) return fail(NSM_ERR_INVALID_ARG, "n_rays is 0");
  if (b->n_candidates == 0) return fail(NSM_ERR_INVALID_ARG, "n_candidates is 0");
  if (!(b->t_max > b->t_min) || !std::isfinite(b->t_min) || !std::isfinite(b->t_max))
    return fail(NSM_ERR_INVALID_ARG, "need finite t_min < t_max");
  if (!chunked && b->n_rays > f->cfg.max_rays) return fail(NSM_ERR_CAPACITY, "n_rays %u > max_rays %u", b->n_rays, f->cfg.max_rays);
  if (b->n_candidates > f->cfg.max_candidates)
    return fail(NSM_ERR_CAPACITY, "n_candidates %u > max_candidates %u", b->n_candidates, f->cfg.max_candidates);
  return NSM_OK;
}

// launch one kernel class, counted and (optionally) timed
#define RUN(f, id, call) RUN_ON(f, id, (f)->stream, call)
#define RUN_ON(f, id, st_, call)                                            \
  do {                                                                      \
    g_cur_kernel = (id);                                                    \
    if ((f)->prof.on) {                                                     \
      Profiler::Rec r_{id, (f)->prof.get(), (f)->prof.get()};               \
      const cudaError_t ea_ = cudaEventRecord(r_.a, (st_));                 \
      int n_ = (call);                                                      \
      const cudaError_t eb_ = cudaEventRecord(r_.b, (st_));                 \
      if (ea_ != cudaSuccess || eb_ != cudaSuccess)                         \
        (f)->prof.failed = true;   /* reported by nsm_profile_read */       \
      (f)->prof.pending.push_back(r_);                                      \
      (f)->launches += n_; (f)->launches_by[id] += n_;                      \
    } else {                                                                \
      int n_ = (call);                                                      \
      (f)->launches += n_; (f)->launches_by[id] += n_;                      \
    }                                                                       \
  } while (0)

// The side stream's last work (the MLP Adam of the previous step) is joined into the main stream lazily: a training
// step that marches on the side stream joins behind its marcher anyway, every other entry point joins here.
cudaError_t join_side(nsm_field *f) {
  cudaError_t e = cudaSuccess;
  if (f->join_pending) {
    e = cudaStreamWaitEvent(f->stream, f->ev_side, 0);
    f->join_pending = false;
  }
  return e;
}
// Every entry point other than a training step calls this first: it makes the field's device current, joins the side
// stream and leaves the two-stream fast path.  A failure here is reported by the entry point's own CUDA_TRY of
// cudaGetLastError / its first CUDA call (the error is sticky).
cudaError_t leave_fast_path(nsm_field *f) {
  cudaError_t e = cudaSetDevice(f->device);
  const cudaError_t e2 = join_side(f);
  f->side_ok = false;
  return e != cudaSuccess ? e : e2;
}
#define LEAVE_FAST_PATH(f) CUDA_TRY(leave_fast_path(f))

// cells of the occupancy structure: occ_cascades nested grids of occ_res^3 (F4, reading R23)
uint32_t occ_cascades(const nsm_field *f) { return f->cfg.occ_cascades ? f->cfg.occ_cascades : 1u; }
uint64_t occ_cells(const nsm_field *f) { return (uint64_t)occ_cascades(f) * f->cfg.occ_res * f->cfg.occ_res * f->cfg.occ_res; }

MarchParams make_march(const nsm_field *f, const nsm_ray_batch *b, uint32_t R, bool jitter, uint32_t step) {
  MarchParams mp;
  for (int a = 0; a < 3; ++a) mp.aabb_min[a] = f->cfg.aabb_min[a];
  mp.inv_extent = 1.0f / f->cfg.aabb_extent;                     // S0 host constant, one fp32 divide
  mp.t_min = b->t_min;
  mp.dt = (b->t_max - b->t_min) / (float)b->n_candidates;        // one fp32 subtract, one fp32 divide
  mp.K = b->n_candidates;
  mp.G = f->cfg.occ_res;
  mp.C = f->cfg.occ_cascades ? f->cfg.occ_cascades : 1u;
  mp.jitter = jitter ? 1u : 0u;
  mp.step = step;
  mp.seed = f->cfg.seed;
  mp.R = R;
  return mp;
}

// S1-S8 forward (+ S9-S12 when train): everything up to, but excluding, Adam.
// march_on_side: the marcher runs on the side stream, behind "scatter of the previous step done" only,
// i.e. beside the previous step's table Adam (NSM_OPT_BATCH_READY; training steps only).
// dirs_copy: see launch_march (zero-copy host batches); the MLP kernels then read the copy.
// sample_draw >= 0: the batch is first drawn from the keyframe store (F1) into b's buffers (the field's staging area),
// on the stream the marcher runs on.
nsm_status enqueue_forward(nsm_field *f, const nsm_ray_batch *b, uint32_t R, bool jitter, uint32_t step, bool train,
                           bool march_on_side = false, float *dirs_copy = nullptr, int64_t sample_draw = -1) {
  const uint32_t *d_S = f->ws.offsets + R;
  const float *mlp_dirs = dirs_copy ? dirs_copy : b->dirs;
  MarchParams mp = make_march(f, b, R, jitter, step);
  if (march_on_side && !f->prof.on) {
    if (!f->side_ok) {   // other work has been enqueued on the main stream since the last Adam: order behind all of it
      CUDA_TRY(cudaEventRecord(f->ev_main, f->stream));
      CUDA_TRY(cudaStreamWaitEvent(f->side, f->ev_main, 0));
    }
    if (sample_draw >= 0)
      RUN_ON(f, K_SAMPLE, f->side, launch_sample_batch(f->kf_dev, (uint32_t)f->kf_host.size(), f->cfg.seed, (uint32_t)sample_draw, R,
                                                       (float *)b->origins, (float *)b->dirs, (float *)b->rgb, (float *)b->depth,
                                                       (float *)b->depth_var, f->pose_grads ? f->ray_kf : nullptr, f->side));
    RUN_ON(f, K_MARCH, f->side, launch_march(mp, f->occ_full ? nullptr : f->fp.occ_bits, b->origins, b->dirs, f->ws, train ? 1 : 0, f->side, dirs_copy));
    CUDA_TRY(cudaEventRecord(f->ev_side, f->side));
    CUDA_TRY(cudaStreamWaitEvent(f->stream, f->ev_side, 0));
    f->join_pending = false;   // behind the marcher is behind the previous step's MLP Adam too
  } else {
    CUDA_TRY(join_side(f));
    if (sample_draw >= 0)
      RUN(f, K_SAMPLE, launch_sample_batch(f->kf_dev, (uint32_t)f->kf_host.size(), f->cfg.seed, (uint32_t)sample_draw, R,
                                           (float *)b->origins, (float *)b->dirs, (float *)b->rgb, (float *)b->depth,
                                           (float *)b->depth_var, f->pose_grads ? f->ray_kf : nullptr, f->stream));
    RUN(f, K_MARCH, launch_march(mp, f->occ_full ? nullptr : f->fp.occ_bits, b->origins, b->dirs, f->ws, train ? 1 : 0, f->stream, dirs_copy));
  }
  const int bf16 = f->cfg.mlp_precision == NSM_MLP_BF16;
  RUN(f, K_ENCODE, launch_encode(f->lv, f->fp.theta, f->ws, d_S, f->use_tc ? 1 + bf16 : 0, f->n_sms, f->stream, f->work_seq++,
                                 (uint64_t)R * b->n_candidates, train));
  f->e_two_term = train;
  if (f->use_tc)
    RUN(f, K_MLP_FWD, launch_mlp_forward_tc(f->ms, bf16, mlp_dirs, f->ws, d_S, 0, train ? 1 : 0, f->n_sms, f->stream));
  else
    RUN(f, K_MLP_FWD, launch_mlp_forward_simt(f->ms, f->fp.mlp_theta, mlp_dirs, f->ws, d_S, 0, f->n_sms, f->stream));
  return NSM_OK;
}

// the tensor-core kernels read 16-bit weight images: repack after every change of the MLP weights
void repack_weights(nsm_field *f) {
  if (f->use_tc)
    RUN(f, K_ADAM_MLP, launch_pack_weights(f->ms, f->cfg.mlp_precision == NSM_MLP_BF16, f->fp.mlp_theta, f->ws, f->stream));
}

nsm_status clear_grads_if_dirty(nsm_field *f) {
  if (f->grads_dirty) {
    RUN(f, K_DEBUG, launch_set_grad(f->fp, nullptr, nullptr, f->stream));
    CUDA_TRY(cudaMemsetAsync(f->fp.mlp_grad, 0, sizeof(float) * f->fp.n_mlp, f->stream));
    f->wgrad_parts = 0;
    f->grads_dirty = false;
  }
  return NSM_OK;
}

nsm_status enqueue_backward(nsm_field *f, const nsm_ray_batch *b, float lambda_d, bool march_on_side = false,
                            float *dirs_copy = nullptr, bool want_stats = false, bool reduce_wgrad_now = false,
                            bool defer_scatter = false, int64_t sample_draw = -1) {
  const uint32_t R = b->n_rays;
  const uint32_t *d_S = f->ws.offsets + R;
  nsm_status st = clear_grads_if_dirty(f);
  if (st != NSM_OK) return st;
  if (f->timeline_on) {   // this step's slot of the ring; the slot used 8 steps from now is reset here, well ahead of its use
    f->ws.timeline = f->timeline_base + (size_t)((f->step + 1) % 64) * 2 * K_COUNT;
    unsigned long long *later = f->timeline_base + (size_t)((f->step + 9) % 64) * 2 * K_COUNT;
    CUDA_TRY(cudaMemsetAsync(later, 0xff, sizeof(unsigned long long) * K_COUNT, f->stream));
    CUDA_TRY(cudaMemsetAsync(later + K_COUNT, 0, sizeof(unsigned long long) * K_COUNT, f->stream));
  }
  st = enqueue_forward(f, b, R, f->cfg.jitter != 0, f->step + 1, true, march_on_side, dirs_copy, sample_draw);
  if (st != NSM_OK) return st;
  f->side_ok = false;
  RUN(f, K_COMPOSITE, launch_composite_train(f->ws, R, b->rgb, b->depth, b->depth_var, lambda_d, f->cfg.bg, f->stream));
  if (want_stats) {
    CUDA_TRY(cudaEventRecord(f->ev_comp, f->stream));
    CUDA_TRY(cudaStreamWaitEvent(f->side, f->ev_comp, 0));
    CUDA_TRY(cudaMemcpyAsync(f->pinned->acc, f->ws.loss_acc, 3 * sizeof(double), cudaMemcpyDeviceToHost, f->side));
    CUDA_TRY(cudaEventRecord(f->ev_stats, f->side));
    f->stats_pending = true;
  }
  if (f->use_tc)
  {
    RUN(f, K_MLP_BWD, launch_mlp_backward_tc(f->ms, f->cfg.mlp_precision == NSM_MLP_BF16, f->ws, d_S, f->n_sms, f->stream));
    f->wgrad_parts = mlp_tc_backward_ctas(f->n_sms);
    if (reduce_wgrad_now) {   // nsm_backward: leave the complete gradient in mlp_grad
      RUN(f, K_MLP_BWD, launch_reduce_wgrad(f->ms, f->ws, f->fp.mlp_grad, f->wgrad_parts, d_S, f->stream));
      f->wgrad_parts = 0;
    }
  }
  else
    RUN(f, K_MLP_BWD, launch_mlp_backward_simt(f->ms, f->fp.mlp_theta, f->fp.mlp_grad, dirs_copy ? dirs_copy : b->dirs,
                                               f->ws, d_S, f->n_sms, f->stream));
  if (f->pose_grads) {   // row f2: needs dL/de, dL/dY of this step and the PRE-update theta: between the MLP backward and Adam
    f->last_sampled = sample_draw >= 0;
    RUN(f, K_POSE, launch_pose_gradients(f->lv, f->fp.theta, f->ws, d_S, R, dirs_copy ? dirs_copy : b->dirs, 1.0f / f->cfg.aabb_extent,
                                         f->cfg.sh_degree, f->pose_go, f->pose_tau, f->last_sampled ? f->ray_kf : nullptr, f->kf_grad,
                                         (uint32_t)f->kf_host.size(), f->n_sms, f->stream, f->pose_levels));
  }
  // train step: the scatter is issued by enqueue_adam, behind the MLP Adam's hand-off to the side stream
  f->scatter_pending = defer_scatter;
  if (!defer_scatter) RUN(f, K_SCATTER, launch_scatter(f->lv, f->fp.grad, f->ws, d_S, f->n_sms, f->stream, f->work_seq++));
  f->grads_dirty = true;
  f->last_R = R;
  f->last_K = b->n_candidates;
  f->last_was_render = false;
  CUDA_TRY(cudaGetLastError());
  return NSM_OK;
}

nsm_status enqueue_adam(nsm_field *f) {
  const uint32_t t = f->step + 1;
  const double bc1 = 1.0 - std::pow((double)f->cfg.beta1, (double)t);
  const double bc2 = 1.0 - std::pow((double)f->cfg.beta2, (double)t);
  // the MLP Adam (9-11 K weights + the 16-bit image refresh) runs on the side stream beside the scatter and the table Adam
  const bool use_side = !f->prof.on;
  cudaStream_t s_mlp = use_side ? f->side : f->stream;
  if (use_side) {
    CUDA_TRY(cudaEventRecord(f->ev_pre_adam, f->stream));
    CUDA_TRY(cudaStreamWaitEvent(f->side, f->ev_pre_adam, 0));
  }
  if (f->use_tc) {
    const AdamConst c{f->cfg.lr, f->cfg.beta1, f->cfg.beta2, f->cfg.eps, (float)(1.0 / bc1), (float)(1.0 / bc2)};
    RUN_ON(f, K_ADAM_MLP, s_mlp, launch_adam_mlp_pack(f->ms, f->cfg.mlp_precision == NSM_MLP_BF16, f->fp, f->ws, c, f->wgrad_parts,
                                                      f->ws.offsets + f->last_R, s_mlp));
    f->wgrad_parts = 0;
  } else {
    RUN_ON(f, K_ADAM_MLP, s_mlp, launch_adam_mlp(f->fp, f->cfg.lr, f->cfg.beta1, f->cfg.beta2, f->cfg.eps, (float)(1.0 / bc1),
                                                 (float)(1.0 / bc2), s_mlp));
  }
  // S12 + S13 on the tables: one scatter, one Adam.  (Issuing them per level group, so that a group's slice of the
  // gradient array stays in L2 between its uses, was measured in round 1 -- profiles/r1j: every extra pair of launches
  // costs ~19 us of ramp and tail, more than the DRAM traffic it saves.)
  if (f->scatter_pending)
    RUN(f, K_SCATTER, launch_scatter(f->lv, f->fp.grad, f->ws, f->ws.offsets + f->last_R, f->n_sms, f->stream, f->work_seq++));
  f->scatter_pending = false;
  if (use_side) {   // the scatter is in: the side stream (next step's marcher) may overwrite the samples
    CUDA_TRY(cudaEventRecord(f->ev_main, f->stream));
    CUDA_TRY(cudaStreamWaitEvent(f->side, f->ev_main, 0));
  }
  RUN(f, K_ADAM_TABLE, launch_adam_table(f->fp, f->cfg.n_features, f->cfg.sparse_table_adam != 0, f->cfg.lr, f->cfg.beta1, f->cfg.beta2,
                                         f->cfg.eps, (float)(1.0 / bc1), (float)(1.0 / bc2), f->stream, f->ws.timeline,
                                         (uint64_t)f->last_R * f->last_K));
  if (use_side) {   // to be joined (lazily, join_side): everything later on the main stream must see the new MLP weights
    CUDA_TRY(cudaEventRecord(f->ev_side, f->side));
    f->join_pending = true;
    f->side_ok = true;
  }
  f->step = t;
  if (f->prof.on) f->prof.collect();
  f->grads_dirty = false;   // the Adam kernels clear what they consume
  CUDA_TRY(cudaGetLastError());
  return NSM_OK;
}

nsm_status read_stats(nsm_field *f, uint32_t R, nsm_step_stats *out) {
  if (!out) return NSM_OK;
  if (!f->stats_pending) return fail(NSM_ERR_INVALID_ARG, "internal: statistics were not requested for this step");
  CUDA_TRY(cudaEventSynchronize(f->ev_stats));   // S1-S9 of this step are done; S10-S13 may still be running
  f->stats_pending = false;
  f->pinned->S = (uint32_t)f->pinned->acc[2];
  out->loss_rgb = f->pinned->acc[0] / (double)R;
  out->loss_depth = f->pinned->acc[1] / (double)R;
  out->n_samples = f->pinned->S;
  out->n_rays = R;
  out->step = f->step;
  return NSM_OK;
}

// copy a host batch into the device staging area; returns a batch of device pointers
nsm_status stage_batch(nsm_field *f, const nsm_ray_batch *hb, uint32_t first, uint32_t R, bool train, nsm_ray_batch *db) {
  float *p = f->stage_dev;
  const uint32_t M = f->cfg.max_rays;
  *db = *hb;
  db->n_rays = R;
  CUDA_TRY(cudaMemcpyAsync(p, hb->origins + 3 * (size_t)first, sizeof(float) * 3 * R, cudaMemcpyHostToDevice, f->stream));
  db->origins = p;
  CUDA_TRY(cudaMemcpyAsync(p + 3 * M, hb->dirs + 3 * (size_t)first, sizeof(float) * 3 * R, cudaMemcpyHostToDevice, f->stream));
  db->dirs = p + 3 * M;
  if (train) {
    CUDA_TRY(cudaMemcpyAsync(p + 6 * M, hb->rgb + 3 * (size_t)first, sizeof(float) * 3 * R, cudaMemcpyHostToDevice, f->stream));
    CUDA_TRY(cudaMemcpyAsync(p + 9 * M, hb->depth + first, sizeof(float) * R, cudaMemcpyHostToDevice, f->stream));
    CUDA_TRY(cudaMemcpyAsync(p + 10 * M, hb->depth_var + first, sizeof(float) * R, cudaMemcpyHostToDevice, f->stream));
    db->rgb = p + 6 * M;
    db->depth = p + 9 * M;
    db->depth_var = p + 10 * M;
  }
  return NSM_OK;
}

}  // namespace

extern "C" {

const char *nsm_last_error(void) { return g_err.c_str(); }
const char *nsm_version(void) { return "nsm 0.1 (sm_100a)"; }
uint64_t nsm_launch_count(const nsm_field *f) { return f ? f->launches : 0; }
const char *nsm_mlp_path(const nsm_field *f) { return f ? f->mlp_path : ""; }

nsm_status nsm_create_field(const nsm_field_config *cfg, void *cuda_stream, nsm_field **out) {
  if (!out) return fail(NSM_ERR_INVALID_ARG, "out is NULL");
  *out = nullptr;
  nsm_status st = validate_config(cfg);
  if (st != NSM_OK) return st;
  int dev = 0, n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) {
    cudaGetLastError();
    return fail(NSM_ERR_CUDA, "no CUDA device: this library has no CPU fallback");
  }
  CUDA_TRY(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  CUDA_TRY(cudaGetDeviceProperties(&prop, dev));
  if (prop.major != 10 || prop.minor != 0)   // the library holds sm_100a code only (tcgen05 / TMEM paths are not forward-compatible)
    return fail(NSM_ERR_CUDA, "device sm_%d%d is not sm_100: built for B200 (sm_100a) only", prop.major, prop.minor);

  nsm_field *f = new (std::nothrow) nsm_field();
  if (!f) return fail(NSM_ERR_OOM, "host allocation failed");
  f->cfg = *cfg;
  f->device = dev;
  f->stream = (cudaStream_t)cuda_stream;
  f->n_sms = prop.multiProcessorCount;
  build_levels(*cfg, f->lv, f->fp.map);
  MlpShape &ms = f->ms;
  ms.LF = cfg->n_levels * cfg->n_features;
  ms.Hd = cfg->density_hidden; ms.Do = cfg->density_out;
  ms.sh_degree = cfg->sh_degree; ms.n_sh = cfg->sh_degree * cfg->sh_degree;
  ms.geo_off = cfg->geo_offset; ms.geo_cnt = cfg->geo_count;
  ms.Ci = ms.geo_cnt + ms.n_sh; ms.Hc = cfg->color_hidden; ms.n_color_layers = cfg->color_hidden_layers;
  uint32_t o = 0;
  ms.o_d1 = o; o += ms.Hd * ms.LF;
  ms.o_d2 = o; o += ms.Do * ms.Hd;
  ms.o_c1 = o; o += ms.Hc * ms.Ci;
  ms.o_c2 = o; o += (ms.n_color_layers == 2 ? ms.Hc * ms.Hc : 0);
  ms.o_c3 = o; o += 3 * ms.Hc;
  ms.n_mlp = o;
  if (ms.Ci > 128) { delete f; return fail(NSM_ERR_UNIMPLEMENTED, "colour input width > 128"); }
  if (mlp_simt_smem_bytes(ms, 1) > (size_t)prop.sharedMemPerBlockOptin) {
    delete f;
    return fail(NSM_ERR_UNIMPLEMENTED, "MLP shape needs %zu B shared memory (> %zu)", mlp_simt_smem_bytes(ms, 1),
                (size_t)prop.sharedMemPerBlockOptin);
  }

  // 16-bit configurations run the MLPs on tcgen05 when the shapes fit its tiles; the kernels' shared-memory opt-in is a
  // per-device attribute, set here for the field's device
  if (cfg->mlp_precision != NSM_MLP_FP32 && mlp_tc_supported(ms)) {
    f->use_tc = true;
    f->mlp_path = cfg->mlp_precision == NSM_MLP_BF16 ? "tcgen05_bf16" : "tcgen05_f16";
    const cudaError_t ea = mlp_tc_prepare_device();
    if (ea != cudaSuccess) {
      delete f;
      cudaGetLastError();
      return fail(NSM_ERR_CUDA, "tcgen05 kernel attributes: %s", cudaGetErrorString(ea));
    }
  }
  FieldParams &fp = f->fp;
  fp.n_entries = f->lv.offset[cfg->n_levels];
  fp.n_canon = fp.map.canon[cfg->n_levels];
  fp.n_table = fp.n_canon * cfg->n_features;
  fp.n_mlp = ms.n_mlp;
  fp.F = cfg->n_features;
  Workspace &ws = f->ws;
  const uint64_t cap = (((uint64_t)cfg->max_rays * cfg->max_candidates + NSM_TILE - 1) / NSM_TILE) * NSM_TILE;
  ws.cap = cap;
  ws.max_rays = cfg->max_rays;
  const uint64_t G3 = (uint64_t)(cfg->occ_cascades ? cfg->occ_cascades : 1) * cfg->occ_res * cfg->occ_res * cfg->occ_res;   // all cascades
  const uint32_t R = cfg->max_rays;
  cudaError_t e = cudaSuccess;
  auto A = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  const uint64_t n_store = fp.n_entries * cfg->n_features;   // floats of a storage array (padding included)
  A(f->alloc(&fp.theta, n_store)); A(f->alloc(&fp.mv, 2 * n_store));
  A(f->alloc(&fp.mlp_theta, fp.n_mlp)); A(f->alloc(&fp.mlp_m, fp.n_mlp)); A(f->alloc(&fp.mlp_v, fp.n_mlp)); A(f->alloc(&fp.mlp_grad, fp.n_mlp));
  A(f->alloc(&fp.grad, n_store, false)); A(f->alloc(&fp.occ_bits, (G3 + 7) / 8 + 4));
  A(f->alloc(&fp.occ_grid, G3));
  A(f->alloc(&ws.counts, R)); A(f->alloc(&ws.offsets, R + 1)); A(f->alloc(&ws.scan_state, march_scan_state_entries(R) + 1)); A(f->alloc(&ws.scan_ctr, 2)); A(f->alloc(&ws.work_ctr, 8));
  A(f->alloc(&ws.C, 3 * (size_t)R)); A(f->alloc(&ws.D_hat, R)); A(f->alloc(&ws.O, R));
  A(f->alloc(&ws.s_ray, cap)); A(f->alloc(&ws.s_k, cap)); A(f->alloc(&ws.s_t, cap)); A(f->alloc(&ws.s_delta, cap));
  A(f->alloc(&ws.s_x, 3 * cap));
  ws.e = ws.hd = ws.g = ws.h1 = ws.h2 = nullptr;
  ws.blob_e = ws.blob_hd = ws.blob_ci = ws.blob_h1 = ws.blob_h2 = ws.wimg_fwd = ws.wimg_bwd = nullptr;
  ws.wgrad_part = nullptr;
  if (f->use_tc) {   // 16-bit operand-tile blobs: 2 bytes per value, 128-row tiles
    A(f->alloc(&ws.blob_e, 4 * ms.LF * cap));   /* two-term (hi | lo) tiles */ A(f->alloc(&ws.blob_hd, 2 * ms.Hd * cap)); A(f->alloc(&ws.blob_ci, 2 * 32 * cap));
    A(f->alloc(&ws.blob_h1, 2 * ms.Hc * cap)); A(f->alloc(&ws.blob_h2, 2 * (ms.n_color_layers == 2 ? ms.Hc : 1) * cap));
    A(f->alloc(&ws.wimg_fwd, mlp_tc_wimg_bytes(0))); A(f->alloc(&ws.wimg_bwd, mlp_tc_wimg_bytes(1)));
    A(f->alloc(&ws.wgrad_part, (size_t)mlp_tc_backward_ctas(f->n_sms) * ms.n_mlp));
  } else {
    A(f->alloc(&ws.e, ms.LF * cap)); A(f->alloc(&ws.hd, ms.Hd * cap)); A(f->alloc(&ws.g, ms.Do * cap));
    A(f->alloc(&ws.h1, ms.Hc * cap)); A(f->alloc(&ws.h2, (ms.n_color_layers == 2 ? ms.Hc : 1) * cap));
  }
  A(f->alloc(&ws.sigma, cap)); A(f->alloc(&ws.rgb, 3 * cap)); A(f->alloc(&ws.T_excl, cap));
  A(f->alloc(&ws.dsigma, cap)); A(f->alloc(&ws.drgb, 3 * cap)); A(f->alloc(&ws.de, ms.LF * cap));
  A(f->alloc(&f->kf_dev, NSM_MAX_KEYFRAMES));
  ws.dY = ws.dx = nullptr;
  ws.timeline = nullptr;
  A(f->alloc(&ws.loss_acc, 3)); A(f->alloc(&ws.total_samples, 1)); A(f->alloc(&ws.grad_absmax, 1));
  A(f->alloc(&f->stage_dev, 12 * (size_t)R)); A(f->alloc(&f->stage_out, 10 * (size_t)R));
  if (e == cudaSuccess) e = cudaMallocHost((void **)&f->pinned, sizeof(*f->pinned));
  if (e == cudaSuccess) {   // highest priority: the side stream's small grids must not queue behind the table Adam's 3000 blocks
    int prio_lo = 0, prio_hi = 0;
    cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
    e = cudaStreamCreateWithPriority(&f->side, cudaStreamNonBlocking, prio_hi);
  }
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_pre_adam, cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_side, cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_main, cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_comp, cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_stats, cudaEventDisableTiming);
  for (int j = 0; j < 2; ++j) {
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_in[j], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_done[j], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&f->ev_outfree[j], cudaEventDisableTiming);
  }
  if (e != cudaSuccess) {
    nsm_destroy_field(f);
    cudaGetLastError();
    return fail(e == cudaErrorMemoryAllocation ? NSM_ERR_OOM : NSM_ERR_CUDA, "allocation failed: %s", cudaGetErrorString(e));
  }
  RUN(f, K_DEBUG, launch_set_grad(f->fp, nullptr, nullptr, f->stream));   // every gradient word = "untouched"
  repack_weights(f);
  *out = f;
  return NSM_OK;
}

void nsm_destroy_field(nsm_field *f) {
  if (!f) return;
  cudaStreamSynchronize(f->stream);
  if (f->side) { cudaStreamSynchronize(f->side); cudaStreamDestroy(f->side); }
  if (f->ev_pre_adam) cudaEventDestroy(f->ev_pre_adam);
  if (f->ev_side) cudaEventDestroy(f->ev_side);
  if (f->ev_main) cudaEventDestroy(f->ev_main);
  if (f->ev_comp) cudaEventDestroy(f->ev_comp);
  if (f->ev_stats) cudaEventDestroy(f->ev_stats);
  for (int j = 0; j < 2; ++j) {
    if (f->ev_in[j]) cudaEventDestroy(f->ev_in[j]);
    if (f->ev_done[j]) cudaEventDestroy(f->ev_done[j]);
    if (f->ev_outfree[j]) cudaEventDestroy(f->ev_outfree[j]);
  }
  f->prof.destroy();
  for (void *p : f->allocs) cudaFree(p);
  if (f->pinned) cudaFreeHost(f->pinned);
  delete f;
}

nsm_status nsm_total_samples(nsm_field *f, uint64_t *out) {
  if (!f || !out) return fail(NSM_ERR_INVALID_ARG, "NULL argument");
  unsigned long long v = 0;
  LEAVE_FAST_PATH(f);   // the marcher (side stream) maintains the count
  CUDA_TRY(cudaMemcpyAsync(&v, f->ws.total_samples, sizeof v, cudaMemcpyDeviceToHost, f->stream));
  CUDA_TRY(cudaStreamSynchronize(f->stream));
  *out = v;
  return NSM_OK;
}

nsm_status nsm_profile(nsm_field *f, int enable) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  LEAVE_FAST_PATH(f);
  CUDA_TRY(cudaStreamSynchronize(f->stream));
  f->prof.collect();
  f->prof.on = enable != 0;
  if (enable) for (int i = 0; i < K_COUNT; ++i) { f->prof.ms[i] = 0.0; f->prof.n[i] = 0; }
  return NSM_OK;
}

nsm_status nsm_profile_read(nsm_field *f, uint32_t capacity, const char **names, double *total_ms, uint64_t *launches,
                            uint32_t *n_out) {
  if (!f || !n_out) return fail(NSM_ERR_INVALID_ARG, "NULL argument");
  f->prof.collect();
  if (f->prof.failed) {
    f->prof.failed = false;
    return fail(NSM_ERR_CUDA, "a timing event of the per-kernel pass could not be recorded or read");
  }
  *n_out = K_COUNT;
  for (uint32_t i = 0; i < capacity && i < K_COUNT; ++i) {
    if (names) names[i] = kKernelNames[i];
    if (total_ms) total_ms[i] = f->prof.ms[i];
    if (launches) launches[i] = f->prof.on ? f->prof.n[i] : f->launches_by[i];
  }
  return NSM_OK;
}

nsm_status nsm_param_count(const nsm_field *f, uint64_t *n_table, uint64_t *n_mlp) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  if (n_table) *n_table = f->fp.n_table;
  if (n_mlp) *n_mlp = f->fp.n_mlp;
  return NSM_OK;
}

nsm_status nsm_get_level_table(const nsm_field *f, uint32_t *res, uint64_t *offset) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  for (uint32_t l = 0; l < f->lv.n_levels; ++l) {
    if (res) res[l] = f->lv.res[l];
    if (offset) offset[l] = f->fp.map.canon[l];
  }
  if (offset) offset[f->lv.n_levels] = f->fp.map.canon[f->lv.n_levels];
  return NSM_OK;
}

nsm_status nsm_get_params(nsm_field *f, float *d_theta, float *d_m, float *d_v, uint32_t *step) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  LEAVE_FAST_PATH(f);
  const size_t mb = sizeof(float) * f->fp.n_mlp;
  float *dst[3] = {d_theta, d_m, d_v};
  const float *mlp[3] = {f->fp.mlp_theta, f->fp.mlp_m, f->fp.mlp_v};
  const int which[3] = {0, 2, 3};
  for (int i = 0; i < 3; ++i) {
    if (!dst[i]) continue;
    RUN(f, K_DEBUG, launch_unpack_records(f->fp, which[i], dst[i], f->stream));
    CUDA_TRY(cudaMemcpyAsync(dst[i] + f->fp.n_table, mlp[i], mb, cudaMemcpyDeviceToDevice, f->stream));
  }
  if (step) *step = f->step;
  CUDA_TRY(cudaGetLastError());
  return NSM_OK;
}

nsm_status nsm_set_params(nsm_field *f, const float *d_theta, const float *d_m, const float *d_v, uint32_t step) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  LEAVE_FAST_PATH(f);
  const size_t mb = sizeof(float) * f->fp.n_mlp;
  const float *src[3] = {d_theta, d_m, d_v};
  float *mlp[3] = {f->fp.mlp_theta, f->fp.mlp_m, f->fp.mlp_v};
  const int which[3] = {0, 2, 3};
  for (int i = 0; i < 3; ++i) {
    if (!src[i]) continue;
    RUN(f, K_DEBUG, launch_pack_records(f->fp, which[i], src[i], f->stream));
    CUDA_TRY(cudaMemcpyAsync(mlp[i], src[i] + f->fp.n_table, mb, cudaMemcpyDeviceToDevice, f->stream));
  }
  if (d_theta) repack_weights(f);
  f->step = step;
  CUDA_TRY(cudaGetLastError());
  return NSM_OK;
}

nsm_status nsm_get_occupancy(nsm_field *f, uint8_t *d_bits) {
  if (!f || !d_bits) return fail(NSM_ERR_INVALID_ARG, "NULL argument");
  LEAVE_FAST_PATH(f);
  const uint64_t G3 = occ_cells(f);
  if (f->occ_full) CUDA_TRY(cudaMemsetAsync(d_bits, 0xff, (G3 + 7) / 8, f->stream));
  else CUDA_TRY(cudaMemcpyAsync(d_bits, f->fp.occ_bits, (G3 + 7) / 8, cudaMemcpyDeviceToDevice, f->stream));
  return NSM_OK;
}

nsm_status nsm_update_occupancy(nsm_field *f, nsm_occ_mode mode, const uint8_t *d_bits) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  LEAVE_FAST_PATH(f);
  const uint64_t G3 = occ_cells(f);
  switch (mode) {
    case NSM_OCC_FULL:
      f->occ_full = true;
      f->grid_seeded = false;
      f->occ_updates = 0;
      return NSM_OK;
    case NSM_OCC_SET:
      if (!d_bits) return fail(NSM_ERR_INVALID_ARG, "d_bits is NULL");
      CUDA_TRY(cudaMemcpyAsync(f->fp.occ_bits, d_bits, (G3 + 7) / 8, cudaMemcpyDeviceToDevice, f->stream));
      f->occ_full = false;
      f->grid_seeded = false;
      f->occ_updates = 0;
      return NSM_OK;
    case NSM_OCC_FROM_FIELD: {
      // the cell centres go through S4 + S5 in chunks of the workspace capacity (multiples of 32)
      const uint64_t chunk = f->ws.cap & ~uint64_t(31);
      uint32_t *d_S = f->ws.offsets;  // offsets[0] doubles as the chunk's sample count
      for (uint64_t first = 0; first < G3; first += chunk) {
        const uint64_t n = (G3 - first < chunk) ? G3 - first : chunk;
        RUN(f, K_OCC, launch_occ_cells(f->cfg.occ_res, occ_cascades(f), first, 1, n, f->ws, d_S, f->stream));
        RUN(f, K_ENCODE, launch_encode(f->lv, f->fp.theta, f->ws, d_S, f->use_tc ? 1 + (f->cfg.mlp_precision == NSM_MLP_BF16) : 0,
                                       f->n_sms, f->stream, f->work_seq++, n, false));
        f->e_two_term = false;
        if (f->use_tc)
          RUN(f, K_MLP_FWD, launch_mlp_forward_tc(f->ms, f->cfg.mlp_precision == NSM_MLP_BF16, nullptr, f->ws, d_S, 1, 0, f->n_sms,
                                                  f->stream));
        else
          RUN(f, K_MLP_FWD, launch_mlp_forward_simt(f->ms, f->fp.mlp_theta, nullptr, f->ws, d_S, 1, f->n_sms, f->stream));
        RUN(f, K_OCC, launch_occ_threshold(f->cfg.occ_res, first, n, f->ws.sigma, f->cfg.occ_sigma_threshold,
                                           f->fp.occ_bits, f->fp.occ_grid, f->stream));
      }
      f->occ_full = false;
      f->grid_seeded = true;
      f->occ_updates = 0;
      CUDA_TRY(cudaGetLastError());
      return NSM_OK;
    }
  }
  return fail(NSM_ERR_INVALID_ARG, "bad occupancy mode %d", (int)mode);
}

// F4: decayed running maximum + strided partial refresh (paper silent, after [17])
nsm_status nsm_update_occupancy_decay(nsm_field *f, uint32_t n_subsets, float decay) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  if (n_subsets == 0) return fail(NSM_ERR_INVALID_ARG, "n_subsets is 0");
  if (!(decay >= 0.f && decay <= 1.f)) return fail(NSM_ERR_INVALID_ARG, "decay must be in [0, 1]");
  if (!f->grid_seeded)   // after SET / FULL the running grid says nothing about the cells a partial pass does not visit
    return fail(NSM_ERR_INVALID_ARG, "the running density grid is not seeded: call nsm_update_occupancy(NSM_OCC_FROM_FIELD) first");
  LEAVE_FAST_PATH(f);
  const uint64_t G3 = occ_cells(f);
  const uint64_t c0 = f->occ_updates % n_subsets;
  const uint64_t n_vis = c0 < G3 ? (G3 - c0 + n_subsets - 1) / n_subsets : 0;
  const uint64_t chunk = f->ws.cap & ~uint64_t(31);
  const int bf16 = f->cfg.mlp_precision == NSM_MLP_BF16;
  uint32_t *d_S = f->ws.offsets;
  RUN(f, K_OCC, launch_occ_decay(f->fp.occ_grid, G3, decay, f->stream));
  for (uint64_t j0 = 0; j0 < n_vis; j0 += chunk) {
    const uint64_t n = (n_vis - j0 < chunk) ? n_vis - j0 : chunk;
    const uint64_t first = c0 + j0 * n_subsets;
    RUN(f, K_OCC, launch_occ_cells(f->cfg.occ_res, occ_cascades(f), first, n_subsets, n, f->ws, d_S, f->stream));
    RUN(f, K_ENCODE, launch_encode(f->lv, f->fp.theta, f->ws, d_S, f->use_tc ? 1 + bf16 : 0, f->n_sms, f->stream, f->work_seq++, n, false));
    f->e_two_term = false;
    if (f->use_tc)
      RUN(f, K_MLP_FWD, launch_mlp_forward_tc(f->ms, bf16, nullptr, f->ws, d_S, 1, 0, f->n_sms, f->stream));
    else
      RUN(f, K_MLP_FWD, launch_mlp_forward_simt(f->ms, f->fp.mlp_theta, nullptr, f->ws, d_S, 1, f->n_sms, f->stream));
    RUN(f, K_OCC, launch_occ_max_visited(f->fp.occ_grid, first, n_subsets, n, f->ws.sigma, f->stream));
  }
  RUN(f, K_OCC, launch_occ_bits_from_grid(f->fp.occ_grid, G3, f->cfg.occ_sigma_threshold, f->fp.occ_bits, f->stream));
  f->occ_full = false;
  f->occ_updates += 1;
  CUDA_TRY(cudaGetLastError());
  return NSM_OK;
}

// F4, stochastic variant (reading R25): decayed running maximum refreshed at n_draws hashed random points
nsm_status nsm_update_occupancy_stochastic(nsm_field *f, uint32_t n_draws, float decay) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  if (!(decay >= 0.f && decay <= 1.f)) return fail(NSM_ERR_INVALID_ARG, "decay must be in [0, 1]");
  if (!f->grid_seeded)
    return fail(NSM_ERR_INVALID_ARG, "the running density grid is not seeded: call nsm_update_occupancy(NSM_OCC_FROM_FIELD) first");
  LEAVE_FAST_PATH(f);
  const uint64_t G3 = occ_cells(f);
  const uint32_t chunk = (uint32_t)std::min<uint64_t>(f->ws.cap & ~uint64_t(31), 1u << 30);
  const int bf16 = f->cfg.mlp_precision == NSM_MLP_BF16;
  uint32_t *d_S = f->ws.offsets;
  RUN(f, K_OCC, launch_occ_decay(f->fp.occ_grid, G3, decay, f->stream));
  for (uint32_t i0 = 0; i0 < n_draws; i0 += chunk) {
    const uint32_t n = n_draws - i0 < chunk ? n_draws - i0 : chunk;
    RUN(f, K_OCC, launch_occ_cells_stochastic(f->cfg.occ_res, occ_cascades(f), f->cfg.seed, f->occ_draws, i0, n, f->ws, d_S, f->stream));
    RUN(f, K_ENCODE, launch_encode(f->lv, f->fp.theta, f->ws, d_S, f->use_tc ? 1 + bf16 : 0, f->n_sms, f->stream, f->work_seq++, n, false));
    f->e_two_term = false;
    if (f->use_tc)
      RUN(f, K_MLP_FWD, launch_mlp_forward_tc(f->ms, bf16, nullptr, f->ws, d_S, 1, 0, f->n_sms, f->stream));
    else
      RUN(f, K_MLP_FWD, launch_mlp_forward_simt(f->ms, f->fp.mlp_theta, nullptr, f->ws, d_S, 1, f->n_sms, f->stream));
    RUN(f, K_OCC, launch_occ_max_cells(f->fp.occ_grid, f->ws.s_k, n, f->ws.sigma, f->stream));
  }
  RUN(f, K_OCC, launch_occ_bits_from_grid(f->fp.occ_grid, G3, f->cfg.occ_sigma_threshold, f->fp.occ_bits, f->stream));
  f->occ_full = false;
  f->occ_draws += 1;
  CUDA_TRY(cudaGetLastError());
  return NSM_OK;
}

nsm_status nsm_get_occupancy_grid(nsm_field *f, float *d_grid) {
  if (!f || !d_grid) return fail(NSM_ERR_INVALID_ARG, "NULL argument");
  LEAVE_FAST_PATH(f);
  const uint64_t G3 = occ_cells(f);
  CUDA_TRY(cudaMemcpyAsync(d_grid, f->fp.occ_grid, sizeof(float) * G3, cudaMemcpyDeviceToDevice, f->stream));
  return NSM_OK;
}

nsm_status nsm_backward(nsm_field *f, const nsm_ray_batch *batch, float lambda_d, nsm_step_stats *host_stats) {
  nsm_status st = validate_batch(f, batch, true, false);
  if (st != NSM_OK) return st;
  LEAVE_FAST_PATH(f);
  st = enqueue_backward(f, batch, lambda_d, false, nullptr, host_stats != nullptr, true);
  if (st != NSM_OK) return st;
  st = read_stats(f, batch->n_rays, host_stats);
  if (st == NSM_OK && host_stats) host_stats->loss = host_stats->loss_rgb + (double)lambda_d * host_stats->loss_depth;
  return st;
}

nsm_status nsm_apply_adam(nsm_field *f) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  LEAVE_FAST_PATH(f);
  return enqueue_adam(f);
}

static nsm_status train_step_impl(nsm_field *f, const nsm_ray_batch *batch, float lambda_d, nsm_step_stats *host_stats,
                                  bool batch_ready, float *dirs_copy = nullptr, int64_t sample_draw = -1) {
  nsm_status st = validate_batch(f, batch, true, false);
  if (st != NSM_OK) return st;
  st = enqueue_backward(f, batch, lambda_d, batch_ready, dirs_copy, host_stats != nullptr, false, true, sample_draw);
  if (st != NSM_OK) return st;
  st = enqueue_adam(f);
  if (st != NSM_OK) return st;
  st = read_stats(f, batch->n_rays, host_stats);
  if (st == NSM_OK && host_stats) host_stats->loss = host_stats->loss_rgb + (double)lambda_d * host_stats->loss_depth;
  return st;
}

nsm_status nsm_train_step(nsm_field *f, const nsm_ray_batch *batch, float lambda_d, nsm_step_stats *host_stats) {
  return train_step_impl(f, batch, lambda_d, host_stats, f && f->batch_ready);
}

// device alias of a pinned (page-locked, device-mapped) host pointer, or NULL for pageable memory
static const float *host_mapped(const float *p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return a.type == cudaMemoryTypeHost ? (const float *)a.devicePointer : nullptr;
}

nsm_status nsm_train_step_host(nsm_field *f, const nsm_ray_batch *hb, float lambda_d, nsm_step_stats *host_stats) {
  nsm_status st = validate_batch(f, hb, true, false);
  if (st != NSM_OK) return st;
  nsm_step_stats local;
  nsm_ray_batch db = *hb;
  // Pinned host buffers are read IN PLACE over the host link: every input is needed exactly once per ray (origins and
  // directions by the marcher, which leaves a device copy of the directions for the MLPs; colour, depth and variance
  // by the compositor), so there is nothing a staging copy would save -- and five small DMA launches to lose.
  db.origins = host_mapped(hb->origins); db.dirs = host_mapped(hb->dirs); db.rgb = host_mapped(hb->rgb);
  db.depth = host_mapped(hb->depth); db.depth_var = host_mapped(hb->depth_var);
  if (db.origins && db.dirs && db.rgb && db.depth && db.depth_var)   // the call syncs: the host buffers are free on return
    return train_step_impl(f, &db, lambda_d, host_stats ? host_stats : &local, true, f->stage_dev + 3 * (size_t)f->cfg.max_rays);
  LEAVE_FAST_PATH(f);   // pageable memory: staging copies through the main stream
  st = stage_batch(f, hb, 0, hb->n_rays, true, &db);
  if (st != NSM_OK) return st;
  return train_step_impl(f, &db, lambda_d, host_stats ? host_stats : &local, false);  // always syncs: host buffers may be reused
}

nsm_status nsm_debug_timeline(nsm_field *f, uint64_t *h_out, uint64_t capacity_words, uint32_t *n_kernels) {
  if (!f || !h_out) return fail(NSM_ERR_INVALID_ARG, "NULL argument");
  if (!f->timeline_base) return fail(NSM_ERR_INVALID_ARG, "timeline not enabled (nsm_set_option(NSM_OPT_DEBUG_TIMELINE, 1))");
  if (capacity_words < 64ull * 2 * K_COUNT) return fail(NSM_ERR_CAPACITY, "timeline needs %d words", 64 * 2 * K_COUNT);
  CUDA_TRY(cudaStreamSynchronize(f->stream));
  CUDA_TRY(cudaMemcpy(h_out, f->timeline_base, sizeof(uint64_t) * 64 * 2 * K_COUNT, cudaMemcpyDeviceToHost));
  if (n_kernels) *n_kernels = K_COUNT;
  return NSM_OK;
}

// ---- F1: keyframe store and sampled training -------------------------------------------------------------------
nsm_status nsm_add_keyframe(nsm_field *f, const nsm_keyframe_info *info, const float *d_rgb, const float *d_depth,
                            const float *d_depth_var, uint32_t *index_out) {
  if (!f || !info || !d_rgb || !d_depth || !d_depth_var) return fail(NSM_ERR_INVALID_ARG, "NULL argument");
  if (info->width == 0 || info->height == 0 || (uint64_t)info->width * info->height > (1ull << 31))
    return fail(NSM_ERR_INVALID_ARG, "bad keyframe size %u x %u", info->width, info->height);
  if (!(info->fx > 0.f) || !(info->fy > 0.f) || !std::isfinite(info->fx) || !std::isfinite(info->fy))
    return fail(NSM_ERR_INVALID_ARG, "focal lengths must be positive");
  if (f->kf_host.size() >= NSM_MAX_KEYFRAMES) return fail(NSM_ERR_CAPACITY, "keyframe store is full (%d)", NSM_MAX_KEYFRAMES);
  LEAVE_FAST_PATH(f);
  const size_t n = (size_t)info->width * info->height;
  float *buf = nullptr;
  CUDA_TRY(f->alloc(&buf, 5 * n, false));
  CUDA_TRY(cudaMemcpyAsync(buf, d_rgb, sizeof(float) * 3 * n, cudaMemcpyDeviceToDevice, f->stream));
  CUDA_TRY(cudaMemcpyAsync(buf + 3 * n, d_depth, sizeof(float) * n, cudaMemcpyDeviceToDevice, f->stream));
  CUDA_TRY(cudaMemcpyAsync(buf + 4 * n, d_depth_var, sizeof(float) * n, cudaMemcpyDeviceToDevice, f->stream));
  KeyframeDev k;
  k.W = info->width; k.H = info->height;
  k.fx = info->fx; k.fy = info->fy; k.cx = info->cx; k.cy = info->cy;
  for (int i = 0; i < 9; ++i) k.R[i] = info->R[i];
  for (int i = 0; i < 3; ++i) k.t[i] = info->t[i];
  k.rgb = buf; k.depth = buf + 3 * n; k.var = buf + 4 * n;
  f->kf_host.push_back(k);
  const size_t idx = f->kf_host.size() - 1;
  // the directory entry: a pageable source is copied out by the runtime before the call returns
  CUDA_TRY(cudaMemcpyAsync(f->kf_dev + idx, &f->kf_host[idx], sizeof(KeyframeDev), cudaMemcpyHostToDevice, f->stream));
  if (index_out) *index_out = (uint32_t)idx;
  return NSM_OK;
}

nsm_status nsm_keyframe_count(const nsm_field *f, uint32_t *n_out) {
  if (!f || !n_out) return fail(NSM_ERR_INVALID_ARG, "NULL argument");
  *n_out = (uint32_t)f->kf_host.size();
  return NSM_OK;
}

nsm_status nsm_sample_batch(nsm_field *f, uint32_t n_rays, uint32_t draw, float *d_origins, float *d_dirs, float *d_rgb,
                            float *d_depth, float *d_depth_var) {
  if (!f || !d_origins || !d_dirs || !d_rgb || !d_depth || !d_depth_var) return fail(NSM_ERR_INVALID_ARG, "NULL argument");
  if (f->kf_host.empty()) return fail(NSM_ERR_INVALID_ARG, "the keyframe store is empty");
  if (n_rays == 0) return fail(NSM_ERR_INVALID_ARG, "n_rays is 0");
  LEAVE_FAST_PATH(f);
  RUN(f, K_SAMPLE, launch_sample_batch(f->kf_dev, (uint32_t)f->kf_host.size(), f->cfg.seed, draw, n_rays, d_origins, d_dirs, d_rgb,
                                       d_depth, d_depth_var, nullptr, f->stream));
  CUDA_TRY(cudaGetLastError());
  return NSM_OK;
}

nsm_status nsm_train_step_sampled(nsm_field *f, uint32_t n_rays, float t_min, float t_max, uint32_t n_candidates, float lambda_d,
                                  nsm_step_stats *host_stats) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  if (f->kf_host.empty()) return fail(NSM_ERR_INVALID_ARG, "the keyframe store is empty");
  if (n_rays > f->cfg.max_rays) return fail(NSM_ERR_CAPACITY, "n_rays %u > max_rays %u", n_rays, f->cfg.max_rays);
  // the batch lives in the field's staging area; the sampler and the marcher run beside the previous step's table Adam
  const size_t M = f->cfg.max_rays;
  nsm_ray_batch b;
  b.n_rays = n_rays;
  b.origins = f->stage_dev; b.dirs = f->stage_dev + 3 * M; b.rgb = f->stage_dev + 6 * M;
  b.depth = f->stage_dev + 9 * M; b.depth_var = f->stage_dev + 10 * M;
  b.t_min = t_min; b.t_max = t_max; b.n_candidates = n_candidates;
  return train_step_impl(f, &b, lambda_d, host_stats, true, nullptr, (int64_t)(f->step + 1));
}

// ---- row f2: pose gradients --------------------------------------------------------------------------------
nsm_status nsm_pose_gradients(nsm_field *f, float *d_g_o, float *d_tau) {
  if (!f || !d_g_o || !d_tau) return fail(NSM_ERR_INVALID_ARG, "NULL argument");
  if (!f->pose_grads || f->last_R == 0 || f->last_was_render)
    return fail(NSM_ERR_INVALID_ARG, "no pose gradients: set NSM_OPT_POSE_GRADIENTS and run a training step / nsm_backward first");
  LEAVE_FAST_PATH(f);
  CUDA_TRY(cudaMemcpyAsync(d_g_o, f->pose_go, sizeof(float) * 3 * f->last_R, cudaMemcpyDeviceToDevice, f->stream));
  CUDA_TRY(cudaMemcpyAsync(d_tau, f->pose_tau, sizeof(float) * 3 * f->last_R, cudaMemcpyDeviceToDevice, f->stream));
  return NSM_OK;
}

nsm_status nsm_keyframe_pose_gradients(nsm_field *f, float *d_out) {
  if (!f || !d_out) return fail(NSM_ERR_INVALID_ARG, "NULL argument");
  if (!f->pose_grads || !f->last_sampled || f->last_was_render)
    return fail(NSM_ERR_INVALID_ARG, "no keyframe gradients: set NSM_OPT_POSE_GRADIENTS and run nsm_train_step_sampled first");
  LEAVE_FAST_PATH(f);
  CUDA_TRY(cudaMemcpy2DAsync(d_out, sizeof(float) * 6, f->kf_grad, sizeof(float) * NSM_KF_GRAD_STRIDE, sizeof(float) * 6,
                             f->kf_host.size(), cudaMemcpyDeviceToDevice, f->stream));
  return NSM_OK;
}

nsm_status nsm_apply_pose_step(nsm_field *f, float lr_translation, float lr_rotation) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  if (!f->pose_grads || !f->last_sampled || f->last_was_render)
    return fail(NSM_ERR_INVALID_ARG, "no keyframe gradients: set NSM_OPT_POSE_GRADIENTS and run nsm_train_step_sampled first");
  if (!(lr_translation >= 0.f) || !(lr_rotation >= 0.f)) return fail(NSM_ERR_INVALID_ARG, "learning rates must be >= 0");
  LEAVE_FAST_PATH(f);
  RUN(f, K_POSE, launch_pose_step(f->kf_dev, (uint32_t)f->kf_host.size(), f->kf_grad, f->kf_pose_m, f->kf_pose_v, f->kf_pose_cnt,
                                  lr_translation, lr_rotation, f->cfg.beta1, f->cfg.beta2, f->cfg.eps, f->stream));
  f->last_sampled = false;   // the gradients are consumed
  CUDA_TRY(cudaGetLastError());
  return NSM_OK;
}

nsm_status nsm_get_keyframe_pose(nsm_field *f, uint32_t index, float *h_R, float *h_t) {
  if (!f || !h_R || !h_t) return fail(NSM_ERR_INVALID_ARG, "NULL argument");
  if (index >= f->kf_host.size()) return fail(NSM_ERR_INVALID_ARG, "keyframe index %u out of range", index);
  LEAVE_FAST_PATH(f);
  KeyframeDev k;
  CUDA_TRY(cudaMemcpyAsync(&k, f->kf_dev + index, sizeof k, cudaMemcpyDeviceToHost, f->stream));
  CUDA_TRY(cudaStreamSynchronize(f->stream));
  for (int i = 0; i < 9; ++i) h_R[i] = k.R[i];
  for (int i = 0; i < 3; ++i) h_t[i] = k.t[i];
  return NSM_OK;
}

nsm_status nsm_set_option(nsm_field *f, nsm_option opt, uint32_t value) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  switch (opt) {
    case NSM_OPT_BATCH_READY: f->batch_ready = value != 0; LEAVE_FAST_PATH(f); return NSM_OK;
    case NSM_OPT_POSE_GRADIENTS: {
      LEAVE_FAST_PATH(f);
      if (value && !f->ws.dY) {   // workspace of row f2, allocated on first use
        cudaError_t e = cudaSuccess;
        auto A = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
        A(f->alloc(&f->ws.dY, 16 * f->ws.cap)); A(f->alloc(&f->ws.dx, 3 * f->ws.cap));
        A(f->alloc(&f->pose_go, 3 * (size_t)f->cfg.max_rays)); A(f->alloc(&f->pose_tau, 3 * (size_t)f->cfg.max_rays));
        A(f->alloc(&f->kf_grad, NSM_KF_GRAD_STRIDE * NSM_MAX_KEYFRAMES)); A(f->alloc(&f->ray_kf, f->cfg.max_rays));
        A(f->alloc(&f->kf_pose_m, 6 * NSM_MAX_KEYFRAMES)); A(f->alloc(&f->kf_pose_v, 6 * NSM_MAX_KEYFRAMES));
        A(f->alloc(&f->kf_pose_cnt, NSM_MAX_KEYFRAMES));
        if (e != cudaSuccess) { cudaGetLastError(); return fail(NSM_ERR_OOM, "pose-gradient workspace: %s", cudaGetErrorString(e)); }
      }
      f->pose_grads = value != 0;
      return NSM_OK;
    }
    case NSM_OPT_POSE_LEVELS: f->pose_levels = value; return NSM_OK;
    case NSM_OPT_DEBUG_TIMELINE: {
      LEAVE_FAST_PATH(f);
      if (value && !f->timeline_base) {
        CUDA_TRY(f->alloc(&f->timeline_base, 64 * 2 * K_COUNT));
        for (int i = 0; i < 64; ++i)
          CUDA_TRY(cudaMemsetAsync(f->timeline_base + (size_t)i * 2 * K_COUNT, 0xff, sizeof(unsigned long long) * K_COUNT, f->stream));
      }
      if (!value) f->ws.timeline = nullptr;   // the ring stays allocated; kernels stop stamping
      f->timeline_on = value != 0;
      return NSM_OK;
    }
  }
  return fail(NSM_ERR_INVALID_ARG, "unknown option %d", (int)opt);
}

nsm_status nsm_debug_set_grad(nsm_field *f, const float *d_grad, const uint8_t *d_touched) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  LEAVE_FAST_PATH(f);
  if (!d_grad) return fail(NSM_ERR_INVALID_ARG, "d_grad is NULL");
  f->wgrad_parts = 0;
  RUN(f, K_DEBUG, launch_set_grad(f->fp, d_grad, d_touched, f->stream));
  CUDA_TRY(cudaMemcpyAsync(f->fp.mlp_grad, d_grad + f->fp.n_table, sizeof(float) * f->fp.n_mlp, cudaMemcpyDeviceToDevice, f->stream));
  f->grads_dirty = true;
  return NSM_OK;
}

// nsm_render_host: the chunks' rays go in and their images come out by copies on the side stream, through two staging
// buffers each way, while the field's stream renders: chunk i + 1's rays arrive and chunk i - 1's image leaves under chunk
// i's kernels (config 5: the copies are 36 MB per view, 1.1 ms at the host link's rate, and were serialised with the
// kernels before: 6.96 -> 5.94 ms per view end to end, 137 M rays/s against 139 M with device buffers).  Unlike a training batch a frame is not read in place from pinned memory:
// with the marcher fetching 24 B per ray and the compositor storing 20 B per ray over the host link a 816 000-ray view
// took 8.85 ms.  Pageable buffers work too (their copies block the host).  Synchronises: on return the image is in the
// host buffers and the rays are free.
static nsm_status render_chunks_host(nsm_field *f, const nsm_ray_batch *b, float cut, float *rgb, float *depth, float *opacity) {
  const uint32_t M = f->cfg.max_rays;
  const uint32_t n_chunks = (b->n_rays + M - 1) / M;
  auto rays_of = [&](uint32_t i) { return (b->n_rays - i * M < M) ? b->n_rays - i * M : M; };
  auto copy_in = [&](uint32_t i) -> cudaError_t {   // side stream: rays of chunk i -> staging buffer i & 1
    const uint32_t j = i & 1u, R = rays_of(i);
    float *p = f->stage_dev + (size_t)j * 6 * M;
    cudaError_t e = cudaSuccess;
    if (i >= 2) e = cudaStreamWaitEvent(f->side, f->ev_done[j], 0);   // the chunk that used this buffer has consumed it
    if (e == cudaSuccess) e = cudaMemcpyAsync(p, b->origins + 3 * (size_t)i * M, sizeof(float) * 3 * R, cudaMemcpyHostToDevice, f->side);
    if (e == cudaSuccess) e = cudaMemcpyAsync(p + 3 * (size_t)M, b->dirs + 3 * (size_t)i * M, sizeof(float) * 3 * R, cudaMemcpyHostToDevice, f->side);
    if (e == cudaSuccess) e = cudaEventRecord(f->ev_in[j], f->side);
    return e;
  };
  // the side stream starts behind everything enqueued on the field's stream so far
  CUDA_TRY(cudaEventRecord(f->ev_main, f->stream));
  CUDA_TRY(cudaStreamWaitEvent(f->side, f->ev_main, 0));
  CUDA_TRY(copy_in(0));
  for (uint32_t i = 0; i < n_chunks; ++i) {
    const uint32_t j = i & 1u, R = rays_of(i);
    const size_t first = (size_t)i * M;
    if (i + 1 < n_chunks) CUDA_TRY(copy_in(i + 1));
    nsm_ray_batch cb = *b;
    cb.n_rays = R;
    cb.origins = f->stage_dev + (size_t)j * 6 * M;
    cb.dirs = cb.origins + 3 * (size_t)M;
    float *o = f->stage_out + (size_t)j * 5 * M;
    CUDA_TRY(cudaStreamWaitEvent(f->stream, f->ev_in[j], 0));
    if (i >= 2) CUDA_TRY(cudaStreamWaitEvent(f->stream, f->ev_outfree[j], 0));   // this output buffer's last image is out
    nsm_status st = enqueue_forward(f, &cb, R, false, 0, false);
    if (st != NSM_OK) return st;
    RUN(f, K_COMPOSITE, launch_composite_render(f->ws, R, cut, f->cfg.bg, o, o + 3 * (size_t)M, o + 4 * (size_t)M, f->stream));
    if (f->prof.on) f->prof.collect();
    CUDA_TRY(cudaEventRecord(f->ev_done[j], f->stream));
    CUDA_TRY(cudaStreamWaitEvent(f->side, f->ev_done[j], 0));
    CUDA_TRY(cudaMemcpyAsync(rgb + 3 * first, o, sizeof(float) * 3 * R, cudaMemcpyDeviceToHost, f->side));
    CUDA_TRY(cudaMemcpyAsync(depth + first, o + 3 * (size_t)M, sizeof(float) * R, cudaMemcpyDeviceToHost, f->side));
    if (opacity) CUDA_TRY(cudaMemcpyAsync(opacity + first, o + 4 * (size_t)M, sizeof(float) * R, cudaMemcpyDeviceToHost, f->side));
    CUDA_TRY(cudaEventRecord(f->ev_outfree[j], f->side));
    f->last_R = R;
    f->last_K = b->n_candidates;
    f->last_was_render = true;
  }
  CUDA_TRY(cudaStreamSynchronize(f->side));     // the last image copy is behind every kernel
  CUDA_TRY(cudaStreamSynchronize(f->stream));
  CUDA_TRY(cudaGetLastError());
  return NSM_OK;
}

static nsm_status render_chunks(nsm_field *f, const nsm_ray_batch *b, float cut, float *rgb, float *depth, float *opacity,
                                bool host) {
  nsm_status st = validate_batch(f, b, false, true);
  if (st != NSM_OK) return st;
  LEAVE_FAST_PATH(f);
  if (!rgb || !depth) return fail(NSM_ERR_INVALID_ARG, "output pointers are NULL");
  if (!(cut >= 0.f)) return fail(NSM_ERR_INVALID_ARG, "transmittance_cut must be >= 0");
  const uint32_t M = f->cfg.max_rays;
  if (host) return render_chunks_host(f, b, cut, rgb, depth, opacity);
  for (uint32_t first = 0; first < b->n_rays; first += M) {
    const uint32_t R = (b->n_rays - first < M) ? b->n_rays - first : M;
    nsm_ray_batch cb = *b;
    cb.n_rays = R;
    cb.origins = b->origins + 3 * (size_t)first;
    cb.dirs = b->dirs + 3 * (size_t)first;
    st = enqueue_forward(f, &cb, R, false, 0, false);
    if (st != NSM_OK) return st;
    RUN(f, K_COMPOSITE, launch_composite_render(f->ws, R, cut, f->cfg.bg, rgb + 3 * (size_t)first, depth + first,
                                                opacity ? opacity + first : nullptr, f->stream));
    if (f->prof.on) f->prof.collect();
    f->last_R = R;
    f->last_K = b->n_candidates;
    f->last_was_render = true;
  }
  CUDA_TRY(cudaGetLastError());
  return NSM_OK;
}

nsm_status nsm_render(nsm_field *f, const nsm_ray_batch *batch, float cut, float *d_rgb, float *d_depth, float *d_opacity) {
  return render_chunks(f, batch, cut, d_rgb, d_depth, d_opacity, false);
}

nsm_status nsm_render_host(nsm_field *f, const nsm_ray_batch *hb, float cut, float *h_rgb, float *h_depth, float *h_opacity) {
  return render_chunks(f, hb, cut, h_rgb, h_depth, h_opacity, true);
}

nsm_status nsm_debug_last_step(nsm_field *f, int item, void *d_out, uint64_t capacity_bytes, uint64_t *n_bytes_out) {
  if (!f) return fail(NSM_ERR_INVALID_ARG, "field is NULL");
  LEAVE_FAST_PATH(f);
  if (f->last_R == 0) return fail(NSM_ERR_INVALID_ARG, "no step has been run yet");
  const uint32_t R = f->last_R;
  const uint32_t *d_S = f->ws.offsets + R;
  uint32_t S = 0;
  CUDA_TRY(cudaMemcpyAsync(&f->pinned->S, d_S, sizeof(uint32_t), cudaMemcpyDeviceToHost, f->stream));
  CUDA_TRY(cudaStreamSynchronize(f->stream));
  S = f->pinned->S;
  const uint32_t L = f->lv.n_levels;
  const Workspace &ws = f->ws;
  const void *src = nullptr;
  uint64_t bytes = 0;
  switch (item) {
    case NSM_DBG_COUNTS: src = ws.counts; bytes = 4ull * R; break;
    case NSM_DBG_OFFSETS: src = ws.offsets; bytes = 4ull * (R + 1); break;
    case NSM_DBG_SAMPLE_RAY: src = ws.s_ray; bytes = 4ull * S; break;
    case NSM_DBG_SAMPLE_K: src = ws.s_k; bytes = 4ull * S; break;
    case NSM_DBG_SAMPLE_T: src = ws.s_t; bytes = 4ull * S; break;
    case NSM_DBG_SAMPLE_DELTA: src = ws.s_delta; bytes = 4ull * S; break;
    case NSM_DBG_SIGMA: src = ws.sigma; bytes = 4ull * S; break;
    case NSM_DBG_RGB: src = ws.rgb; bytes = 12ull * S; break;
    case NSM_DBG_C: src = ws.C; bytes = 12ull * R; break;
    case NSM_DBG_D_HAT: src = ws.D_hat; bytes = 4ull * R; break;
    case NSM_DBG_O: src = ws.O; bytes = 4ull * R; break;
    case NSM_DBG_DSIGMA: src = ws.dsigma; bytes = 4ull * S; break;
    case NSM_DBG_DRGB: src = ws.drgb; bytes = 12ull * S; break;
    case NSM_DBG_GRAD: bytes = 4ull * (f->fp.n_table + f->fp.n_mlp); break;
    case NSM_DBG_TOUCHED: bytes = f->fp.n_canon; break;
    case NSM_DBG_SAMPLE_X: bytes = 12ull * S; break;
    case NSM_DBG_E: bytes = 4ull * S * f->ms.LF; break;
    case NSM_DBG_SLOTS: bytes = 4ull * S * L * 8; break;
    case NSM_DBG_W: bytes = 4ull * S * L * 3; break;
    case NSM_DBG_HIDDEN_DENSITY: bytes = 4ull * S * f->ms.Hd; break;
    case NSM_DBG_HIDDEN_COLOR1: bytes = 4ull * S * f->ms.Hc; break;
    case NSM_DBG_HIDDEN_COLOR2: bytes = f->ms.n_color_layers == 2 ? 4ull * S * f->ms.Hc : 0; break;
    default: return fail(NSM_ERR_INVALID_ARG, "unknown debug item %d", item);
  }
  if (n_bytes_out) *n_bytes_out = bytes;
  if (!d_out) return NSM_OK;  // size query
  if (bytes > capacity_bytes) return fail(NSM_ERR_CAPACITY, "debug item needs %llu bytes, capacity %llu", (unsigned long long)bytes, (unsigned long long)capacity_bytes);
  if (f->last_was_render && (item == NSM_DBG_C || item == NSM_DBG_D_HAT || item == NSM_DBG_O || item >= NSM_DBG_DSIGMA))
    return fail(NSM_ERR_INVALID_ARG, "item %d is not produced by nsm_render", item);
  if (bytes == 0) return NSM_OK;
  if (src) {
    CUDA_TRY(cudaMemcpyAsync(d_out, src, bytes, cudaMemcpyDeviceToDevice, f->stream));
  } else if (item == NSM_DBG_TOUCHED) {
    RUN(f, K_DEBUG, launch_get_touched(f->fp, (uint8_t *)d_out, f->stream));
  } else if (item == NSM_DBG_GRAD) {
    RUN(f, K_DEBUG, launch_unpack_records(f->fp, 1, (float *)d_out, f->stream));
    CUDA_TRY(cudaMemcpyAsync((float *)d_out + f->fp.n_table, f->fp.mlp_grad, sizeof(float) * f->fp.n_mlp, cudaMemcpyDeviceToDevice, f->stream));
  } else if (item == NSM_DBG_SAMPLE_X) {
    RUN(f, K_DEBUG, launch_planes_to_rows(ws.s_x, ws.cap, 3, d_S, (float *)d_out, f->stream));
  } else if (item == NSM_DBG_E) {
    if (f->use_tc)
      RUN(f, K_DEBUG, launch_blob_to_rows(f->cfg.mlp_precision == NSM_MLP_BF16, ws.blob_e, f->ms.LF, f->e_two_term ? 1 : 2, d_S, (float *)d_out, f->stream));
    else
      RUN(f, K_DEBUG, launch_planes_to_rows(ws.e, ws.cap, f->ms.LF, d_S, (float *)d_out, f->stream));
  } else if (item == NSM_DBG_HIDDEN_DENSITY || item == NSM_DBG_HIDDEN_COLOR1 || item == NSM_DBG_HIDDEN_COLOR2) {
    const uint32_t n_cols = item == NSM_DBG_HIDDEN_DENSITY ? f->ms.Hd : f->ms.Hc;
    if (f->use_tc) {
      const uint8_t *blob = item == NSM_DBG_HIDDEN_DENSITY ? ws.blob_hd : (item == NSM_DBG_HIDDEN_COLOR1 ? ws.blob_h1 : ws.blob_h2);
      RUN(f, K_DEBUG, launch_blob_to_rows(f->cfg.mlp_precision == NSM_MLP_BF16, blob, n_cols, 0, d_S, (float *)d_out, f->stream));
    } else {
      const float *planes = item == NSM_DBG_HIDDEN_DENSITY ? ws.hd : (item == NSM_DBG_HIDDEN_COLOR1 ? ws.h1 : ws.h2);
      RUN(f, K_DEBUG, launch_planes_to_rows(planes, ws.cap, n_cols, d_S, (float *)d_out, f->stream));
    }
  } else if (item == NSM_DBG_SLOTS) {
    RUN(f, K_DEBUG, launch_debug_slots(f->lv, ws, d_S, (uint32_t *)d_out, nullptr, f->stream));
  } else {
    RUN(f, K_DEBUG, launch_debug_slots(f->lv, ws, d_S, nullptr, (float *)d_out, f->stream));
  }
  CUDA_TRY(cudaGetLastError());
  return NSM_OK;
}

}  // extern "C"
