/*
 * nsm.h — C-ABI boundary of the B200-native NeRF-SLAM mapping step ("nsm").
 *
 * One thing is behind this header: the radiance-field training step of NeRF-SLAM's mapping
 * thread (arxiv 2210.13641; PAPER.md = the paper text) and its forward-only render, as
 * hand-written CUDA for sm_100a.  PAPER.md section 3.2 defines what is minimised:
 *
 *     L_M(T, Theta) = L_rgb + lambda_D * L_D                      (Eq. 3)
 *     L_D   = || D - D*(T,Theta) ||^2_{Sigma_D}                    (Eq. 4)
 *     d*    = sum_i T_i (1 - exp(-sigma_i delta_i)) d_i            (Eq. 5)
 *     T_i   = exp(- sum_{j<i} sigma_j delta_j)                     (Eq. 6)
 *     L_rgb = || I - I*(T,Theta) ||^2                              (Eq. 7)
 *
 * with the field (hash-grid encoding + density MLP + colour MLP) delegated to Instant-NGP
 * (PAPER.md:143, 167).  The readings of everything the paper leaves open are in DESIGN.md
 * ("Readings", R1..R22) and the step-by-step algorithm S0..S15 in DESIGN.md "Algorithm".
 *
 * Conventions
 *   - Plain C types only.  Every pointer in nsm_ray_batch and every d_* argument is a DEVICE
 *     pointer owned by the caller (e.g. torch.Tensor.data_ptr()); the *_host entry points take
 *     HOST pointers instead and perform the copies themselves.  The library never retains a
 *     caller pointer past the call.
 *   - The field owns parameters, Adam state, occupancy bits and workspace.  A field is used from one host thread
 *     at a time (different fields may be driven from different threads).
 *   - All work is enqueued on the CUDA stream given at creation (plus an internal side stream that
 *     is joined back into it before the call returns); calls return without waiting unless a host
 *     stats pointer is passed or the entry point takes host buffers.  Such a call waits until the
 *     step's statistics are final and its inputs have been consumed (end of S9, the loss) -- NOT
 *     until the backward pass and Adam (S10-S13) have run: those stay queued on the stream, and every
 *     later call is ordered behind them.
 *   - Every entry point returns an nsm_status; nsm_last_error() gives a thread-local message.
 *     Arguments are validated before anything is launched: a failed call leaves the field
 *     unchanged.  There is no CPU fallback: without a CUDA device nsm_create_field fails with
 *     NSM_ERR_CUDA.
 *   - Canonical layouts (what getters, setters and the oracle agree on):
 *       table parameter   theta[(offset_l + slot) * F + f]
 *       MLP matrices      row-major [out][in], in the order W_d1, W_d2, W_c1, (W_c2,) W_c3,
 *                         appended after the tables
 *       occupancy bit     i = j*G^3 + gx + G*(gy + G*gz) is bit (i & 7) of byte (i >> 3); j = cascade (0 with one grid)
 *       samples           ordered by (ray, candidate k)
 */
#ifndef NSM_H
#define NSM_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct nsm_field nsm_field; /* opaque */

typedef enum {
  NSM_OK = 0,
  NSM_ERR_INVALID_ARG = 1,
  NSM_ERR_OOM = 2,
  NSM_ERR_CUDA = 3,
  NSM_ERR_CAPACITY = 4,
  NSM_ERR_UNIMPLEMENTED = 5
} nsm_status;

/* Arithmetic of the two MLPs (S5, S7, S11).  FP32: CUDA-core fp32 throughout.  FP16 / BF16:
 * 16-bit operands on the tcgen05 tensor cores with fp32 accumulation. */
typedef enum { NSM_MLP_FP32 = 0, NSM_MLP_FP16 = 1, NSM_MLP_BF16 = 2 } nsm_precision;

/* S14. */
typedef enum { NSM_OCC_FULL = 0, NSM_OCC_SET = 1, NSM_OCC_FROM_FIELD = 2 } nsm_occ_mode;

typedef struct {
  uint32_t struct_size;              /* sizeof(nsm_field_config), ABI check */
  float    aabb_min[3], aabb_extent; /* cube: x = (p - aabb_min) / aabb_extent in [0,1)^3 */
  uint32_t n_levels, n_features;     /* L <= 32, F in {1,2,4,8} */
  uint32_t log2_table_size;          /* T = 2^log2_table_size entries per hashed level */
  uint32_t n_min, n_max;             /* coarsest / finest resolution (S0) */
  uint32_t occ_res;                  /* G, power of two, G^3 bits */
  uint32_t density_hidden, density_out;   /* one hidden layer; density_out <= 16 */
  uint32_t geo_offset, geo_count;    /* slice of the density output fed to the colour MLP */
  uint32_t sh_degree;                /* n -> n*n real SH coefficients, n <= 4 */
  uint32_t color_hidden, color_hidden_layers; /* 1 or 2 hidden layers */
  uint32_t mlp_precision;            /* nsm_precision */
  float    bg[3];                    /* background colour (R12) */
  float    occ_sigma_threshold;      /* FROM_FIELD: bit = sigma > threshold */
  float    lr, beta1, beta2, eps;    /* Adam (S13) */
  uint32_t sparse_table_adam;        /* 1: only table entries touched this step are updated */
  uint32_t jitter;                   /* 1: per-(ray,bin) stratified jitter in training (S1) */
  uint64_t seed;                     /* jitter stream */
  uint32_t max_rays, max_candidates; /* workspace capacity per call / per render chunk */
  uint32_t occ_cascades;             /* row f4: C nested occupancy grids of G^3 cells (0 or 1: one grid), C <= 8 */
} nsm_field_config;

typedef struct {
  uint32_t     n_rays;               /* R */
  const float *origins, *dirs;       /* [R,3] row-major fp32; dirs unit length (R5) */
  const float *rgb;                  /* [R,3] target colour in [0,1]; NULL for render */
  const float *depth;                /* [R] SLAM depth as range along the ray; <= 0: no depth term */
  const float *depth_var;            /* [R] variance Sigma_D; <= 0 or non-finite: no depth term */
  float        t_min, t_max;         /* candidate lattice: dt = (t_max - t_min) / K */
  uint32_t     n_candidates;         /* K */
} nsm_ray_batch;

typedef struct {
  double   loss, loss_rgb, loss_depth; /* L_M, L_rgb, L_D of Eqs. 3, 7, 4 (means over the batch) */
  uint64_t n_samples;                  /* S, live samples this step */
  uint32_t n_rays, step;               /* step = number of Adam steps taken so far */
} nsm_step_stats;

/* Items nsm_debug_last_step can copy out (state left by the last backward / train / render). */
typedef enum {
  NSM_DBG_COUNTS = 0,    /* u32 [R]        n_r */
  NSM_DBG_OFFSETS = 1,   /* u32 [R+1]      exclusive scan; [R] = S */
  NSM_DBG_SAMPLE_RAY = 2,/* u32 [S] */
  NSM_DBG_SAMPLE_K = 3,  /* u32 [S] */
  NSM_DBG_SAMPLE_T = 4,  /* f32 [S] */
  NSM_DBG_SAMPLE_DELTA = 5, /* f32 [S] */
  NSM_DBG_SAMPLE_X = 6,  /* f32 [S,3] */
  NSM_DBG_SLOTS = 7,     /* u32 [S,L,8]    corner bit0=x, bit1=y, bit2=z */
  NSM_DBG_W = 8,         /* f32 [S,L,3] */
  NSM_DBG_E = 9,         /* f32 [S,L*F] */
  NSM_DBG_SIGMA = 10,    /* f32 [S] */
  NSM_DBG_RGB = 11,      /* f32 [S,3] */
  NSM_DBG_C = 12,        /* f32 [R,3] */
  NSM_DBG_D_HAT = 13,    /* f32 [R] */
  NSM_DBG_O = 14,        /* f32 [R] */
  NSM_DBG_DSIGMA = 15,   /* f32 [S] */
  NSM_DBG_DRGB = 16,     /* f32 [S,3] */
  NSM_DBG_GRAD = 17,     /* f32 [P]        canonical layout; valid after nsm_backward */
  NSM_DBG_TOUCHED = 18,  /* u8  [n_entries] valid after nsm_backward */
  /* the hidden activations the backward pass takes its ReLU masks from (training steps / nsm_backward only) */
  NSM_DBG_HIDDEN_DENSITY = 19, /* f32 [S, density_hidden]  h  = ReLU(W_d1 e) */
  NSM_DBG_HIDDEN_COLOR1 = 20,  /* f32 [S, color_hidden]    h1 = ReLU(W_c1 [g slice, Y]) */
  NSM_DBG_HIDDEN_COLOR2 = 21   /* f32 [S, color_hidden]    h2 = ReLU(W_c2 h1); empty with one hidden colour layer */
} nsm_debug_item;

/* Create a field on the current CUDA device (which must be an sm_100 part: the library holds sm_100a code only); the
 * field stays on that device and every later call makes it current.  cuda_stream: a cudaStream_t (NULL = default
 * stream).  Parameters start at zero (tables) / zero (MLPs): upload theta_0 with
 * nsm_set_params.  Occupancy starts FULL.  Fails with NSM_ERR_INVALID_ARG on a bad config,
 * NSM_ERR_UNIMPLEMENTED on an unsupported shape, NSM_ERR_OOM / NSM_ERR_CUDA otherwise. */
nsm_status nsm_create_field(const nsm_field_config *cfg, void *cuda_stream, nsm_field **out);
void       nsm_destroy_field(nsm_field *f);

/* S14.  SET: d_bits = C*G^3/8 bytes (device) in the canonical layout (C = occ_cascades, 1 by default).  FULL: all ones.
 * FROM_FIELD: bit = sigma(cell centre) > occ_sigma_threshold from the current parameters. */
nsm_status nsm_update_occupancy(nsm_field *f, nsm_occ_mode mode, const uint8_t *d_bits);
/* Copy the current C*G^3/8 occupancy bytes to d_bits (device). */
nsm_status nsm_get_occupancy(nsm_field *f, uint8_t *d_bits);

/* S1-S13: one training step of L_M (Eq. 3) on a ray batch: march, encode, MLPs, composite
 * (Eqs. 5, 6), loss (Eqs. 3, 4, 7), backward, Adam.  host_stats may be NULL (no sync). */
nsm_status nsm_train_step(nsm_field *f, const nsm_ray_batch *batch, float lambda_d,
                          nsm_step_stats *host_stats);
/* The same with HOST pointers in *batch.  Pinned (page-locked) buffers are read in place by the kernels over
 * the host link -- each input is needed once per ray -- and pageable ones are staged with host-to-device
 * copies.  Always waits for the end of S9 (host_stats may still be NULL): the host buffers are free on return. */
nsm_status nsm_train_step_host(nsm_field *f, const nsm_ray_batch *host_batch, float lambda_d,
                               nsm_step_stats *host_stats);

/* Debug: with NSM_OPT_DEBUG_TIMELINE set, every hot-path kernel stamps its first block's start and last block's end
 * (%globaltimer, ns) into a ring of the last 64 training steps.  h_out (HOST) receives 64 x [2][n_kernels] words,
 * slot = step % 64, kernel classes in the order of nsm_profile_read; a start of ~0 / end of 0 means "did not run".
 * Synchronises.  Costs a few atomics per block: not for timing runs. */
nsm_status nsm_debug_timeline(nsm_field *f, uint64_t *h_out, uint64_t capacity_words, uint32_t *n_kernels);

/* ---- Row f4: decayed partial occupancy refresh (the paper is silent; [17] keeps a decayed running maximum of the
 * density and refreshes part of the grid per update).  The library keeps a running density per cell, seeded by
 * nsm_update_occupancy(NSM_OCC_FROM_FIELD).  One call:  every cell  grid <- decay * grid;  the cells
 * c = (k mod n_subsets) + j * n_subsets (k = number of decay updates since the last full refresh)
 * grid <- max(grid, sigma(cell centre));  bit = grid > occ_sigma_threshold.  n_subsets consecutive calls visit every
 * cell exactly once; (n_subsets = 1, decay = 0) equals FROM_FIELD.  Costs G^3 / n_subsets field evaluations.
 * NSM_OCC_SET and NSM_OCC_FULL discard the running grid: until the next FROM_FIELD pass has seeded it again this call
 * fails with NSM_ERR_INVALID_ARG (a partial pass would cull every cell it does not visit). */
nsm_status nsm_update_occupancy_decay(nsm_field *f, uint32_t n_subsets, float decay);
/* Stochastic variant ([17] refreshes a random subset of cells per update, each at a random point inside the cell;
 * DESIGN.md 8e reading R25): every cell grid <- decay * grid; then for draw i < n_draws of update number u (u counts these
 * calls since creation)   cell = (h(seed, u, i, 0xffff0003) * n_cells) >> 32,   offsets u_a = (h(seed, u, i, 0xffff0004 + a)
 * >> 8) * 2^-24 inside the cell (h = the jitter hash of DESIGN.md S1),   grid[cell] <- max(grid[cell], sigma(point));
 * bit = grid > occ_sigma_threshold.  A cell drawn twice keeps the larger density.  Needs a seeded grid like the call above. */
nsm_status nsm_update_occupancy_stochastic(nsm_field *f, uint32_t n_draws, float decay);
/* Nested occupancy cascades (config occ_cascades = C > 1; DESIGN.md 8e reading R23; the paper is silent, PAPER.md:266 asks
 * for a map around "the region of interest"): C grids of G^3 cells share the centre of the field cube; in normalised
 * coordinates cascade j (0 = finest) is the cube |x - 0.5|_max < 2^(j-C) and cascade C-1 the whole cube.  The marcher (S2)
 * tests a candidate against the finest cascade that contains it; SET / nsm_get_occupancy move C*G^3/8 bytes (cascade-
 * major), FROM_FIELD and the two partial refreshes evaluate the cells of all cascades. */
/* The running density grid [C*G^3] (DEVICE output), for inspection and parity. */
nsm_status nsm_get_occupancy_grid(nsm_field *f, float *d_grid);

/* ---- Row F1: keyframe store and ray-batch sampler (the mapping thread optimises over all
 * keyframes received so far, each with its pose, image, depth map and the depth's marginal variance). ----
 * A keyframe is a pinhole view: pixel (u, v) looks along the camera-frame direction ((u-cx)/fx, (v-cy)/fy, 1);
 * R (row-major) rotates camera to world, t is the camera centre in the world. */
typedef struct {
  uint32_t width, height;
  float fx, fy, cx, cy;
  float R[9];
  float t[3];
} nsm_keyframe_info;
/* Copies the image [H,W,3], the z-depth map [H,W] and its variance [H,W] (DEVICE pointers, caller-owned, free after
 * the call's work on the stream) into the library's store.  NSM_ERR_CAPACITY beyond 1024 keyframes. */
nsm_status nsm_add_keyframe(nsm_field *f, const nsm_keyframe_info *info, const float *d_rgb, const float *d_depth,
                            const float *d_depth_var, uint32_t *index_out);
nsm_status nsm_keyframe_count(const nsm_field *f, uint32_t *n_out);
/* Draw number `draw` of n_rays rays, uniform over (keyframe, pixel): for ray r
 *   kf = (h(seed, draw, r, 0xffff0001) * n_keyframes) >> 32,  pix = (h(seed, draw, r, 0xffff0002) * (W H)) >> 32
 * (h = the jitter hash of DESIGN.md S1, seed = config seed), unit world direction, origin t, colour, and the
 * z-depth / variance converted to RANGE along the ray (x |(xc,yc,1)| and x its square).  Outputs are DEVICE
 * buffers in the layout of nsm_ray_batch; bit-identical to the oracle's sampler. */
nsm_status nsm_sample_batch(nsm_field *f, uint32_t n_rays, uint32_t draw, float *d_origins, float *d_dirs, float *d_rgb,
                            float *d_depth, float *d_depth_var);
/* nsm_train_step on the batch nsm_sample_batch would draw with draw = (steps taken so far) + 1, without the batch
 * leaving the library: the sampler and the marcher of step i+1 run beside the table update of step i. */
nsm_status nsm_train_step_sampled(nsm_field *f, uint32_t n_rays, float t_min, float t_max, uint32_t n_candidates,
                                  float lambda_d, nsm_step_stats *host_stats);

/* ---- Row f2: pose gradients (L_M(T, Theta) is minimised over the poses T too). ----
 * With NSM_OPT_POSE_GRADIENTS set, after nsm_backward / a training step:
 *   d_g_o [R,3]  dL/do_r                                    (a keyframe's translation gradient is the sum over its rays)
 *   d_tau [R,3]  d/d(omega) L for d_r <- exp(omega^) d_r    (= d_r x dL/dd_r; its rotation gradient likewise)
 * through the sample positions (S4's trilinear weights) and the direction encoding (S6), with the parameters the
 * step's forward pass used.  After nsm_train_step_sampled, nsm_keyframe_pose_gradients returns those sums per
 * keyframe: d_out [n_keyframes, 6] = (translation | rotation), in the world frame, rotation about the camera centre. */
nsm_status nsm_pose_gradients(nsm_field *f, float *d_g_o, float *d_tau);
nsm_status nsm_keyframe_pose_gradients(nsm_field *f, float *d_out);
/* The update: one Adam step (the field's beta1, beta2, eps; bias correction by the number of updates the keyframe has
 * received) on the 6-vector of every keyframe that had rays in the last sampled batch, then t <- t - delta_t and
 * R <- exp(-[delta_omega]x) R in the keyframe store.  Consumes the gradients of the last nsm_train_step_sampled. */
nsm_status nsm_apply_pose_step(nsm_field *f, float lr_translation, float lr_rotation);
/* Current pose of a keyframe (HOST outputs R [9] row-major camera-to-world, t [3]); synchronises. */
nsm_status nsm_get_keyframe_pose(nsm_field *f, uint32_t index, float *h_R, float *h_t);

/* Options.
 * NSM_OPT_BATCH_READY (default 0).  With 0 the library reads a batch strictly in the order of the field's
 * stream.  With 1 the caller declares that the device buffers of every batch handed to nsm_train_step are
 * complete when the call is made (e.g. a pre-staged keyframe store) and stay unmodified until the step has
 * run: the library may then march the batch (S1-S3 read origins/dirs only) on an internal stream BESIDE the
 * previous step's table update, ahead of work queued earlier on the field's stream.  Results are identical. */
/* NSM_OPT_POSE_GRADIENTS (default 0).  With 1 every training step / nsm_backward also computes the gradients of
 * the loss with respect to the rays (row f2, below); costs two extra kernels per step and 19 floats per sample
 * of workspace. */
/* NSM_OPT_DEBUG_TIMELINE (default 0).  With 1 the kernels of every training step record the in-kernel timeline that
 * nsm_debug_timeline reads. */
/* NSM_OPT_POSE_LEVELS (default 0 = all).  Coarse-to-fine pose refinement (reading R26): the pose gradients
 * differentiate the sample positions through the encoding levels l < value only; the field itself is always evaluated
 * with all levels and the parameter gradients do not change.  May be changed between steps (a schedule). */
typedef enum { NSM_OPT_BATCH_READY = 0, NSM_OPT_POSE_GRADIENTS = 1, NSM_OPT_DEBUG_TIMELINE = 2, NSM_OPT_POSE_LEVELS = 3 } nsm_option;
nsm_status nsm_set_option(nsm_field *f, nsm_option opt, uint32_t value);

/* S1-S12 only: forward + backward, gradients left in place for nsm_debug_last_step; and S13
 * alone on the gradients in place.  nsm_train_step == nsm_backward + nsm_apply_adam. */
nsm_status nsm_backward(nsm_field *f, const nsm_ray_batch *batch, float lambda_d,
                        nsm_step_stats *host_stats);
nsm_status nsm_apply_adam(nsm_field *f);
/* Overwrite the gradient buffer (d_grad: [n_table + n_mlp], canonical layout, required) and the
 * touched set (d_touched: one byte per table entry, or NULL = every entry touched). */
nsm_status nsm_debug_set_grad(nsm_field *f, const float *d_grad, const uint8_t *d_touched);

/* S15: forward-only render, u == 0.5, a ray stops after T < transmittance_cut (0 = never).
 * d_rgb [R,3], d_depth [R], d_opacity [R] or NULL.  R may exceed max_rays (chunked). */
nsm_status nsm_render(nsm_field *f, const nsm_ray_batch *batch, float transmittance_cut,
                      float *d_rgb, float *d_depth, float *d_opacity);
/* The same with HOST pointers in *host_batch and for the three outputs (pinned or pageable).  The chunks' rays and images
 * cross the host link by copies on an internal stream, double-buffered, under the kernels of the neighbouring chunks
 * (pinned buffers; copies of pageable ones block the host).  Synchronises: on return the image is complete and the ray
 * buffers are free. */
nsm_status nsm_render_host(nsm_field *f, const nsm_ray_batch *host_batch, float transmittance_cut,
                           float *h_rgb, float *h_depth, float *h_opacity);

/* Parameter access (canonical flat layout; device pointers; any of d_theta/d_m/d_v/step may
 * be NULL). */
nsm_status nsm_param_count(const nsm_field *f, uint64_t *n_table, uint64_t *n_mlp);
nsm_status nsm_get_params(nsm_field *f, float *d_theta, float *d_m, float *d_v, uint32_t *step);
nsm_status nsm_set_params(nsm_field *f, const float *d_theta, const float *d_m, const float *d_v,
                          uint32_t step);
/* S0 tables: res[L] resolutions, offset[L+1] entry offsets (host pointers). */
nsm_status nsm_get_level_table(const nsm_field *f, uint32_t *res, uint64_t *offset);

/* Copy a debug item of the last step to d_out (device); fails with NSM_ERR_CAPACITY if
 * capacity_bytes is too small.  *n_bytes_out (may be NULL) receives the item's size. */
nsm_status nsm_debug_last_step(nsm_field *f, int item, void *d_out, uint64_t capacity_bytes,
                               uint64_t *n_bytes_out);

/* Live samples processed by all training / backward steps since creation (a device counter
 * updated by the compaction kernel; this call synchronises the stream). */
nsm_status nsm_total_samples(nsm_field *f, uint64_t *out);

/* Per-kernel timing for roofline reports: when enabled, every kernel launch is bracketed by CUDA
 * events on the field's stream and each step ends with a synchronise (so do not enable it for
 * whole-step timing).  nsm_profile_read fills up to `capacity` entries: kernel-class names
 * (static strings), summed milliseconds and launch counts since enabling; *n_out = number of
 * kernel classes. */
nsm_status nsm_profile(nsm_field *f, int enable);
nsm_status nsm_profile_read(nsm_field *f, uint32_t capacity, const char **names, double *total_ms,
                            uint64_t *launches, uint32_t *n_out);

/* ---- S1-S3 alone, allocating nothing -----------------------------------------------------------
 * For callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops): the marcher of
 * S1-S3 ("sampling 3D positions along the pixel's ray", delta_i = d_{i+1} - d_i; the occupancy
 * test of DESIGN.md S2 with the cascades of reading R23; compaction in (ray, k) order) as ONE call that takes every
 * input and output from the caller and needs no nsm_field.  It is the same kernel the training step launches; the only
 * scratch memory it needs, the chained scan's ticket counters and per-block status words, lives in a file-scope
 * `static __device__` array inside the library sized for NSM_MARCH_STATIC_MAX_RAYS rays (512 KiB + 256 B, held by
 * every GPU that loads the library until the process exits).  The call makes no cudaMalloc / cudaFree and calls no
 * allocating routine: it enqueues one memset of the scratch words it uses and one kernel on `cuda_stream`, and
 * returns without synchronising.
 *
 * cfg: the cube, the occupancy structure's shape and the jitter stream (the values an nsm_field_config carries;
 * step = the jitter stream's step index, which nsm_train_step sets to the Adam step count + 1).  rays: origins, dirs,
 * t_min, t_max, n_candidates as for nsm_train_step (DEVICE pointers; rgb / depth / depth_var are ignored).
 * d_occ_bits: the bit i = j*G^3 + gx + G*(gy + G*gz) layout of nsm_update_occupancy, ceil(C*G^3 / 8) bytes, or
 * NULL = every cell live.  out: caller-owned DEVICE arrays; capacity = samples each per-sample array can hold and
 * must be >= n_rays * n_candidates (the kernel is unchanged and does not bounds-check its writes against less).
 * On return (stream order): counts[r] = n_r, offsets = exclusive scan with offsets[n_rays] = S, and the first S
 * entries of s_ray, s_k, s_t, s_delta and of each of the three planes s_x[a * capacity + s] are the live samples
 * in (ray, k) order, bit-identical to what the field's own step computes for the same inputs.
 *
 * The current CUDA device must be the one that owns the pointers and the stream (the scratch address is looked up
 * once per device, with that device current).  Every call on a device shares the one scratch array: calls in one
 * stream are ordered and safe, calls that OVERLAP on the GPU (two streams, two host threads) race on it and give
 * wrong offsets or hang the look-back -- serialise them.  nsm_field calls use the field's own scratch and do not
 * interfere.  Errors: NSM_ERR_INVALID_ARG (NULL / malformed arguments, pointers of another device),
 * NSM_ERR_CAPACITY (n_rays > NSM_MARCH_STATIC_MAX_RAYS, n_candidates > 4096, out->capacity too small),
 * NSM_ERR_CUDA; nothing is enqueued on a failed call. */
#define NSM_MARCH_STATIC_MAX_RAYS (1u << 20)

typedef struct {
  uint32_t struct_size;              /* sizeof(nsm_march_config), ABI check */
  float    aabb_min[3], aabb_extent; /* cube: x = (p - aabb_min) / aabb_extent in [0,1)^3 */
  uint32_t occ_res;                  /* G, power of two <= 1024 */
  uint32_t occ_cascades;             /* C <= 8 (0 or 1: one grid) */
  uint32_t jitter;                   /* 0: interval midpoints; else the stratified jitter u(seed, step, ray, k) of S1 */
  uint32_t step;                     /* step index of the jitter stream */
  uint64_t seed;                     /* jitter stream */
} nsm_march_config;

typedef struct {
  uint64_t  capacity;                /* samples per per-sample array, >= n_rays * n_candidates */
  uint32_t *counts;                  /* [n_rays] */
  uint32_t *offsets;                 /* [n_rays + 1] */
  uint32_t *s_ray, *s_k;             /* [capacity] */
  float    *s_t, *s_delta;           /* [capacity] */
  float    *s_x;                     /* [3][capacity] planes */
} nsm_march_result;

nsm_status nsm_march_static(const nsm_march_config *cfg, const nsm_ray_batch *rays, const uint8_t *d_occ_bits,
                            const nsm_march_result *out, void *cuda_stream);

/* Number of this library's kernels launched by this field so far (bench.py's gpu_launches). */
uint64_t    nsm_launch_count(const nsm_field *f);
/* Which MLP path the field runs: "simt_fp32", "tcgen05_f16", "tcgen05_bf16". */
const char *nsm_mlp_path(const nsm_field *f);
const char *nsm_last_error(void);
const char *nsm_version(void);

#ifdef __cplusplus
}
#endif
#endif
