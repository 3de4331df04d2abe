/*
 * nsm_oracle.h — float64 CPU ORACLE of the NeRF-SLAM mapping step (arxiv 2210.13641).
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this.  It shares no code,
 * header, table or constant generator with the CUDA path (paper_2210_13641_b200/csrc); the
 * product never links or imports it.
 *
 * What it computes (PAPER.md = /root/reference/PAPER.md, DESIGN.md "Readings" = R-numbers):
 *   S0  level tables                      DESIGN.md R11 (PAPER.md:65,167 delegate to [17])
 *   S1  candidate samples t, delta, x     PAPER.md:139,143 (Eq. 5 text), R6, R14
 *   S2  occupancy test                    R17 (paper silent)
 *   S3  compaction in (ray,k) order       BASELINE.json north_star
 *   S4  multiresolution hash encoding     PAPER.md:65,143,167 -> [17]; R11
 *   S5  density MLP, sigma = exp(g0)      PAPER.md:143; R10
 *   S6  spherical-harmonics direction enc R9
 *   S7  colour MLP, sigmoid               PAPER.md:151; R8, R10
 *   S8  transmittance + compositing       PAPER.md:141 (Eq. 5), 145 (Eq. 6), 151
 *   S9  loss L_M = L_rgb + lambda_D L_D   PAPER.md:130 (Eq. 3), 137 (Eq. 4), 149 (Eq. 7); R2, R4, R13
 *   S10-S12 backward (analytic derivative of the above, written out)
 *   S13 Adam                              R16 (paper names no optimiser)
 *   S14 occupancy from field              R17
 *   S15 render with transmittance cut     PAPER.md:163; R15
 *   F1  ray-batch sampler over keyframes   PAPER.md:157-159; DESIGN.md "F1"
 *   F2  pose gradients dL/do, d x dL/dd    PAPER.md:120,130-133 (Eq. 3 over T); DESIGN.md "F2" (row f2)
 *   F4  decayed partial occupancy refresh (strided and stochastic), nested occupancy cascades
 *                                          paper silent -> [17]; DESIGN.md "F4" R23-R25 (row f4)
 *
 * Precision: the INDEX PATH (everything that decides an integer, and the fp32 quantities
 * t, delta, x, w) is a fixed sequence of IEEE binary32 operations (compile with
 * -ffp-contract=off; fmaf where an fma is specified).  The VALUE PATH is float64.
 *
 * Pins (tests/test_oracle_*.py): level tables printed in SURVEY.md section 8, hand-computed hash
 * slots, partition of unity / affine reproduction of the trilinear interpolation, SH
 * orthonormality by quadrature and the addition theorem, compositing closed forms
 * (constant-density slab, opaque shell), loss special cases, central finite differences on
 * every parameter of a tiny field, an independent float64 torch-autograd restatement, and
 * torch.optim.Adam.  Parity unpinned: none of the paper's printed numbers (Table 1, fps)
 * concern this path; the jitter hash's statistical quality and the Adam hyper-parameters are
 * conventions fixed in DESIGN.md.
 */
#ifndef NSM_ORACLE_H
#define NSM_ORACLE_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
  float    aabb_min[3];
  float    aabb_extent;
  uint32_t n_levels, n_features, log2_table_size, n_min, n_max;
  uint32_t occ_res;
  uint32_t density_hidden, density_out;
  uint32_t geo_offset, geo_count;
  uint32_t sh_degree;
  uint32_t color_hidden, color_hidden_layers;
  float    bg[3];
  float    occ_sigma_threshold;
  float    lr, beta1, beta2, eps;
  uint32_t sparse_table_adam;
  uint64_t seed;
  uint32_t occ_cascades;   /* F4 / R23: number of nested occupancy grids (0 or 1: the single grid of S2) */
  uint32_t pose_levels;    /* F2 / R26: the pose gradients differentiate the sample position through the encoding levels
                            * l < pose_levels only (0 or >= L: all levels).  The field itself is always evaluated with all
                            * levels; only dL/dx -- hence g_o and the geometric part of tau -- is restricted.  The paper is
                            * silent (PAPER.md:120, 130-133 only name T among the variables of Eq. 3); the fine levels of a
                            * hash grid vary on a scale far below a pose error and their spatial derivative misleads a
                            * first-order pose step, so a refinement runs coarse to fine. */
} orc_config;

typedef struct {
  uint32_t     n_rays;
  const float *origins, *dirs;      /* [R,3] */
  const float *rgb;                 /* [R,3] */
  const float *depth, *depth_var;   /* [R] */
  float        t_min, t_max;
  uint32_t     n_candidates;        /* K */
} orc_batch;

typedef struct {
  double   loss, loss_rgb, loss_depth;
  uint64_t n_samples;
  uint32_t n_rays, step;
} orc_stats;

/* Optional outputs of one step; any pointer may be NULL.  Capacities are the caller's duty:
 * per-sample arrays hold R*K entries, per-ray arrays R. */
typedef struct {
  uint32_t *counts;      /* [R]    n_r */
  uint32_t *offsets;     /* [R+1]  exclusive scan */
  uint32_t *s_ray, *s_k; /* [S] */
  float    *s_t, *s_delta, *s_x; /* [S], [S], [S,3]  index-path fp32 outputs */
  uint32_t *slots;       /* [S, L, 8]  table slot of every corner (corner bit0=x, bit1=y, bit2=z) */
  float    *w;           /* [S, L, 3]  trilinear fractions */
  double   *e;           /* [S, L*F] */
  double   *sigma;       /* [S] */
  double   *rgb;         /* [S,3] */
  double   *C, *D_hat, *O; /* [R,3], [R], [R] */
  double   *dsigma, *drgb; /* [S], [S,3]  dL/dsigma_i, dL/dc_i */
  double   *grad;        /* [P]  canonical flat layout: tables then MLP matrices */
  uint8_t  *touched;     /* [n_entries]  1 if the (level,slot) entry was referenced this step */
  /* Row f2 (L_M is minimised over the poses T as well): per-ray gradients of L with respect to the
   * ray, through x = (o + t d - aabb_min) / extent into the encoding (S4's trilinear weights) and through Y(d) (S6):
   *   g_o[r]  = dL/do_r                                         (translation part of the keyframe's se(3) gradient: sum over its rays)
   *   tau[r]  = d/d(omega) L with d_r <- exp(omega^) d_r at omega = 0  (rotation part: d x dL/dd, tangential, so the value
   *             of Y off the unit sphere never enters) */
  double   *g_o;         /* [R,3] */
  double   *tau;         /* [R,3] */
  double   *dx;          /* [S,3]  dL/dx_s, x the normalised sample position */
} orc_trace;

/* S0.  res[L], offset[L+1] (in entries).  Returns 0, or -1 on a bad config. */
int orc_level_table(const orc_config *cfg, uint32_t *res, uint64_t *offset);
/* Parameter counts: table floats (= F * sum E_l) and MLP floats. */
int orc_param_count(const orc_config *cfg, uint64_t *n_table, uint64_t *n_mlp);
/* Offsets (in floats, relative to the start of the MLP block) of W_d1, W_d2, W_c1, [W_c2,] W_c3
 * and the end; out has color_hidden_layers + 4 entries. */
int orc_mlp_offsets(const orc_config *cfg, uint64_t *out);

/* S1.1: jitter hash -> 24-bit uniform in [0,1). */
uint32_t orc_hash32(uint64_t seed, uint32_t step, uint32_t r, uint32_t k);
float    orc_jitter_u(uint64_t seed, uint32_t step, uint32_t r, uint32_t k);

/* S1-S3.  jitter=0 => u == 0.5.  step = the 1-based step about to be taken.  Returns S (or -1). */
int64_t orc_march(const orc_config *cfg, const uint8_t *bits, const orc_batch *b, int jitter,
                  uint32_t step, uint32_t *counts, uint32_t *offsets, uint32_t *s_ray,
                  uint32_t *s_k, float *s_t, float *s_delta, float *s_x);

/* S4 for S points x[S,3] in [0,1)^3.  slots/w may be NULL. */
int orc_encode(const orc_config *cfg, const double *theta, uint64_t S, const float *x,
               uint32_t *slots, float *w, double *e);

/* S6: n*n real orthonormal SH of the unit vector d. */
void orc_sh(uint32_t n, const double d[3], double *Y);

/* S5+S7 for one sample: e[L*F], Y[n*n] -> sigma, rgb[3] (theta_mlp = start of the MLP block). */
int orc_field_eval(const orc_config *cfg, const double *theta_mlp, const double *e, const double *Y,
                   double *sigma, double *rgb);

/* S8 for one ray: n samples (sigma, rgb[n,3], t, delta) -> C[3], D_hat, O.  cut<=0: none (S15). */
void orc_composite(uint32_t n, const double *sigma, const double *rgb, const float *t,
                   const float *delta, const float bg[3], double cut, double *C, double *D_hat,
                   double *O);

/* S1-S13: one training step.  theta/m/v: [P] float64 state, updated in place iff apply_adam.
 * *step_inout is the number of steps already taken; incremented iff apply_adam. */
int orc_train_step(const orc_config *cfg, double *theta, double *m, double *v, uint32_t *step_inout,
                   const uint8_t *bits, const orc_batch *b, double lambda_d, int jitter,
                   int apply_adam, orc_stats *stats, orc_trace *trace);

/* S13 alone: one Adam step on n parameters given gradient g; mask (may be NULL) selects entries. */
void orc_adam(uint64_t n, double *theta, double *m, double *v, const double *g, const uint8_t *mask,
              uint32_t mask_group, uint32_t step, double lr, double beta1, double beta2, double eps);

/* S2 / F4 (R23; the paper is silent on the occupancy structure and delegates to [17]; PAPER.md:266 asks
 * for a map that follows "the region of interest"): occ_cascades = C nested occupancy grids of G^3 cells each around the
 * centre of the field cube.  In normalised coordinates cascade j (0 = finest) is the cube |x - 0.5|_max < 2^(j-C);
 * cascade C-1 is the whole cube [0,1)^3.  A point is tested against the finest cascade that contains it:
 *   q_c = x_c - 0.5 (binary32),  m = max_c |q_c|,  j = the smallest j in [0, C-1) with m < 2^(j-C), else C-1;
 *   x'_c = fma(q_c, 2^(C-1-j), 0.5) for j < C-1,  x'_c = x_c for j = C-1;   g_c = min(floor(x'_c G), G-1);
 *   bit index = j G^3 + g_x + G (g_y + G g_z).
 * C = 1 is S2's single grid, with identical arithmetic.  Returns the bit index; *cascade_out (may be NULL) gets j. */
uint64_t orc_occupancy_cell(const orc_config *cfg, const float x[3], uint32_t *cascade_out);
/* The inverse map: the normalised position of the point at offsets u in [0,1)^3 inside the cell with that bit index
 * (u = 0.5: the cell centre, which FROM_FIELD evaluates):  x'_c = (g_c + u_c) / G (an addition and a division in
 * binary32), x_c = fma(x'_c - 0.5, 2^(j-(C-1)), 0.5) for j < C-1, x_c = x'_c for j = C-1. */
void orc_occupancy_cell_point(const orc_config *cfg, uint64_t cell, const float u[3], float x_out[3]);

/* S14 FROM_FIELD: bits_out has C G^3/8 bytes (C = occ_cascades, cascade-major).  sigma_out (may be NULL) gets the
 * C G^3 densities at the cell centres. */
int orc_occupancy_from_field(const orc_config *cfg, const double *theta, uint8_t *bits_out,
                             double *sigma_out);

/* F4 (the paper is silent, [17] keeps a decayed running maximum of the density and refreshes only
 * part of the grid per update): `grid` [C G^3] (all cascades, index = the bit index) is the running density, `update_index` the number of decay updates done so far.
 *   every cell:                                   grid[c] <- decay * grid[c]
 *   cells with c mod n_sub == update_index mod n_sub:   grid[c] <- max(grid[c], sigma(centre of c))      (1/n_sub of the grid)
 *   bit[c] = grid[c] > occ_sigma_threshold
 * so n_sub consecutive updates visit every cell exactly once, and n_sub = 1, decay = 0 is S14's FROM_FIELD.  A FROM_FIELD
 * refresh sets grid[c] = sigma(c).  visited_sigma (may be NULL) gets sigma for the visited cells and -1 elsewhere. */
int orc_occupancy_decay_update(const orc_config *cfg, const double *theta, double *grid, uint32_t update_index,
                               uint32_t n_sub, double decay, uint8_t *bits_out, double *visited_sigma);

/* F4, stochastic variant ([17] refreshes a random subset of the cells per update, each at a random point inside the cell;
 * reading R25: uniform draws over all C G^3 cells, no second draw among the occupied ones):
 *   every cell:  grid[c] <- decay * grid[c]
 *   for i < n_draws:  c_i = (h(seed, update_index, i, 0xffff0003) * n_cells) >> 32           (h = orc_hash32, n_cells <= 2^31)
 *                     u_a = (h(seed, update_index, i, 0xffff0004 + a) >> 8) * 2^-24,  a = 0, 1, 2
 *                     grid[c_i] <- max(grid[c_i], sigma(orc_occupancy_cell_point(c_i, u)))
 *   bit[c] = grid[c] > occ_sigma_threshold
 * A cell drawn twice keeps the larger density, so the result does not depend on the order of the draws.
 * cells_out [n_draws], x_out [n_draws,3], sigma_out [n_draws] may be NULL. */
int orc_occupancy_stochastic_update(const orc_config *cfg, const double *theta, double *grid, uint32_t update_index,
                                    uint32_t n_draws, double decay, uint8_t *bits_out, uint64_t *cells_out, float *x_out,
                                    double *sigma_out);

/* S15. */
int orc_render(const orc_config *cfg, const double *theta, const uint8_t *bits, const orc_batch *b,
               double cut, double *rgb, double *depth, double *opacity, uint64_t *n_samples);

/* F1 ("the mapping thread ... optimizes all keyframes received", each with
 * pose, image, depth map and the depth's marginal variance): the ray-batch sampler over a keyframe store.
 * A keyframe is a pinhole view: pixel (u, v) has the camera-frame direction (xc, yc, 1), xc = (u - cx) / fx,
 * yc = (v - cy) / fy; R (row-major) rotates camera to world, t is the camera centre.  depth is the z-depth map
 * D(u, v) (what a SLAM front end estimates), depth_var its variance; rgb is [H, W, 3].
 * For ray r of draw number `draw`:
 *   kf   = (orc_hash32(seed, draw, r, 0xffff0001) * n_kf)      >> 32     uniform keyframe
 *   pix  = (orc_hash32(seed, draw, r, 0xffff0002) * (W_kf H_kf)) >> 32   uniform pixel of it, u = pix % W, v = pix / W
 *   n2   = fma(xc, xc, fma(yc, yc, 1)),  n = sqrt(n2)                     |(xc, yc, 1)|, all binary32, round to nearest
 *   d_i  = fma(R[i][0], xc / n, fma(R[i][1], yc / n, R[i][2] * (1 / n)))  unit direction in the world
 *   o    = t;  rgb copied;  depth_out = D * n  (range along the ray, reading R5);  var_out = depth_var * n2
 * Every float operation above is one IEEE binary32 operation in the order written (index-path rule), so the CUDA
 * sampler must reproduce the outputs bit for bit.  kf_out / pix_out may be NULL. */
typedef struct {
  uint32_t width, height;
  float fx, fy, cx, cy;
  float R[9];
  float t[3];
  const float *rgb, *depth, *depth_var;
} orc_keyframe;
void orc_sample_batch(const orc_keyframe *kfs, uint32_t n_kf, uint64_t seed, uint32_t draw, uint32_t n_rays,
                      uint32_t *kf_out, uint32_t *pix_out, float *origins, float *dirs, float *rgb, float *depth,
                      float *depth_var);

/* F2, the update: one Adam step on a keyframe's se(3) gradient g = (dL/dt | dL/d(omega)) (translation of the camera
 * centre; rotation about it, world frame, as delivered by the per-ray sums of orc_trace.g_o / tau):
 *   m <- b1 m + (1-b1) g,  v <- b2 v + (1-b2) g^2,  delta = lr * (m / (1-b1^k)) / (sqrt(v / (1-b2^k)) + eps)   per component,
 *   lr = lr_t for the three translation components and lr_r for the three rotation components, k = *count + 1
 *   (the number of updates this keyframe has received: a keyframe without rays in the batch is not updated at all);
 *   t <- t - delta_t;   R <- exp(-[delta_omega]x) R   (Rodrigues' formula; R rotates camera to world).
 * R [9] row-major, t [3], m [6], v [6] are updated in place. */
void orc_pose_step(double *R, double *t, double *m, double *v, uint32_t *count, const double *g, double lr_t, double lr_r,
                   double beta1, double beta2, double eps);

/* Threads the library will use (1 unless built with -fopenmp). */
int orc_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
