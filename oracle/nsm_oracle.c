/*
 * nsm_oracle.c — float64 CPU ORACLE (test infrastructure only; see nsm_oracle.h).
 *
 * Plain C, one loop per step of the algorithm, in the order and notation of DESIGN.md
 * "Algorithm" (S0..S15), which restates PAPER.md Eqs. 3-7 and fixes the
 * readings the paper delegates to [17].  No blocking, fusion or reordering.  Build with
 * -O2 -ffp-contract=off (the index path must execute exactly the fp32 operations written).
 * An optional -fopenmp build parallelises the per-sample / per-ray loops; the arithmetic per
 * sample is unchanged (only the order of gradient accumulation differs).
 */
#include "nsm_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAX_LEVELS 32
#define ORC_MAX_WIDTH 256

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------ S0: static tables ---- */

/* DESIGN.md S0: N_l = floor(N_min * exp(l * ln(N_max/N_min)/(L-1)) + 1e-6) in float64, with
 * N_0 = N_min and N_{L-1} = N_max forced; E_l = min((N_l+1)^3, T); dense iff (N_l+1)^3 <= T. */
int orc_level_table(const orc_config *cfg, uint32_t *res, uint64_t *offset) {
  uint32_t L = cfg->n_levels;
  if (L < 1 || L > ORC_MAX_LEVELS || cfg->n_min < 1 || cfg->n_max < cfg->n_min ||
      cfg->log2_table_size > 30)
    return -1;
  uint64_t T = 1ull << cfg->log2_table_size;
  offset[0] = 0;
  for (uint32_t l = 0; l < L; ++l) {
    uint32_t N;
    if (l == 0)
      N = cfg->n_min;
    else if (l == L - 1)
      N = cfg->n_max;
    else {
      double growth = log((double)cfg->n_max / (double)cfg->n_min) / (double)(L - 1);
      N = (uint32_t)floor((double)cfg->n_min * exp((double)l * growth) + 1e-6);
    }
    res[l] = N;
    uint64_t side = (uint64_t)N + 1;
    uint64_t dense = side * side * side;
    uint64_t E = dense <= T ? dense : T;
    offset[l + 1] = offset[l] + E;
  }
  return 0;
}

static uint32_t color_in_width(const orc_config *cfg) {
  return cfg->geo_count + cfg->sh_degree * cfg->sh_degree;
}

int orc_mlp_offsets(const orc_config *cfg, uint64_t *out) {
  uint32_t LF = cfg->n_levels * cfg->n_features;
  uint32_t Hd = cfg->density_hidden, Do = cfg->density_out, Hc = cfg->color_hidden;
  uint32_t Ci = color_in_width(cfg);
  if (cfg->color_hidden_layers < 1 || cfg->color_hidden_layers > 2) return -1;
  if (cfg->geo_offset + cfg->geo_count > Do || Do < 1) return -1;
  if (LF > ORC_MAX_WIDTH || Hd > ORC_MAX_WIDTH || Hc > ORC_MAX_WIDTH || Ci > ORC_MAX_WIDTH ||
      Do > ORC_MAX_WIDTH)
    return -1;
  uint64_t o = 0;
  uint32_t i = 0;
  out[i++] = o; o += (uint64_t)Hd * LF;          /* W_d1 [Hd][LF] */
  out[i++] = o; o += (uint64_t)Do * Hd;          /* W_d2 [Do][Hd] */
  out[i++] = o; o += (uint64_t)Hc * Ci;          /* W_c1 [Hc][Ci] */
  if (cfg->color_hidden_layers == 2) {
    out[i++] = o; o += (uint64_t)Hc * Hc;        /* W_c2 [Hc][Hc] */
  }
  out[i++] = o; o += (uint64_t)3 * Hc;           /* W_c3 [3][Hc] */
  out[i++] = o;
  return 0;
}

int orc_param_count(const orc_config *cfg, uint64_t *n_table, uint64_t *n_mlp) {
  uint32_t res[ORC_MAX_LEVELS];
  uint64_t off[ORC_MAX_LEVELS + 1], mo[8];
  if (orc_level_table(cfg, res, off) != 0) return -1;
  if (orc_mlp_offsets(cfg, mo) != 0) return -1;
  if (n_table) *n_table = off[cfg->n_levels] * cfg->n_features;
  if (n_mlp) *n_mlp = mo[cfg->color_hidden_layers + 3];
  return 0;
}

/* ------------------------------------------------------------------ S1: jitter stream ---- */

/* DESIGN.md S1.1: a pure 32-bit integer hash of (seed, step, r, k).  mix() is the two-multiply
 * xorshift finaliser with the published constants 0x7feb352d / 0x846ca68b; the four words are
 * absorbed one at a time.  Both sides implement this from the DESIGN.md text. */
static uint32_t mix32(uint32_t x) {
  x ^= x >> 16;
  x *= 0x7feb352du;
  x ^= x >> 15;
  x *= 0x846ca68bu;
  x ^= x >> 16;
  return x;
}

uint32_t orc_hash32(uint64_t seed, uint32_t step, uint32_t r, uint32_t k) {
  uint32_t h = mix32((uint32_t)(seed & 0xffffffffu) ^ 0x9e3779b9u);
  h = mix32(h ^ (uint32_t)(seed >> 32));
  h = mix32(h ^ step);
  h = mix32(h ^ r);
  h = mix32(h ^ k);
  return h;
}

float orc_jitter_u(uint64_t seed, uint32_t step, uint32_t r, uint32_t k) {
  return (float)(orc_hash32(seed, step, r, k) >> 8) * 0x1p-24f; /* exact in fp32 */
}

/* ------------------------------------------------------------------ S2 / F4: occupancy cells */

/* R23 (the paper is silent, [17] keeps a pyramid of grids): C = occ_cascades nested cubes share the
 * centre of the field cube; cascade j has half-side 2^(j-C) in normalised coordinates (j = C-1 is the whole cube) and
 * its own G^3 cells.  A point belongs to the finest cascade that contains it, by the max-norm of x - 0.5. */
static uint32_t n_cascades(const orc_config *cfg) { return cfg->occ_cascades ? cfg->occ_cascades : 1u; }

uint64_t orc_occupancy_cell(const orc_config *cfg, const float x[3], uint32_t *cascade_out) {
  const uint32_t C = n_cascades(cfg), G = cfg->occ_res;
  uint32_t j = C - 1;
  float xp[3] = {x[0], x[1], x[2]};   /* the outermost cascade (and C = 1) uses the normalised position itself */
  if (C > 1) {
    float q[3], m = 0.0f;
    for (int c = 0; c < 3; ++c) {
      q[c] = x[c] - 0.5f;                      /* one binary32 subtraction */
      float a = fabsf(q[c]);
      if (a > m) m = a;
    }
    for (j = 0; j + 1 < C; ++j)
      if (m < ldexpf(1.0f, (int)j - (int)C)) break;   /* smallest j with m < 2^(j-C); none: j = C-1 */
    if (j + 1 < C) {
      const float s = ldexpf(1.0f, (int)(C - 1 - j));  /* zoom of cascade j: 2^(C-1-j), exact */
      for (int c = 0; c < 3; ++c) xp[c] = fmaf(q[c], s, 0.5f);   /* one rounding */
    }
  }
  uint32_t g[3];
  for (int c = 0; c < 3; ++c) {
    float s = xp[c] * (float)G;
    int gi = (int)floorf(s);
    if (gi > (int)G - 1) gi = (int)G - 1;
    if (gi < 0) gi = 0;                        /* unreachable for x in [0,1); keeps the index in range for any input */
    g[c] = (uint32_t)gi;
  }
  if (cascade_out) *cascade_out = j;
  return (uint64_t)j * G * G * G + (uint64_t)g[0] + (uint64_t)G * ((uint64_t)g[1] + (uint64_t)G * g[2]);
}

/* The inverse map: the normalised position of the point at fractional offsets u in [0,1)^3 inside cell `cell`
 * (global index j G^3 + gx + G (gy + G gz)); u = 0.5 is the cell centre.  x' = (g + u) / G in the cascade's own
 * coordinates (an addition and a division in binary32), then x = fma(x' - 0.5, 2^(j-(C-1)), 0.5) for j < C-1. */
void orc_occupancy_cell_point(const orc_config *cfg, uint64_t cell, const float u[3], float x_out[3]) {
  const uint32_t C = n_cascades(cfg), G = cfg->occ_res;
  const uint64_t G3 = (uint64_t)G * G * G;
  const uint32_t j = (uint32_t)(cell / G3);
  const uint64_t loc = cell % G3;
  const uint32_t g[3] = {(uint32_t)(loc % G), (uint32_t)((loc / G) % G), (uint32_t)(loc / ((uint64_t)G * G))};
  for (int c = 0; c < 3; ++c) {
    float xp = ((float)g[c] + u[c]) / (float)G;
    if (j + 1 < C) {
      float q = xp - 0.5f;
      xp = fmaf(q, ldexpf(1.0f, (int)j - (int)(C - 1)), 0.5f);
    }
    x_out[c] = xp;
  }
}

/* ------------------------------------------------------------------ S1-S3: march ---------- */

int64_t orc_march(const orc_config *cfg, const uint8_t *bits, const orc_batch *b, int jitter,
                  uint32_t step, uint32_t *counts, uint32_t *offsets, uint32_t *s_ray,
                  uint32_t *s_k, float *s_t, float *s_delta, float *s_x) {
  const uint32_t R = b->n_rays, K = b->n_candidates;
  if (K == 0) return -1;
  /* S0 host constants, fp32 */
  const float dt = (b->t_max - b->t_min) / (float)K;
  const float inv_extent = 1.0f / cfg->aabb_extent;
  uint64_t S = 0;
  for (uint32_t r = 0; r < R; ++r) {
    if (offsets) offsets[r] = (uint32_t)S;
    uint32_t n_r = 0;
    const float *o = b->origins + 3 * (size_t)r, *d = b->dirs + 3 * (size_t)r;
    for (uint32_t k = 0; k < K; ++k) {
      /* S1.1 */
      float u = jitter ? orc_jitter_u(cfg->seed, step, r, k) : 0.5f;
      /* S1.2: t = fma((float)k + u, dt, t_min) */
      float ku = (float)k + u;
      float t = fmaf(ku, dt, b->t_min);
      /* S1.3: spacing to the next CANDIDATE (Eq. 5's delta_i = d_{i+1} - d_i) */
      float delta;
      if (k + 1 < K) {
        float u1 = jitter ? orc_jitter_u(cfg->seed, step, r, k + 1) : 0.5f;
        float a = 1.0f + u1;
        float bb = a - u;
        delta = bb * dt;
      } else {
        float a = 1.0f - u;
        delta = a * dt;
      }
      /* S1.4 */
      float x[3];
      int inside = 1;
      for (int c = 0; c < 3; ++c) {
        float p = fmaf(t, d[c], o[c]);
        float q = p - cfg->aabb_min[c];
        x[c] = q * inv_extent;
        /* S2: NaN compares false => not inside */
        if (!(x[c] >= 0.0f && x[c] < 1.0f)) inside = 0;
      }
      if (!inside) continue;
      /* S2: occupancy cell (of the finest cascade that contains x, F4 / R23) and bit */
      uint64_t cell = orc_occupancy_cell(cfg, x, NULL);
      int bit = bits ? ((bits[cell >> 3] >> (cell & 7)) & 1) : 1; /* bits==NULL: FULL */
      if (!bit) continue;
      /* S3: append in (ray, k) order */
      if (s_ray) s_ray[S] = r;
      if (s_k) s_k[S] = k;
      if (s_t) s_t[S] = t;
      if (s_delta) s_delta[S] = delta;
      if (s_x) { s_x[3 * S] = x[0]; s_x[3 * S + 1] = x[1]; s_x[3 * S + 2] = x[2]; }
      ++S;
      ++n_r;
    }
    if (counts) counts[r] = n_r;
  }
  if (offsets) offsets[R] = (uint32_t)S;
  return (int64_t)S;
}

/* ------------------------------------------------------------------ S4: encoding ---------- */

typedef struct {
  uint32_t L, F;
  uint32_t res[ORC_MAX_LEVELS];
  uint64_t off[ORC_MAX_LEVELS + 1];
  int dense[ORC_MAX_LEVELS];
  uint32_t Tmask;
} orc_levels;

static int levels_init(const orc_config *cfg, orc_levels *lv) {
  if (orc_level_table(cfg, lv->res, lv->off) != 0) return -1;
  lv->L = cfg->n_levels;
  lv->F = cfg->n_features;
  uint64_t T = 1ull << cfg->log2_table_size;
  lv->Tmask = (uint32_t)(T - 1);
  for (uint32_t l = 0; l < lv->L; ++l) {
    uint64_t side = (uint64_t)lv->res[l] + 1;
    lv->dense[l] = side * side * side <= T;
  }
  return 0;
}

/* Index path of S4 for one point and one level: 8 slots + the 3 fractions (all fp32/integer). */
static void encode_index(const orc_levels *lv, uint32_t l, const float x[3], uint32_t slot[8],
                         float w[3]) {
  const uint32_t N = lv->res[l];
  uint32_t c0[3];
  for (int c = 0; c < 3; ++c) {
    float pos = x[c] * (float)N;
    int ci = (int)floorf(pos);
    if (ci > (int)N - 1) ci = (int)N - 1;
    if (ci < 0) ci = 0;
    c0[c] = (uint32_t)ci;
    w[c] = pos - (float)ci;
  }
  for (uint32_t corner = 0; corner < 8; ++corner) {
    uint32_t vx = c0[0] + (corner & 1u), vy = c0[1] + ((corner >> 1) & 1u),
             vz = c0[2] + ((corner >> 2) & 1u);
    if (lv->dense[l]) {
      uint32_t side = N + 1;
      slot[corner] = vx + side * (vy + side * vz);
    } else {
      /* XOR-of-products spatial hash with the constants published in [17] (uint32 wrap-around) */
      slot[corner] = ((vx * 1u) ^ (vy * 2654435761u) ^ (vz * 805459861u)) & lv->Tmask;
    }
  }
}

/* Value path: trilinear weight of a corner from the fp32 fractions promoted to float64. */
static double corner_weight(uint32_t corner, const float w[3]) {
  double om = 1.0;
  for (int c = 0; c < 3; ++c) {
    double wc = (double)w[c];
    om *= ((corner >> c) & 1u) ? wc : 1.0 - wc;
  }
  return om;
}

static void encode_point(const orc_levels *lv, const double *theta, const float x[3],
                         uint32_t *slots, float *wout, double *e) {
  const uint32_t F = lv->F;
  for (uint32_t l = 0; l < lv->L; ++l) {
    uint32_t slot[8];
    float w[3];
    encode_index(lv, l, x, slot, w);
    for (uint32_t f = 0; f < F; ++f) e[l * F + f] = 0.0;
    for (uint32_t corner = 0; corner < 8; ++corner) {
      double om = corner_weight(corner, w);
      const double *entry = theta + (lv->off[l] + slot[corner]) * F;
      for (uint32_t f = 0; f < F; ++f) e[l * F + f] += om * entry[f];
    }
    if (slots) memcpy(slots + 8 * (size_t)l, slot, sizeof slot);
    if (wout) memcpy(wout + 3 * (size_t)l, w, sizeof w);
  }
}

int orc_encode(const orc_config *cfg, const double *theta, uint64_t S, const float *x,
               uint32_t *slots, float *w, double *e) {
  orc_levels lv;
  if (levels_init(cfg, &lv) != 0) return -1;
  const uint32_t L = lv.L, F = lv.F;
  for (uint64_t s = 0; s < S; ++s)
    encode_point(&lv, theta, x + 3 * s, slots ? slots + s * L * 8 : NULL, w ? w + s * L * 3 : NULL,
                 e + s * L * F);
  return 0;
}

/* ------------------------------------------------------------------ S6: SH ---------------- */

static double factorial(int n) {
  double f = 1.0;
  for (int i = 2; i <= n; ++i) f *= (double)i;
  return f;
}

/* Associated Legendre function P_l^m(z), m >= 0, WITHOUT the Condon-Shortley phase:
 * P_m^m = (2m-1)!! (1-z^2)^{m/2}; P_{m+1}^m = z (2m+1) P_m^m;
 * (l-m) P_l^m = (2l-1) z P_{l-1}^m - (l+m-1) P_{l-2}^m. */
static double legendre_P(int l, int m, double z) {
  double pmm = 1.0;
  double s = sqrt(fmax(0.0, 1.0 - z * z));
  for (int i = 1; i <= m; ++i) pmm *= (double)(2 * i - 1) * s;
  if (l == m) return pmm;
  double pm1 = z * (double)(2 * m + 1) * pmm;
  if (l == m + 1) return pm1;
  double pll = 0.0;
  for (int ll = m + 2; ll <= l; ++ll) {
    pll = ((double)(2 * ll - 1) * z * pm1 - (double)(ll + m - 1) * pmm) / (double)(ll - m);
    pmm = pm1;
    pm1 = pll;
  }
  return pll;
}

/* DESIGN.md S6: index l^2 + l + m; Y_l^0 = K P_l; Y_l^m = sqrt2 K cos(m phi) P_l^m;
 * Y_l^{-m} = sqrt2 K sin(m phi) P_l^m; K = sqrt((2l+1)/(4 pi) (l-m)!/(l+m)!). */
void orc_sh(uint32_t n, const double d[3], double *Y) {
  const double pi = 3.14159265358979323846;
  double phi = atan2(d[1], d[0]);
  double z = d[2];
  for (int l = 0; l < (int)n; ++l) {
    for (int m = 0; m <= l; ++m) {
      double K = sqrt((double)(2 * l + 1) / (4.0 * pi) * factorial(l - m) / factorial(l + m));
      double P = legendre_P(l, m, z);
      if (m == 0) {
        Y[l * l + l] = K * P;
      } else {
        Y[l * l + l + m] = sqrt(2.0) * K * cos((double)m * phi) * P;
        Y[l * l + l - m] = sqrt(2.0) * K * sin((double)m * phi) * P;
      }
    }
  }
}

/* F2: rotation derivative of the direction encoding.  For d <- exp(omega^) d the first-order change is
 * delta d = omega x d, i.e. delta z = omega_x y - omega_y x and delta phi = omega_z - z (omega_x x + omega_y y) / (x^2 + y^2)
 * (phi = atan2(y, x)).  With dY/dz from (1 - z^2) dP_l^m/dz = (l + m) P_{l-1}^m - l z P_l^m and dY/dphi from the
 * cos / sin factors, out[k] = sum_j gY[j] dY_j/d(omega_k).  Undefined at the poles (x = y = 0). */
static void sh_rotation_gradient(uint32_t n, const double d[3], const double *gY, double out[3]) {
  const double pi = 3.14159265358979323846;
  const double x = d[0], y = d[1], z = d[2], rho2 = x * x + y * y;
  const double phi = atan2(y, x);
  double gz = 0.0, gphi = 0.0; /* dL/dz, dL/dphi */
  for (int l = 0; l < (int)n; ++l) {
    for (int m = 0; m <= l; ++m) {
      double K = sqrt((double)(2 * l + 1) / (4.0 * pi) * factorial(l - m) / factorial(l + m));
      double P = legendre_P(l, m, z);
      double Pm1 = (l - 1 >= m) ? legendre_P(l - 1, m, z) : 0.0;
      double dP = ((double)(l + m) * Pm1 - (double)l * z * P) / (1.0 - z * z);
      if (m == 0) {
        gz += gY[l * l + l] * K * dP;
      } else {
        double c = cos((double)m * phi), sn = sin((double)m * phi), a = sqrt(2.0) * K;
        gz += gY[l * l + l + m] * a * c * dP + gY[l * l + l - m] * a * sn * dP;
        gphi += gY[l * l + l + m] * a * (-(double)m * sn) * P + gY[l * l + l - m] * a * ((double)m * c) * P;
      }
    }
  }
  out[0] = gz * y + gphi * (-z * x / rho2);
  out[1] = gz * (-x) + gphi * (-z * y / rho2);
  out[2] = gphi;
}

/* ------------------------------------------------------------------ S5, S7: MLPs ---------- */

typedef struct {
  uint32_t LF, Hd, Do, Ci, Hc, nc_layers, n_sh, geo_off, geo_cnt;
  uint64_t o_d1, o_d2, o_c1, o_c2, o_c3, n_mlp;
  /* per-sample activation record (doubles): */
  uint32_t a_e, a_hd, a_g, a_ci, a_h1, a_h2, a_rgb, a_sigma, a_stride;
} orc_mlp;

static int mlp_init(const orc_config *cfg, orc_mlp *M) {
  uint64_t mo[8];
  if (orc_mlp_offsets(cfg, mo) != 0) return -1;
  M->LF = cfg->n_levels * cfg->n_features;
  M->Hd = cfg->density_hidden;
  M->Do = cfg->density_out;
  M->n_sh = cfg->sh_degree * cfg->sh_degree;
  M->Ci = color_in_width(cfg);
  M->Hc = cfg->color_hidden;
  M->nc_layers = cfg->color_hidden_layers;
  M->geo_off = cfg->geo_offset;
  M->geo_cnt = cfg->geo_count;
  uint32_t i = 0;
  M->o_d1 = mo[i++];
  M->o_d2 = mo[i++];
  M->o_c1 = mo[i++];
  M->o_c2 = (M->nc_layers == 2) ? mo[i++] : 0;
  M->o_c3 = mo[i++];
  M->n_mlp = mo[i];
  uint32_t a = 0;
  M->a_e = a; a += M->LF;
  M->a_hd = a; a += M->Hd;
  M->a_g = a; a += M->Do;
  M->a_ci = a; a += M->Ci;
  M->a_h1 = a; a += M->Hc;
  M->a_h2 = a; a += (M->nc_layers == 2) ? M->Hc : 0;
  M->a_rgb = a; a += 3;
  M->a_sigma = a; a += 1;
  M->a_stride = a;
  return 0;
}

/* y[n_out] = W[n_out][n_in] x, optionally ReLU.  No biases (R10). */
static void linear(const double *W, uint32_t n_out, uint32_t n_in, const double *x, double *y,
                   int relu) {
  for (uint32_t o = 0; o < n_out; ++o) {
    double acc = 0.0;
    for (uint32_t i = 0; i < n_in; ++i) acc += W[(size_t)o * n_in + i] * x[i];
    y[o] = (relu && acc < 0.0) ? 0.0 : acc;
  }
}

/* Forward of S5 + S7 on one activation record whose e[] is filled; Y = SH of the ray. */
static void mlp_forward(const orc_mlp *M, const double *Wm, const double *Y, double *act) {
  double *e = act + M->a_e, *hd = act + M->a_hd, *g = act + M->a_g, *ci = act + M->a_ci;
  double *h1 = act + M->a_h1, *h2 = act + M->a_h2, *rgb = act + M->a_rgb;
  /* S5 */
  linear(Wm + M->o_d1, M->Hd, M->LF, e, hd, 1);
  linear(Wm + M->o_d2, M->Do, M->Hd, hd, g, 0);
  double g0 = g[0];
  double g0c = g0 < -15.0 ? -15.0 : (g0 > 15.0 ? 15.0 : g0);
  act[M->a_sigma] = exp(g0c);
  /* S7 */
  for (uint32_t i = 0; i < M->geo_cnt; ++i) ci[i] = g[M->geo_off + i];
  for (uint32_t i = 0; i < M->n_sh; ++i) ci[M->geo_cnt + i] = Y[i];
  linear(Wm + M->o_c1, M->Hc, M->Ci, ci, h1, 1);
  const double *last = h1;
  if (M->nc_layers == 2) {
    linear(Wm + M->o_c2, M->Hc, M->Hc, h1, h2, 1);
    last = h2;
  }
  double pre[3];
  linear(Wm + M->o_c3, 3, M->Hc, last, pre, 0);
  for (int c = 0; c < 3; ++c) rgb[c] = 1.0 / (1.0 + exp(-pre[c]));
}

int orc_field_eval(const orc_config *cfg, const double *theta_mlp, const double *e, const double *Y,
                   double *sigma, double *rgb) {
  orc_mlp M;
  if (mlp_init(cfg, &M) != 0) return -1;
  double act[8 * ORC_MAX_WIDTH];
  memcpy(act + M.a_e, e, sizeof(double) * M.LF);
  mlp_forward(&M, theta_mlp, Y, act);
  *sigma = act[M.a_sigma];
  for (int c = 0; c < 3; ++c) rgb[c] = act[M.a_rgb + c];
  return 0;
}

/* y^T W: dx[n_in] = sum_o W[o][i] dy[o];  dW[o][i] += dy[o] x[i]. */
static void linear_backward(const double *W, double *dW, uint32_t n_out, uint32_t n_in,
                            const double *x, const double *dy, double *dx) {
  if (dx)
    for (uint32_t i = 0; i < n_in; ++i) dx[i] = 0.0;
  for (uint32_t o = 0; o < n_out; ++o) {
    double d = dy[o];
    for (uint32_t i = 0; i < n_in; ++i) {
      dW[(size_t)o * n_in + i] += d * x[i];
      if (dx) dx[i] += W[(size_t)o * n_in + i] * d;
    }
  }
}

/* S11 for one sample: given dL/dsigma and dL/drgb, accumulate dW (MLP block) and return dL/de. */
static void mlp_backward(const orc_mlp *M, const double *Wm, double *dWm, const double *act,
                         double dsigma, const double drgb[3], double *de, double *dci_out) {
  const double *e = act + M->a_e, *hd = act + M->a_hd, *g = act + M->a_g, *ci = act + M->a_ci;
  const double *h1 = act + M->a_h1, *h2 = act + M->a_h2, *rgb = act + M->a_rgb;
  double dpre[3], dh2[ORC_MAX_WIDTH], dh1[ORC_MAX_WIDTH], dci[ORC_MAX_WIDTH], dg[ORC_MAX_WIDTH],
      dhd[ORC_MAX_WIDTH];
  /* sigmoid */
  for (int c = 0; c < 3; ++c) dpre[c] = drgb[c] * rgb[c] * (1.0 - rgb[c]);
  if (M->nc_layers == 2) {
    linear_backward(Wm + M->o_c3, dWm + M->o_c3, 3, M->Hc, h2, dpre, dh2);
    for (uint32_t i = 0; i < M->Hc; ++i)
      if (!(h2[i] > 0.0)) dh2[i] = 0.0; /* ReLU mask */
    linear_backward(Wm + M->o_c2, dWm + M->o_c2, M->Hc, M->Hc, h1, dh2, dh1);
  } else {
    linear_backward(Wm + M->o_c3, dWm + M->o_c3, 3, M->Hc, h1, dpre, dh1);
  }
  for (uint32_t i = 0; i < M->Hc; ++i)
    if (!(h1[i] > 0.0)) dh1[i] = 0.0;
  linear_backward(Wm + M->o_c1, dWm + M->o_c1, M->Hc, M->Ci, ci, dh1, dci);
  if (dci_out)
    for (uint32_t i = 0; i < M->Ci; ++i) dci_out[i] = dci[i]; /* dL/d(colour input): geo slice, then the SH terms */
  /* density outputs: geo slice from the colour net, g0 from sigma (0 if clamped) */
  for (uint32_t i = 0; i < M->Do; ++i) dg[i] = 0.0;
  for (uint32_t i = 0; i < M->geo_cnt; ++i) dg[M->geo_off + i] += dci[i];
  if (g[0] > -15.0 && g[0] < 15.0) dg[0] += dsigma * act[M->a_sigma];
  linear_backward(Wm + M->o_d2, dWm + M->o_d2, M->Do, M->Hd, hd, dg, dhd);
  for (uint32_t i = 0; i < M->Hd; ++i)
    if (!(hd[i] > 0.0)) dhd[i] = 0.0;
  linear_backward(Wm + M->o_d1, dWm + M->o_d1, M->Hd, M->LF, e, dhd, de);
}

/* ------------------------------------------------------------------ S8: compositing ------- */

/* Eqs. 5, 6 and the colour sum, in sample order.
 * Tr[] (optional, n+1 entries) receives T_1..T_{n+1}; wgt[] (optional) the weights w_i.
 * Returns the number of samples consumed (S15: stops after T_{i+1} < cut). */
static uint32_t composite_ray(uint32_t n, const double *sigma, size_t sigma_stride,
                              const double *rgb, size_t rgb_stride, const float *t,
                              const float *delta, const float bg[3], double cut, double *C,
                              double *D_hat, double *O, double *Tr, double *wgt) {
  double T = 1.0, Cacc[3] = {0, 0, 0}, Dacc = 0.0, Oacc = 0.0;
  uint32_t used = 0;
  if (Tr) Tr[0] = 1.0;
  for (uint32_t i = 0; i < n; ++i) {
    double a = sigma[i * sigma_stride] * (double)delta[i];
    double alpha = -expm1(-a);       /* 1 - exp(-sigma_i delta_i) */
    double w = T * alpha;            /* T_i alpha_i */
    for (int c = 0; c < 3; ++c) Cacc[c] += w * rgb[i * rgb_stride + c];
    Dacc += w * (double)t[i];
    Oacc += w;
    T = T * exp(-a);                 /* T_{i+1} = exp(-sum_{j<=i} sigma_j delta_j), Eq. 6 */
    if (Tr) Tr[i + 1] = T;
    if (wgt) wgt[i] = w;
    used = i + 1;
    if (cut > 0.0 && T < cut) break;
  }
  for (int c = 0; c < 3; ++c) C[c] = Cacc[c] + T * (double)bg[c];
  *D_hat = Dacc;
  *O = Oacc;
  return used;
}

void orc_composite(uint32_t n, const double *sigma, const double *rgb, const float *t,
                   const float *delta, const float bg[3], double cut, double *C, double *D_hat,
                   double *O) {
  composite_ray(n, sigma, 1, rgb, 3, t, delta, bg, cut, C, D_hat, O, NULL, NULL);
}

/* ------------------------------------------------------------------ S13: Adam ------------- */

void orc_adam(uint64_t n, double *theta, double *m, double *v, const double *g, const uint8_t *mask,
              uint32_t mask_group, uint32_t step, double lr, double beta1, double beta2,
              double eps) {
  double bc1 = 1.0 - pow(beta1, (double)step);
  double bc2 = 1.0 - pow(beta2, (double)step);
  for (uint64_t i = 0; i < n; ++i) {
    if (mask && !mask[i / mask_group]) continue;
    m[i] = beta1 * m[i] + (1.0 - beta1) * g[i];
    v[i] = beta2 * v[i] + (1.0 - beta2) * g[i] * g[i];
    double mhat = m[i] / bc1;
    double vhat = v[i] / bc2;
    theta[i] = theta[i] - lr * mhat / (sqrt(vhat) + eps);
  }
}

/* ------------------------------------------------------------------ the training step ----- */

int orc_train_step(const orc_config *cfg, double *theta, double *m, double *v, uint32_t *step_inout,
                   const uint8_t *bits, const orc_batch *b, double lambda_d, int jitter,
                   int apply_adam, orc_stats *stats, orc_trace *trace) {
  orc_levels lv;
  orc_mlp M;
  if (levels_init(cfg, &lv) != 0 || mlp_init(cfg, &M) != 0) return -1;
  const uint32_t R = b->n_rays, K = b->n_candidates, L = lv.L, F = lv.F;
  const uint64_t n_entries = lv.off[L];
  const uint64_t n_table = n_entries * F;
  const uint64_t P = n_table + M.n_mlp;
  const uint64_t cap = (uint64_t)R * K;
  const uint32_t step = *step_inout + 1; /* the 1-based step about to be taken */
  orc_trace none;
  memset(&none, 0, sizeof none);
  if (!trace) trace = &none;
  int rc = -2;

  uint32_t *counts = malloc(sizeof(uint32_t) * (R + 1)), *offsets = malloc(sizeof(uint32_t) * (R + 1));
  uint32_t *s_ray = malloc(sizeof(uint32_t) * (cap + 1)), *s_k = malloc(sizeof(uint32_t) * (cap + 1));
  float *s_t = malloc(sizeof(float) * (cap + 1)), *s_delta = malloc(sizeof(float) * (cap + 1));
  float *s_x = malloc(sizeof(float) * 3 * (cap + 1));
  double *act = NULL, *Tr = NULL, *wgt = NULL, *dsigma = NULL, *drgb = NULL, *grad = NULL;
  double *C = malloc(sizeof(double) * 3 * (R + 1)), *Dh = malloc(sizeof(double) * (R + 1)),
         *Op = malloc(sizeof(double) * (R + 1)), *Ysh = malloc(sizeof(double) * (size_t)(M.n_sh + 1) * (R + 1));
  uint8_t *touched = NULL;
  uint32_t *slots = NULL;
  float *wfr = NULL;
  if (!counts || !offsets || !s_ray || !s_k || !s_t || !s_delta || !s_x || !C || !Dh || !Op || !Ysh)
    goto done;

  /* S1-S3 */
  int64_t S64 = orc_march(cfg, bits, b, jitter, step, counts, offsets, s_ray, s_k, s_t, s_delta, s_x);
  if (S64 < 0) { rc = -1; goto done; }
  const uint64_t S = (uint64_t)S64;

  act = malloc(sizeof(double) * (size_t)M.a_stride * (S + 1));
  slots = malloc(sizeof(uint32_t) * (size_t)L * 8 * (S + 1));
  wfr = malloc(sizeof(float) * (size_t)L * 3 * (S + 1));
  Tr = malloc(sizeof(double) * (S + R + 1));
  wgt = malloc(sizeof(double) * (S + 1));
  dsigma = malloc(sizeof(double) * (S + 1));
  drgb = malloc(sizeof(double) * 3 * (S + 1));
  grad = calloc(P + 1, sizeof(double));
  touched = calloc(n_entries + 1, 1);
  if (!act || !slots || !wfr || !Tr || !wgt || !dsigma || !drgb || !grad || !touched) goto done;

  /* S6 per ray (broadcast to its samples) */
  for (uint32_t r = 0; r < R; ++r) {
    double d[3] = {(double)b->dirs[3 * (size_t)r], (double)b->dirs[3 * (size_t)r + 1],
                   (double)b->dirs[3 * (size_t)r + 2]};
    orc_sh(cfg->sh_degree, d, Ysh + (size_t)M.n_sh * r);
  }

  /* S4, S5, S7 per sample */
  const double *Wm = theta + n_table;
#pragma omp parallel for schedule(static)
  for (int64_t s = 0; s < (int64_t)S; ++s) {
    double *a = act + (size_t)M.a_stride * s;
    encode_point(&lv, theta, s_x + 3 * s, slots + (size_t)s * L * 8, wfr + (size_t)s * L * 3,
                 a + M.a_e);
    mlp_forward(&M, Wm, Ysh + (size_t)M.n_sh * s_ray[s], a);
  }

  /* S8 per ray, S9 */
  double Lrgb = 0.0, Ld = 0.0;
  for (uint32_t r = 0; r < R; ++r) {
    uint32_t o = offsets[r], n = counts[r];
    composite_ray(n, act + (size_t)M.a_stride * o + M.a_sigma, M.a_stride,
                  act + (size_t)M.a_stride * o + M.a_rgb, M.a_stride, s_t + o, s_delta + o, cfg->bg,
                  0.0, C + 3 * (size_t)r, Dh + r, Op + r, Tr + o + r, wgt + o);
    for (int c = 0; c < 3; ++c) {
      double d = C[3 * (size_t)r + c] - (double)b->rgb[3 * (size_t)r + c];
      Lrgb += d * d;                                     /* Eq. 7 */
    }
    double Dsl = (double)b->depth[r], var = (double)b->depth_var[r];
    int mask = (Dsl > 0.0) && (var > 0.0) && isfinite(var); /* R13 */
    if (mask) {
      double d = Dh[r] - Dsl;
      Ld += d * d / var;                                 /* Eq. 4, Sigma_D a per-pixel variance */
    }
  }
  Lrgb /= (double)R;
  Ld /= (double)R;
  double Ltot = Lrgb + lambda_d * Ld;                    /* Eq. 3 */

  /* S10 per ray: dL/dc_i, dL/dsigma_i */
  for (uint32_t r = 0; r < R; ++r) {
    uint32_t o = offsets[r], n = counts[r];
    double gC[3], gD = 0.0;
    for (int c = 0; c < 3; ++c)
      gC[c] = 2.0 / (double)R * (C[3 * (size_t)r + c] - (double)b->rgb[3 * (size_t)r + c]);
    double Dsl = (double)b->depth[r], var = (double)b->depth_var[r];
    if ((Dsl > 0.0) && (var > 0.0) && isfinite(var))
      gD = 2.0 * lambda_d / (double)R * (Dh[r] - Dsl) / var;
    const double *TrR = Tr + o + r; /* T_1..T_{n+1} */
    double T_end = TrR[n];
    double bgdot = 0.0;
    for (int c = 0; c < 3; ++c) bgdot += (double)cfg->bg[c] * gC[c];
    double suffix = 0.0; /* sum_{j>i} w_j q_j */
    for (int64_t i = (int64_t)n - 1; i >= 0; --i) {
      const double *a = act + (size_t)M.a_stride * (o + i);
      double q = (double)s_t[o + i] * gD;
      for (int c = 0; c < 3; ++c) q += a[M.a_rgb + c] * gC[c];
      for (int c = 0; c < 3; ++c) drgb[3 * (size_t)(o + i) + c] = wgt[o + i] * gC[c];
      dsigma[o + i] = (double)s_delta[o + i] * (TrR[i + 1] * q - suffix - T_end * bgdot);
      suffix += wgt[o + i] * q;
    }
  }

  /* S11, S12 per sample */
  /* F2 accumulators: dL/do, sum_s t_s dL/dp_s, sum_s dL/dY_s per ray */
  const int want_pose = trace->g_o || trace->tau || trace->dx;
  double *pose_o = NULL, *pose_d = NULL, *pose_Y = NULL;
  if (want_pose) {
    pose_o = calloc(3 * (size_t)R + 1, sizeof(double));
    pose_d = calloc(3 * (size_t)R + 1, sizeof(double));
    pose_Y = calloc((size_t)(M.n_sh + 1) * R + 1, sizeof(double));
    if (!pose_o || !pose_d || !pose_Y) { free(pose_o); free(pose_d); free(pose_Y); goto done; }
  }
  {
    double *dWm = grad + n_table;
#pragma omp parallel
    {
      double *dW_local = calloc(M.n_mlp + 1, sizeof(double));
      double de[ORC_MAX_WIDTH], dci[ORC_MAX_WIDTH];
#pragma omp for schedule(static)
      for (int64_t s = 0; s < (int64_t)S; ++s) {
        const double *a = act + (size_t)M.a_stride * s;
        mlp_backward(&M, Wm, dW_local, a, dsigma[s], drgb + 3 * s, de, dci);
        if (want_pose) {
          /* dL/dx_c = sum_l N_l sum_corners (d omega / d w_c) (theta[corner] . dL/de_l): w_c = x_c N_l - c0_c */
          double dxs[3] = {0.0, 0.0, 0.0};
          /* R26 (coarse-to-fine pose gradients): only the levels l < pose_levels carry the position's derivative */
          const uint32_t L_pose = (cfg->pose_levels == 0 || cfg->pose_levels > L) ? L : cfg->pose_levels;
          for (uint32_t l = 0; l < L_pose; ++l) {
            const uint32_t *slot = slots + ((size_t)s * L + l) * 8;
            const float *w = wfr + ((size_t)s * L + l) * 3;
            for (uint32_t corner = 0; corner < 8; ++corner) {
              const double *entry = theta + (lv.off[l] + slot[corner]) * F;
              double dot = 0.0;
              for (uint32_t f = 0; f < F; ++f) dot += entry[f] * de[l * F + f];
              for (int c = 0; c < 3; ++c) {
                double dom = ((corner >> c) & 1u) ? 1.0 : -1.0;
                for (int c2 = 0; c2 < 3; ++c2)
                  if (c2 != c) dom *= ((corner >> c2) & 1u) ? (double)w[c2] : 1.0 - (double)w[c2];
                dxs[c] += (double)lv.res[l] * dom * dot;
              }
            }
          }
          if (trace->dx) for (int c = 0; c < 3; ++c) trace->dx[3 * (size_t)s + c] = dxs[c];
          const uint32_t r = s_ray[s];
          const double inv_extent = (double)(1.0f / cfg->aabb_extent);
          for (int c = 0; c < 3; ++c) {
            const double dp = dxs[c] * inv_extent;
#pragma omp atomic
            pose_o[3 * (size_t)r + c] += dp;
#pragma omp atomic
            pose_d[3 * (size_t)r + c] += (double)s_t[s] * dp;
          }
          for (uint32_t j = 0; j < M.n_sh; ++j) {
#pragma omp atomic
            pose_Y[(size_t)M.n_sh * r + j] += dci[M.geo_cnt + j];
          }
        }
        for (uint32_t l = 0; l < L; ++l) {
          const uint32_t *slot = slots + ((size_t)s * L + l) * 8;
          const float *w = wfr + ((size_t)s * L + l) * 3;
          for (uint32_t corner = 0; corner < 8; ++corner) {
            double om = corner_weight(corner, w);
            uint64_t entry = lv.off[l] + slot[corner];
            for (uint32_t f = 0; f < F; ++f) {
              double contrib = om * de[l * F + f];
#pragma omp atomic
              grad[entry * F + f] += contrib;
            }
            touched[entry] = 1; /* structural touched set U (R16) */
          }
        }
      }
#pragma omp critical
      for (uint64_t i = 0; i < M.n_mlp; ++i) dWm[i] += dW_local[i];
      free(dW_local);
    }
  }

  if (want_pose) {
    for (uint32_t r = 0; r < R; ++r) {
      const double d[3] = {(double)b->dirs[3 * (size_t)r], (double)b->dirs[3 * (size_t)r + 1], (double)b->dirs[3 * (size_t)r + 2]};
      const double *gd = pose_d + 3 * (size_t)r;
      double rot[3];
      sh_rotation_gradient(cfg->sh_degree, d, pose_Y + (size_t)M.n_sh * r, rot);
      if (trace->g_o) for (int c = 0; c < 3; ++c) trace->g_o[3 * (size_t)r + c] = pose_o[3 * (size_t)r + c];
      if (trace->tau) {
        trace->tau[3 * (size_t)r + 0] = d[1] * gd[2] - d[2] * gd[1] + rot[0];
        trace->tau[3 * (size_t)r + 1] = d[2] * gd[0] - d[0] * gd[2] + rot[1];
        trace->tau[3 * (size_t)r + 2] = d[0] * gd[1] - d[1] * gd[0] + rot[2];
      }
    }
    free(pose_o); free(pose_d); free(pose_Y);
  }

  /* trace copies before the update */
  if (trace->counts) memcpy(trace->counts, counts, sizeof(uint32_t) * R);
  if (trace->offsets) memcpy(trace->offsets, offsets, sizeof(uint32_t) * (R + 1));
  if (trace->s_ray) memcpy(trace->s_ray, s_ray, sizeof(uint32_t) * S);
  if (trace->s_k) memcpy(trace->s_k, s_k, sizeof(uint32_t) * S);
  if (trace->s_t) memcpy(trace->s_t, s_t, sizeof(float) * S);
  if (trace->s_delta) memcpy(trace->s_delta, s_delta, sizeof(float) * S);
  if (trace->s_x) memcpy(trace->s_x, s_x, sizeof(float) * 3 * S);
  if (trace->slots) memcpy(trace->slots, slots, sizeof(uint32_t) * (size_t)L * 8 * S);
  if (trace->w) memcpy(trace->w, wfr, sizeof(float) * (size_t)L * 3 * S);
  for (uint64_t s = 0; s < S; ++s) {
    const double *a = act + (size_t)M.a_stride * s;
    if (trace->e) memcpy(trace->e + s * M.LF, a + M.a_e, sizeof(double) * M.LF);
    if (trace->sigma) trace->sigma[s] = a[M.a_sigma];
    if (trace->rgb) memcpy(trace->rgb + 3 * s, a + M.a_rgb, sizeof(double) * 3);
  }
  if (trace->C) memcpy(trace->C, C, sizeof(double) * 3 * R);
  if (trace->D_hat) memcpy(trace->D_hat, Dh, sizeof(double) * R);
  if (trace->O) memcpy(trace->O, Op, sizeof(double) * R);
  if (trace->dsigma) memcpy(trace->dsigma, dsigma, sizeof(double) * S);
  if (trace->drgb) memcpy(trace->drgb, drgb, sizeof(double) * 3 * S);
  if (trace->grad) memcpy(trace->grad, grad, sizeof(double) * P);
  if (trace->touched) memcpy(trace->touched, touched, n_entries);

  /* S13 */
  if (apply_adam) {
    orc_adam(n_table, theta, m, v, grad, cfg->sparse_table_adam ? touched : NULL, F, step,
             (double)cfg->lr, (double)cfg->beta1, (double)cfg->beta2, (double)cfg->eps);
    orc_adam(M.n_mlp, theta + n_table, m + n_table, v + n_table, grad + n_table, NULL, 1, step,
             (double)cfg->lr, (double)cfg->beta1, (double)cfg->beta2, (double)cfg->eps);
    *step_inout = step;
  }
  if (stats) {
    stats->loss = Ltot;
    stats->loss_rgb = Lrgb;
    stats->loss_depth = Ld;
    stats->n_samples = S;
    stats->n_rays = R;
    stats->step = apply_adam ? step : *step_inout;
  }
  rc = 0;
done:
  free(counts); free(offsets); free(s_ray); free(s_k); free(s_t); free(s_delta); free(s_x);
  free(act); free(slots); free(wfr); free(Tr); free(wgt); free(dsigma); free(drgb); free(grad);
  free(touched); free(C); free(Dh); free(Op); free(Ysh);
  return rc;
}

/* ------------------------------------------------------------------ S14: occupancy -------- */

/* sigma (S4 + S5 + exp) at the normalised position x */
static double point_sigma(const orc_levels *lv, const orc_mlp *M, const double *theta, const float x[3]) {
  const double *Wm = theta + lv->off[lv->L] * lv->F;
  double e[ORC_MAX_WIDTH], hd[ORC_MAX_WIDTH];
  encode_point(lv, theta, x, NULL, NULL, e);
  linear(Wm + M->o_d1, M->Hd, M->LF, e, hd, 1);
  double g0 = 0.0;
  for (uint32_t i = 0; i < M->Hd; ++i) g0 += Wm[M->o_d2 + i] * hd[i]; /* row 0 of W_d2 */
  double g0c = g0 < -15.0 ? -15.0 : (g0 > 15.0 ? 15.0 : g0);
  return exp(g0c);
}

/* sigma at the centre of occupancy cell `cell` (global index over the cascades); the centre of a cell of a
 * power-of-two grid is exact in fp32 */
static double cell_sigma(const orc_config *cfg, const orc_levels *lv, const orc_mlp *M, const double *theta, uint64_t cell) {
  const float half[3] = {0.5f, 0.5f, 0.5f};
  float x[3];
  orc_occupancy_cell_point(cfg, cell, half, x);
  return point_sigma(lv, M, theta, x);
}

int orc_occupancy_from_field(const orc_config *cfg, const double *theta, uint8_t *bits_out,
                             double *sigma_out) {
  orc_levels lv;
  orc_mlp M;
  if (levels_init(cfg, &lv) != 0 || mlp_init(cfg, &M) != 0) return -1;
  const uint32_t G = cfg->occ_res;
  const uint64_t cells = (uint64_t)n_cascades(cfg) * G * G * G;
  memset(bits_out, 0, (cells + 7) / 8);
  int64_t w;
  /* one 8-cell byte of the bitfield per iteration, so no two threads write the same byte */
#pragma omp parallel for schedule(static)
  for (w = 0; w < (int64_t)((cells + 7) / 8); ++w)
    for (uint64_t cell = 8 * (uint64_t)w; cell < 8 * (uint64_t)w + 8 && cell < cells; ++cell) {
      const double sigma = cell_sigma(cfg, &lv, &M, theta, cell);
      if (sigma_out) sigma_out[cell] = sigma;
      if (sigma > (double)cfg->occ_sigma_threshold) bits_out[cell >> 3] |= (uint8_t)(1u << (cell & 7));
    }
  return 0;
}

/* F4: decayed running maximum with a strided partial refresh (header comment of orc_occupancy_decay_update). */
int orc_occupancy_decay_update(const orc_config *cfg, const double *theta, double *grid, uint32_t update_index,
                               uint32_t n_sub, double decay, uint8_t *bits_out, double *visited_sigma) {
  orc_levels lv;
  orc_mlp M;
  if (levels_init(cfg, &lv) != 0 || mlp_init(cfg, &M) != 0 || n_sub == 0) return -1;
  const uint64_t cells = (uint64_t)n_cascades(cfg) * cfg->occ_res * cfg->occ_res * cfg->occ_res;
  memset(bits_out, 0, (cells + 7) / 8);
  for (uint64_t c = 0; c < cells; ++c) {
    grid[c] *= decay;
    if (visited_sigma) visited_sigma[c] = -1.0;
    if (c % n_sub == update_index % n_sub) {
      const double s = cell_sigma(cfg, &lv, &M, theta, c);
      if (s > grid[c]) grid[c] = s;
      if (visited_sigma) visited_sigma[c] = s;
    }
    if (grid[c] > (double)cfg->occ_sigma_threshold) bits_out[c >> 3] |= (uint8_t)(1u << (c & 7));
  }
  return 0;
}

/* F4, stochastic refresh (header comment of orc_occupancy_stochastic_update). */
int orc_occupancy_stochastic_update(const orc_config *cfg, const double *theta, double *grid, uint32_t update_index,
                                    uint32_t n_draws, double decay, uint8_t *bits_out, uint64_t *cells_out, float *x_out,
                                    double *sigma_out) {
  orc_levels lv;
  orc_mlp M;
  if (levels_init(cfg, &lv) != 0 || mlp_init(cfg, &M) != 0) return -1;
  const uint64_t cells = (uint64_t)n_cascades(cfg) * cfg->occ_res * cfg->occ_res * cfg->occ_res;
  if (cells > (1ull << 31)) return -1;            /* (hash * cells) >> 32 in 64 bits */
  for (uint64_t c = 0; c < cells; ++c) grid[c] *= decay;
  for (uint32_t i = 0; i < n_draws; ++i) {
    const uint64_t cell = ((uint64_t)orc_hash32(cfg->seed, update_index, i, 0xffff0003u) * cells) >> 32;
    float u[3], x[3];
    for (uint32_t a = 0; a < 3; ++a)
      u[a] = (float)(orc_hash32(cfg->seed, update_index, i, 0xffff0004u + a) >> 8) * 0x1p-24f;   /* exact */
    orc_occupancy_cell_point(cfg, cell, u, x);
    const double s = point_sigma(&lv, &M, theta, x);
    if (s > grid[cell]) grid[cell] = s;           /* a cell drawn twice keeps the larger density: order-free */
    if (cells_out) cells_out[i] = cell;
    if (x_out) { x_out[3 * i] = x[0]; x_out[3 * i + 1] = x[1]; x_out[3 * i + 2] = x[2]; }
    if (sigma_out) sigma_out[i] = s;
  }
  memset(bits_out, 0, (cells + 7) / 8);
  for (uint64_t c = 0; c < cells; ++c)
    if (grid[c] > (double)cfg->occ_sigma_threshold) bits_out[c >> 3] |= (uint8_t)(1u << (c & 7));
  return 0;
}

/* ------------------------------------------------------------------ S15: render ----------- */

int orc_render(const orc_config *cfg, const double *theta, const uint8_t *bits, const orc_batch *b,
               double cut, double *rgb, double *depth, double *opacity, uint64_t *n_samples) {
  orc_levels lv;
  orc_mlp M;
  if (levels_init(cfg, &lv) != 0 || mlp_init(cfg, &M) != 0) return -1;
  const uint32_t R = b->n_rays, K = b->n_candidates;
  const uint64_t n_table = lv.off[lv.L] * lv.F;
  const double *Wm = theta + n_table;
  uint64_t total = 0;
  int64_t r;
#pragma omp parallel for schedule(dynamic, 16) reduction(+ : total)
  for (r = 0; r < (int64_t)R; ++r) {
    /* one ray at a time: S1-S3 with u == 0.5 on a 1-ray batch */
    orc_batch one = *b;
    one.n_rays = 1;
    one.origins = b->origins + 3 * r;
    one.dirs = b->dirs + 3 * r;
    uint32_t cnt, off[2];
    uint32_t *sr = malloc(sizeof(uint32_t) * K), *sk = malloc(sizeof(uint32_t) * K);
    float *st = malloc(sizeof(float) * K), *sd = malloc(sizeof(float) * K),
          *sx = malloc(sizeof(float) * 3 * K);
    double *sig = malloc(sizeof(double) * K), *col = malloc(sizeof(double) * 3 * K);
    int64_t n = orc_march(cfg, bits, &one, 0, 0, &cnt, off, sr, sk, st, sd, sx);
    double d[3] = {(double)one.dirs[0], (double)one.dirs[1], (double)one.dirs[2]};
    double Y[ORC_MAX_WIDTH], act[8 * ORC_MAX_WIDTH];
    orc_sh(cfg->sh_degree, d, Y);
    /* S4-S7 on the ray's samples in order, stopping where S8 stops (S15) */
    double T = 1.0;
    int64_t used = 0;
    for (int64_t i = 0; i < n; ++i) {
      encode_point(&lv, theta, sx + 3 * i, NULL, NULL, act + M.a_e);
      mlp_forward(&M, Wm, Y, act);
      sig[i] = act[M.a_sigma];
      for (int c = 0; c < 3; ++c) col[3 * i + c] = act[M.a_rgb + c];
      used = i + 1;
      T *= exp(-sig[i] * (double)sd[i]);
      if (cut > 0.0 && T < cut) break;
    }
    composite_ray((uint32_t)used, sig, 1, col, 3, st, sd, cfg->bg, cut, rgb + 3 * r, depth + r,
                  opacity ? opacity + r : &T, NULL, NULL);
    total += (uint64_t)used;
    free(sr); free(sk); free(st); free(sd); free(sx); free(sig); free(col);
  }
  if (n_samples) *n_samples = total;
  return 0;
}

/* ---- F1: ray-batch sampler over a keyframe store (header comment of orc_sample_batch) ---------
 * Plain loop over rays; every float operation is a single binary32 operation (the file is compiled with
 * -ffp-contract=off, and fmaf / sqrtf / division are correctly rounded). */
void orc_sample_batch(const orc_keyframe *kfs, uint32_t n_kf, uint64_t seed, uint32_t draw, uint32_t n_rays,
                      uint32_t *kf_out, uint32_t *pix_out, float *origins, float *dirs, float *rgb, float *depth,
                      float *depth_var) {
  for (uint32_t r = 0; r < n_rays; ++r) {
    const uint32_t h1 = orc_hash32(seed, draw, r, 0xffff0001u);
    const uint32_t kf = (uint32_t)(((uint64_t)h1 * (uint64_t)n_kf) >> 32);
    const orc_keyframe *k = &kfs[kf];
    const uint32_t h2 = orc_hash32(seed, draw, r, 0xffff0002u);
    const uint32_t pix = (uint32_t)(((uint64_t)h2 * ((uint64_t)k->width * k->height)) >> 32);
    const uint32_t u = pix % k->width, v = pix / k->width;
    const float xc = ((float)u - k->cx) / k->fx;
    const float yc = ((float)v - k->cy) / k->fy;
    const float n2 = fmaf(xc, xc, fmaf(yc, yc, 1.0f));
    const float n = sqrtf(n2);
    const float dx = xc / n, dy = yc / n, dz = 1.0f / n;
    for (int i = 0; i < 3; ++i) {
      float acc = k->R[3 * i + 2] * dz;
      acc = fmaf(k->R[3 * i + 1], dy, acc);
      acc = fmaf(k->R[3 * i + 0], dx, acc);
      dirs[3 * (size_t)r + i] = acc;
      origins[3 * (size_t)r + i] = k->t[i];
      rgb[3 * (size_t)r + i] = k->rgb[3 * (size_t)pix + i];
    }
    depth[r] = k->depth[pix] * n;
    depth_var[r] = k->depth_var[pix] * n2;
    if (kf_out) kf_out[r] = kf;
    if (pix_out) pix_out[r] = pix;
  }
}

/* ---- F2, the update (header comment of orc_pose_step) ---------------------------------------------------------- */
void orc_pose_step(double *R, double *t, double *m, double *v, uint32_t *count, const double *g, double lr_t, double lr_r,
                   double beta1, double beta2, double eps) {
  const uint32_t k = *count + 1;
  const double bc1 = 1.0 - pow(beta1, (double)k), bc2 = 1.0 - pow(beta2, (double)k);
  double delta[6];
  for (int i = 0; i < 6; ++i) {
    m[i] = beta1 * m[i] + (1.0 - beta1) * g[i];
    v[i] = beta2 * v[i] + (1.0 - beta2) * g[i] * g[i];
    delta[i] = (i < 3 ? lr_t : lr_r) * (m[i] / bc1) / (sqrt(v[i] / bc2) + eps);
  }
  for (int i = 0; i < 3; ++i) t[i] -= delta[i];
  /* E = exp(-[w]x), w = delta_omega: E = I - sin(a)/a [w]x + (1 - cos a)/a^2 [w]x^2, a = |w| */
  const double w[3] = {delta[3], delta[4], delta[5]};
  const double a2 = w[0] * w[0] + w[1] * w[1] + w[2] * w[2], a = sqrt(a2);
  const double A = a > 1e-12 ? sin(a) / a : 1.0, B = a > 1e-12 ? (1.0 - cos(a)) / a2 : 0.5;
  const double K[9] = {0.0, -w[2], w[1], w[2], 0.0, -w[0], -w[1], w[0], 0.0};
  double K2[9], E[9], Rn[9];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      K2[3 * i + j] = 0.0;
      for (int q = 0; q < 3; ++q) K2[3 * i + j] += K[3 * i + q] * K[3 * q + j];
    }
  for (int i = 0; i < 9; ++i) E[i] = ((i % 4 == 0) ? 1.0 : 0.0) - A * K[i] + B * K2[i];
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      Rn[3 * i + j] = 0.0;
      for (int q = 0; q < 3; ++q) Rn[3 * i + j] += E[3 * i + q] * R[3 * q + j];
    }
  for (int i = 0; i < 9; ++i) R[i] = Rn[i];
  *count = k;
}
