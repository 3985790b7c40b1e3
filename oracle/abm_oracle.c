/*
 * abm_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.  See abm_oracle.h.
 *
 * The method is an iteration (a discretised SDE), so this file follows the algorithm step by
 * step in the order of SURVEY.md 8(c) / DESIGN.md "Oracle", in plain fp64, one trajectory at a
 * time, with no blocking, fusion or reordering.
 */
#include "abm_oracle.h"

#include <math.h>

#define ABO_TWO_PI 6.283185307179586476925286766559

/* ---- 8(c)-1: Philox4x32-10 ------------------------------------------------------------- */

void abo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0; /* (hi0, lo0) */
    uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2; /* (hi1, lo1) */
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; /* key schedule, after each round */
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ---- 8(c)-2: stream layout --------------------------------------------------------------- */

void abo_block(uint64_t seed, uint64_t traj, uint64_t b, uint32_t out[4]) {
  uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
  uint32_t ctr[4] = {(uint32_t)(b & 0xffffffffu), (uint32_t)(b >> 32),
                     (uint32_t)(traj & 0xffffffffu), (uint32_t)(traj >> 32)};
  abo_philox4x32_10(ctr, key, out);
}

/* ---- 8(c)-3: uniform map ----------------------------------------------------------------- */

double abo_uniform(uint32_t w, int32_t precision) {
  if (precision == 0) return ((double)(w >> 9) + 0.5) * (1.0 / 8388608.0);   /* 2^-23 */
  return ((double)w + 0.5) * (1.0 / 4294967296.0);                           /* 2^-32 */
}

/* ---- 8(c)-4: Box-Muller normal of step n ------------------------------ */

double abo_normal(uint64_t seed, uint64_t traj, uint64_t n, int32_t precision) {
  uint32_t w[4];
  abo_block(seed, traj, n >> 2, w);
  int p = (int)((n >> 1) & 1u);
  double u1 = abo_uniform(w[2 * p], precision);
  double u2 = abo_uniform(w[2 * p + 1], precision);
  double r = sqrt(-2.0 * log(u1));
  if ((n & 1u) == 0) return r * cos(ABO_TWO_PI * u2);
  return r * sin(ABO_TWO_PI * u2);
}

void abo_normals(uint64_t seed, uint64_t traj_first, uint64_t n_traj, uint64_t step_first,
                 uint64_t n_steps, int32_t precision, double* out) {
  for (uint64_t k = 0; k < n_traj; ++k)
    for (uint64_t j = 0; j < n_steps; ++j)
      out[k * n_steps + j] = abo_normal(seed, traj_first + k, step_first + j, precision);
}

/* ---- NEXT-4: the paper's generator family -------------------------------------- */

uint32_t abo_xorshift128(uint32_t s[4]) {
  uint32_t t = s[0] ^ (s[0] << 11);
  s[0] = s[1]; s[1] = s[2]; s[2] = s[3];
  s[3] = s[3] ^ (s[3] >> 19) ^ t ^ (t >> 8);
  return s[3];
}

void abo_xorshift_seed(uint64_t seed, uint64_t traj, uint32_t s[4]) {
  abo_block(seed, traj, UINT64_MAX - 1u, s);
  if ((s[0] | s[1] | s[2] | s[3]) == 0u) s[3] = 1u; /* the one forbidden state */
}

static double normal_from_pair(uint32_t a, uint32_t b, uint64_t n, int32_t precision) {
  double u1 = abo_uniform(a, precision);
  double u2 = abo_uniform(b, precision);
  double r = sqrt(-2.0 * log(u1));
  if ((n & 1u) == 0) return r * cos(ABO_TWO_PI * u2);
  return r * sin(ABO_TWO_PI * u2);
}

double abo_normal_xorshift(uint64_t seed, uint64_t traj, uint64_t n, int32_t precision) {
  uint32_t s[4];
  abo_xorshift_seed(seed, traj, s);
  for (uint64_t j = 0; j < 2u * (n >> 1); ++j) (void)abo_xorshift128(s); /* outputs of earlier pairs */
  uint32_t a = abo_xorshift128(s);
  uint32_t b = abo_xorshift128(s);
  return normal_from_pair(a, b, n, precision);
}

/* ---- 8(c)-6: right-hand side (Eqs. 1-3) --------------------------------------------------- */

double abo_potential(const abo_params* p, double x) {
  double th = ABO_TWO_PI * (x + p->phi) / p->L;
  return p->A1 * sin(th) + p->A2 * sin(2.0 * th);
}

void abo_rhs(const abo_params* p, double x, double v, double e, double t, double* ax, double* av,
             double* ae) {
  double th = ABO_TWO_PI * (x + p->phi) / p->L;
  double dU = (ABO_TWO_PI / p->L) * (p->A1 * cos(th) + 2.0 * p->A2 * cos(2.0 * th)); /* U'(x) */
  *ax = v;                                                                   /* dx/dt = v */
  *av = -p->gamma0 * v + p->d * e * v - dU + p->F0 + p->A * cos(p->omega * t); /* Eq. 2 */
  *ae = p->q - p->c * e - p->d * e * v * v;                                    /* Eq. 1 */
}

/* ---- 8(c)-5: initial state from the init block ------------------------------------------- */

void abo_init(const abo_params* p, uint64_t seed, uint64_t traj, double* x, double* v, double* e) {
  uint32_t w[4];
  abo_block(seed, traj, UINT64_MAX, w);
  if (p->precision == 0)
    *x = p->L * ((double)(w[0] >> 8) * (1.0 / 16777216.0)); /* L (w0 >> 8) 2^-24 */
  else
    *x = p->L * ((double)w[0] * (1.0 / 4294967296.0));      /* L w0 2^-32 */
  if (p->init_v == 0) {
    *v = p->v0;
  } else {
    double u1 = abo_uniform(w[2], p->precision);
    double u2 = abo_uniform(w[3], p->precision);
    *v = sqrt(p->D / p->gamma0) * sqrt(-2.0 * log(u1)) * cos(ABO_TWO_PI * u2);
  }
  *e = p->e0;
  /* w[1] is reserved. */
}

/* ---- 8(c)-7/8: one step ------------------------------------------------------------------- */

static void step_with_normal(const abo_params* p, uint64_t n, double z, double* x, double* v,
                             double* e) {
  double dt = p->dt;
  double t_n = (double)n * dt;
  double sigma = sqrt(2.0 * p->D * dt);
  double ax, av, ae;
  abo_rhs(p, *x, *v, *e, t_n, &ax, &av, &ae);
  if (p->integrator == 0) {
    /* Euler-Maruyama: every right-hand side at the old state (reading G4). */
    double xn = *x + ax * dt;
    double vn = *v + av * dt + sigma * z;
    double en = *e + ae * dt;
    *x = xn; *v = vn; *e = en;
  } else {
    /* Stochastic Heun: predictor with the full noise increment, corrector averages the
     * drift at (X, t_n) and (X~, t_{n+1}); same z in both (reading G16). */
    double t_n1 = (double)(n + 1) * dt;
    double xp = *x + ax * dt;
    double vp = *v + av * dt + sigma * z;
    double ep = *e + ae * dt;
    double bx, bv, be;
    abo_rhs(p, xp, vp, ep, t_n1, &bx, &bv, &be);
    double xn = *x + 0.5 * (ax + bx) * dt;
    double vn = *v + 0.5 * (av + bv) * dt + sigma * z;
    double en = *e + 0.5 * (ae + be) * dt;
    *x = xn; *v = vn; *e = en;
  }
}

void abo_step(const abo_params* p, uint64_t seed, uint64_t traj, uint64_t n, double* x, double* v,
              double* e) {
  double z = p->rng == 0 ? abo_normal(seed, traj, n, p->precision)
                         : abo_normal_xorshift(seed, traj, n, p->precision);
  step_with_normal(p, n, z, x, v, e);
}

/* ---- ensembles ----------------------------------------------------------------------------- */

void abo_init_many(const abo_params* p, uint64_t seed, uint64_t traj_first, uint64_t traj_stride,
                   uint64_t n_traj, double* x, double* v, double* e) {
  for (uint64_t k = 0; k < n_traj; ++k)
    abo_init(p, seed, traj_first + k * traj_stride, &x[k], &v[k], &e[k]);
}

void abo_run(const abo_params* p, uint64_t seed, uint64_t traj_first, uint64_t traj_stride,
             uint64_t n_traj, uint64_t step_first, uint64_t n_steps, double* x, double* v,
             double* e) {
  for (uint64_t k = 0; k < n_traj; ++k) {
    uint64_t traj = traj_first + k * traj_stride;
    if (p->rng == 0) {
      for (uint64_t n = step_first; n < step_first + n_steps; ++n)
        abo_step(p, seed, traj, n, &x[k], &v[k], &e[k]);
    } else {
      /* xorshift mode: the same steps with the generator carried along instead of re-run from its
       * seed at every step (abo_step does that; tests check the two agree). */
      uint32_t s[4], a = 0, b = 0;
      abo_xorshift_seed(seed, traj, s);
      for (uint64_t j = 0; j < 2u * (step_first >> 1); ++j) (void)abo_xorshift128(s);
      int have_pair = 0;
      for (uint64_t n = step_first; n < step_first + n_steps; ++n) {
        if (!have_pair || (n & 1u) == 0) {
          a = abo_xorshift128(s);
          b = abo_xorshift128(s);
          have_pair = 1;
        }
        step_with_normal(p, n, normal_from_pair(a, b, n, p->precision), &x[k], &v[k], &e[k]);
      }
    }
  }
}

/* ---- 8(c)-9: moments (two-pass, population normalisation) ---------------------------------- */

void abo_moments(const double* x, const double* v, const double* e, const double* x0, uint64_t n,
                 double out[8]) {
  double N = (double)n;
  double sx = 0, sv = 0, se = 0, sdx = 0, sdx2 = 0, sx2 = 0;
  for (uint64_t k = 0; k < n; ++k) {
    double dx = x[k] - x0[k];
    sx += x[k]; sv += v[k]; se += e[k];
    sdx += dx; sdx2 += dx * dx; sx2 += x[k] * x[k];
  }
  double mx = sx / N, mv = sv / N;
  double vx = 0, vv = 0;
  for (uint64_t k = 0; k < n; ++k) {
    vx += (x[k] - mx) * (x[k] - mx);
    vv += (v[k] - mv) * (v[k] - mv);
  }
  out[0] = mx; out[1] = vx / N; out[2] = mv; out[3] = vv / N;
  out[4] = se / N; out[5] = sdx / N; out[6] = sdx2 / N; out[7] = sx2 / N;
}

/* Headless presentation (the paper draws each work item as a point of the
 * vertex buffer): 2-D histogram of the points (x mod L, v).  Bin rule as stated in
 * include/abm.h, one IEEE double operation at a time:
 *   xi = x / L; f = xi - floor(xi); ix = min(W - 1, floor(f W))
 *   eta = (v - v_min) / (v_max - v_min); dropped unless 0 <= eta < 1; iy = min(H - 1, floor(eta H))
 * counts[iy * W + ix] += 1.  counts must be zeroed by the caller. */
void abo_raster(const double* x, const double* v, uint64_t n, double L, uint32_t W, uint32_t H,
                double v_min, double v_max, uint32_t* counts) {
  double v_range = v_max - v_min;
  for (uint64_t k = 0; k < n; ++k) {
    double xi = x[k] / L;
    double f = xi - floor(xi);
    double eta = (v[k] - v_min) / v_range;
    if (!(eta >= 0.0) || !(eta < 1.0) || !(f >= 0.0)) continue;
    double fx = floor(f * (double)W), fy = floor(eta * (double)H);
    uint32_t ix = fx >= (double)W ? W - 1 : (uint32_t)fx;
    uint32_t iy = fy >= (double)H ? H - 1 : (uint32_t)fy;
    counts[(uint64_t)iy * W + ix] += 1u;
  }
}

/* Grey ramp of include/abm.h: level = min(255, floor(255 c / saturation)), alpha 255. */
void abo_colormap(const uint32_t* counts, uint64_t n_bins, uint32_t saturation, uint8_t* rgba) {
  for (uint64_t b = 0; b < n_bins; ++b) {
    uint64_t c = counts[b];
    uint64_t lv = c >= saturation ? 255u : (255u * c) / saturation;
    rgba[4 * b + 0] = rgba[4 * b + 1] = rgba[4 * b + 2] = (uint8_t)lv;
    rgba[4 * b + 3] = 255;
  }
}

