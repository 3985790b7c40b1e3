/*
 * abm_oracle.h -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded fp64 CPU oracle for the hot path of arXiv 1104.2499
 * (M. Zabicki, "OpenCL/OpenGL approach for studying active Brownian motion").
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this library.  It shares no code, header, table or constant generator
 * with the CUDA path (paper_1104_2499_b200/csrc, include/abm.h); neither includes the other.
 *
 * What the path computes (citations: PAPER.md line, section/equation):
 *   Eq. 1  de/dt = q - c e - d e v^2                        energy depot
 *   Eq. 2  dv/dt = F0 + d e v - gamma0 v - U'(x) + sqrt(2D) xi(t)
 *                         (the trailing "v" in the extraction is a garble: noise is additive,
 *                          PAPER.md:63 "white Gaussian noise of intensity sqrt(2D)"; reading G1)
 *   Eq. 3  ratchet potential, two harmonics (reading G2):
 *                         U(x) = A1 sin(th) + A2 sin(2 th),  th = 2 pi (x + phi) / L
 *                         (the additive constant 0.499 h does not enter the dynamics)
 *   implied               dx/dt = v   (reading G3)
 *   Fig. 1  per work item: for i = 0..T { uniform RNG; Box-Muller; new v, e }
 *   BASELINE.json         time-periodic tilt A cos(omega t); Euler-Maruyama / stochastic Heun;
 *                         Philox4x32-10 keyed by (seed, trajectory, step); ensemble moments.
 *
 * All arithmetic is IEEE double.  `precision` only selects which uniform map the run uses
 * (reading 8c-3/8c-5 in DESIGN.md), so that an fp32 GPU run and this oracle consume the
 * identical random numbers.
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"):
 *   abo_philox4x32_10 .......... Random123 known-answer vectors (tests/golden/philox4x32_10_kat.txt)
 *   abo_uniform / abo_normal ... range, exactness, moments of 10^7 draws, max |z| bound
 *   abo_potential / abo_rhs .... finite difference of U, Eq. 3 normalisation (min 0 at x=0, max h)
 *   abo_step (EM) .............. exact OU variance recursion, e(t) closed form, x_n closed form,
 *                                depot stationary speed, Boltzmann average, zero current limits
 *   abo_step (Heun) ............ x_n closed form, order-2 convergence, tilt analytic solution
 *   abo_run / abo_init ......... independent numpy restatement at tiny N, split-run invariance
 *   abo_moments ................ numpy mean/var
 *   abo_xorshift128 ............ Marsaglia (2003) xor128 first outputs from the paper's default state
 *                                (tests/golden/xorshift128_kat.txt), invertibility, normal moments
 *   abo_raster / abo_colormap .. numpy.histogram2d on points away from bin edges, a hand-counted
 *                                fixture (tests/golden/raster_small.txt), edge and wrap cases
 * Parity unpinned: the magnitude of the ratchet current <v> (the paper prints no value; its
 * Fig. 2 is not available).
 */
#ifndef ABM_ORACLE_H
#define ABM_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct abo_params {
  int32_t precision;  /* 0: run uses the fp32 uniform maps; 1: the fp64 maps          */
  int32_t integrator; /* 0: Euler-Maruyama; 1: stochastic Heun                         */
  int32_t init_v;     /* 0: v(0) = v0; 1: v(0) ~ N(0, D/gamma0) from the init block    */
  int32_t rng;        /* 0: Philox4x32-10 stream (BASELINE.json); 1: per-trajectory Marsaglia
                         xorshift state as in the paper   */
  double dt;
  double gamma0, q, c, d, D; /* Eqs. 1-2 */
  double F0;                 /* constant load force, enters as +F0 (reading G13)       */
  double A, omega;           /* tilt A cos(omega t), t_n = n dt (reading G15)          */
  double L, A1, A2, phi;     /* potential, see above                                   */
  double v0, e0;             /* constant initial values                                */
} abo_params;

/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): 10 rounds, multipliers 0xD2511F53,
 * 0xCD9E8D57, key increments 0x9E3779B9, 0xBB67AE85. */
void abo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* Stream layout: key = (seed lo, seed hi); ctr = (b lo, b hi, traj lo, traj hi). */
void abo_block(uint64_t seed, uint64_t traj, uint64_t b, uint32_t out[4]);

/* Uniform in (0,1): fp32 runs ((w >> 9) + 0.5) 2^-23; fp64 runs (w + 0.5) 2^-32. */
double abo_uniform(uint32_t w, int32_t precision);

/* Standard normal of global step n (0-based) of trajectory traj:
 * block b = n >> 2, pair p = (n >> 1) & 1, u1 = u(w[2p]), u2 = u(w[2p+1]),
 * r = sqrt(-2 ln u1), z = r cos(2 pi u2) for even n, r sin(2 pi u2) for odd n. */
double abo_normal(uint64_t seed, uint64_t traj, uint64_t n, int32_t precision);

/* Bulk form of abo_normal: out[k * n_steps + j] = normal of trajectory traj_first + k, step
 * step_first + j (a plain double loop over abo_normal). */
void abo_normals(uint64_t seed, uint64_t traj_first, uint64_t n_traj, uint64_t step_first,
                 uint64_t n_steps, int32_t precision, double* out);

/* NEXT-4 generator variant ("Marsaglia xor-shift algorithm"; the exact variant is not
 * printed -- reading: xor128 of G. Marsaglia, "Xorshift RNGs", J. Stat. Softw. 8(14), 2003, p. 5:
 * t = x ^ (x << 11); x = y; y = z; z = w; w = w ^ (w >> 19) ^ t ^ (t >> 8); return w).
 * One state (x, y, z, w) per trajectory, seeded from the Philox block b = 2^64 - 2 of the trajectory
 * (all-zero is replaced by (0, 0, 0, 1)).  Output j (0-based) of the trajectory's generator feeds:
 * pair p = n >> 1 of steps uses u1 = u(output 2p), u2 = u(output 2p + 1); normals as for Philox. */
uint32_t abo_xorshift128(uint32_t s[4]);
void abo_xorshift_seed(uint64_t seed, uint64_t traj, uint32_t s[4]);
/* Normal of step n in xorshift mode, by iterating the generator from its seed (O(n): tests only). */
double abo_normal_xorshift(uint64_t seed, uint64_t traj, uint64_t n, int32_t precision);

/* U(x) without the additive constant, and the right-hand side of Eqs. 1-2 at (x,v,e,t). */
double abo_potential(const abo_params* p, double x);
void abo_rhs(const abo_params* p, double x, double v, double e, double t, double* ax, double* av,
             double* ae);

/* Initial state from the init block b = 2^64 - 1 of the trajectory. */
void abo_init(const abo_params* p, uint64_t seed, uint64_t traj, double* x, double* v, double* e);

/* One step n -> n+1 of one trajectory (in place). */
void abo_step(const abo_params* p, uint64_t seed, uint64_t traj, uint64_t n, double* x, double* v,
              double* e);

/* Trajectories traj_first + k * traj_stride, k < n_traj: initialise / advance steps
 * [step_first, step_first + n_steps).  Arrays are indexed by k. */
void abo_init_many(const abo_params* p, uint64_t seed, uint64_t traj_first, uint64_t traj_stride,
                   uint64_t n_traj, double* x, double* v, double* e);
void abo_run(const abo_params* p, uint64_t seed, uint64_t traj_first, uint64_t traj_stride,
             uint64_t n_traj, uint64_t step_first, uint64_t n_steps, double* x, double* v,
             double* e);

/* Ensemble moments over n entries (population normalisation 1/N, reading G11); x0 = initial
 * positions.  out[8] = mean_x, var_x, mean_v, var_v, mean_e, mean_dx, mean_dx2, mean_x2
 * with dx = x - x0. */
void abo_moments(const double* x, const double* v, const double* e, const double* x0, uint64_t n,
                 double out[8]);

/* Headless presentation: 2-D histogram of (x mod L, v) and its grey-ramp RGBA8 image (include/abm.h
 * states the bin rule). */
void abo_raster(const double* x, const double* v, uint64_t n, double L, uint32_t W, uint32_t H,
                double v_min, double v_max, uint32_t* counts);
void abo_colormap(const uint32_t* counts, uint64_t n_bins, uint32_t saturation, uint8_t* rgba);

#ifdef __cplusplus
}
#endif
#endif
