// abm_device.cuh -- device-side building blocks of the hot path (sm_100a).
//
// S1 Philox4x32-10 block, S2 Box-Muller, S3 force, S4 Euler-Maruyama / stochastic Heun update
// (Fig. 1 loop body, Eqs. 1-3 at PAPER.md:59-69).
//
// Everything is written with explicit fma/mul/add intrinsics so that the unrolled 4-step path
// and the single-step path of the step kernel round identically (abm_step(a); abm_step(b) must
// be bit-identical to abm_step(a+b)).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace abm {

// ---------------------------------------------------------------------------------------------
// S1  Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), restated from the published round
// function: (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2, c' = (hi1^c1^k0, lo1, hi0^c3^k1, lo0),
// key += (W0, W1) after each round.
// ---------------------------------------------------------------------------------------------
constexpr uint32_t PHILOX_M0 = 0xD2511F53u;
constexpr uint32_t PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u;
constexpr uint32_t PHILOX_W1 = 0xBB67AE85u;

// 32 x 32 -> 64 multiply as ONE IMAD.WIDE.U32 (the C++ form `uint64_t(a) * M` makes ptxas add
// a zero high-word correction after every product).
__device__ __forceinline__ void mul_wide(uint32_t a, uint32_t m, uint32_t& hi, uint32_t& lo) {
  asm("{\n\t.reg .u64 p;\n\tmul.wide.u32 p, %2, %3;\n\tmov.b64 {%0, %1}, p;\n\t}"
      : "=r"(lo), "=r"(hi)
      : "r"(a), "r"(m));
}

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               uint32_t k0, uint32_t k1) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    uint32_t hi0, lo0, hi1, lo1;
    mul_wide(c0, PHILOX_M0, hi0, lo0);
    mul_wide(c2, PHILOX_M1, hi1, lo1);
    c0 = hi1 ^ c1 ^ (k0 + PHILOX_W0 * static_cast<uint32_t>(r));  // LOP3 with a uniform operand
    c1 = lo1;
    c2 = hi0 ^ c3 ^ (k1 + PHILOX_W1 * static_cast<uint32_t>(r));
    c3 = lo0;
  }
  return make_uint4(c0, c1, c2, c3);
}

// One Philox round with round key (k0, k1).
__device__ __forceinline__ void philox_round(uint32_t& c0, uint32_t& c1, uint32_t& c2, uint32_t& c3,
                                             uint32_t k0, uint32_t k1) {
  uint32_t hi0, lo0, hi1, lo1;
  mul_wide(c0, PHILOX_M0, hi0, lo0);
  mul_wide(c2, PHILOX_M1, hi1, lo1);
  c0 = hi1 ^ c1 ^ k0;
  c1 = lo1;
  c2 = hi0 ^ c3 ^ k1;
  c3 = lo0;
}

// The first two rounds split by what their inputs depend on, for a run of blocks b = (b_lo, b_hi)
// of ONE trajectory with b_hi fixed ("Philox block table"):
//   after round 0:  c0' = hi(M1 t_lo) ^ b_hi ^ k0      per trajectory, the same for every block
//                   c1' = lo(M1 t_lo)                  per trajectory
//                   c2' = hi(M0 b_lo) ^ t_hi ^ k1      per block, the same for every trajectory
//                   c3' = lo(M0 b_lo)                  per block
//   after round 1:  c0'' = [hi(M1 c2') ^ k0_1] ^ c1'   c1'' = lo(M1 c2')
//                   c2'' = hi(M0 c0') ^ [c3' ^ k1_1]   c3'' = lo(M0 c0')
// PhiloxTraj holds the per-trajectory words (2 multiplies, once per run); PhiloxBlockHead holds
// the bracketed per-block words (2 multiplies per block, shared by all trajectories whose t_hi is
// equal -- the step kernel keeps them in a shared-memory table computed once per CTA).
struct PhiloxTraj {
  uint32_t p1, p2, p3;  // c1', hi(M0 c0'), lo(M0 c0')
};
struct PhiloxBlockHead {
  uint32_t u0, u1, u2;  // hi(M1 c2') ^ k0_1, lo(M1 c2'), c3' ^ k1_1
};
__device__ __forceinline__ PhiloxTraj philox_traj(uint32_t t_lo, uint32_t b_hi, uint32_t k0) {
  uint32_t h1, l1;
  mul_wide(t_lo, PHILOX_M1, h1, l1);
  PhiloxTraj t;
  t.p1 = l1;
  mul_wide(h1 ^ b_hi ^ k0, PHILOX_M0, t.p2, t.p3);
  return t;
}
__device__ __forceinline__ PhiloxBlockHead philox_block_head(uint32_t b_lo, uint32_t t_hi,
                                                             uint32_t k0, uint32_t k1) {
  uint32_t h0, l0, h1, l1;
  mul_wide(b_lo, PHILOX_M0, h0, l0);
  mul_wide(h0 ^ t_hi ^ k1, PHILOX_M1, h1, l1);
  PhiloxBlockHead u;
  u.u0 = h1 ^ (k0 + PHILOX_W0);
  u.u1 = l1;
  u.u2 = l0 ^ (k1 + PHILOX_W1);
  return u;
}
// Rounds 2..9 on the state after round 1 assembled from the two halves.
__device__ __forceinline__ uint4 philox_finish(const PhiloxTraj& t, uint32_t u0, uint32_t u1,
                                               uint32_t u2, uint32_t k0, uint32_t k1) {
  uint32_t c0 = u0 ^ t.p1, c1 = u1, c2 = t.p2 ^ u2, c3 = t.p3;
#pragma unroll
  for (int r = 2; r < 10; ++r)
    philox_round(c0, c1, c2, c3, k0 + PHILOX_W0 * static_cast<uint32_t>(r),
                 k1 + PHILOX_W1 * static_cast<uint32_t>(r));
  return make_uint4(c0, c1, c2, c3);
}

// The same with the round keys read from host-computed tables (kernel parameters: constant-bank
// operands of the LOP3s, no uniform registers or in-loop key arithmetic).
__device__ __forceinline__ uint4 philox_finish_rk(const PhiloxTraj& t, uint32_t u0, uint32_t u1,
                                                  uint32_t u2, const uint32_t (&rk0)[10],
                                                  const uint32_t (&rk1)[10]) {
  uint32_t c0 = u0 ^ t.p1, c1 = u1, c2 = t.p2 ^ u2, c3 = t.p3;
#pragma unroll
  for (int r = 2; r < 10; ++r) philox_round(c0, c1, c2, c3, rk0[r], rk1[r]);
  return make_uint4(c0, c1, c2, c3);
}

// Stream layout: key = (seed lo, seed hi),
// ctr = (block lo, block hi, trajectory lo, trajectory hi).
__device__ __forceinline__ uint4 philox_block(uint64_t seed, uint64_t traj, uint64_t b) {
  return philox4x32_10(static_cast<uint32_t>(b), static_cast<uint32_t>(b >> 32),
                       static_cast<uint32_t>(traj), static_cast<uint32_t>(traj >> 32),
                       static_cast<uint32_t>(seed), static_cast<uint32_t>(seed >> 32));
}

constexpr uint64_t INIT_BLOCK = 0xFFFFFFFFFFFFFFFFull;  // block index of the init block
constexpr uint64_t XS_SEED_BLOCK = 0xFFFFFFFFFFFFFFFEull;  // block that seeds the xorshift state

// ---------------------------------------------------------------------------------------------
// Generator variant: the paper's "Marsaglia xor-shift", read
// as xor128 of Marsaglia (2003): t = x ^ (x << 11); x = y; y = z; z = w;
// w = w ^ (w >> 19) ^ t ^ (t >> 8).  State (x, y, z, w) per trajectory in global memory between
// launches, in registers inside one.  Six ALU-pipe instructions per word and none on the FMA
// dispatch port, against 4 IMAD.WIDE + 4.5 LOP3 per word for Philox4x32-10.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t xorshift128(uint4& s) {
  const uint32_t t = s.x ^ (s.x << 11);
  s.x = s.y;
  s.y = s.z;
  s.z = s.w;
  s.w = s.w ^ (s.w >> 19) ^ t ^ (t >> 8);
  return s.w;
}
__device__ __forceinline__ uint4 xorshift128_x4(uint4& s) {
  uint4 w;
  w.x = xorshift128(s);
  w.y = xorshift128(s);
  w.z = xorshift128(s);
  w.w = xorshift128(s);
  return w;
}
__device__ __forceinline__ uint4 xorshift_seed(uint64_t seed, uint64_t traj) {
  uint4 s = philox_block(seed, traj, XS_SEED_BLOCK);
  if ((s.x | s.y | s.z | s.w) == 0u) s.w = 1u;  // the one forbidden state
  return s;
}

// ---------------------------------------------------------------------------------------------
// Approximate single-precision special functions: one MUFU each (plus the range-scale FMUL the
// hardware wants in front of SIN/COS).  .ftz keeps ptxas from adding denormal fix-up code.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float fast_lg2(float x) {
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float fast_sqrt(float x) {
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float fast_cos(float x) {
  float y;
  asm("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float fast_sin(float x) {
  float y;
  asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// ---------------------------------------------------------------------------------------------
// Per-parameter-set coefficients, precomputed in fp64 on the host and rounded once.
// ---------------------------------------------------------------------------------------------
template <typename Real>
struct Coef {
  Real dt, hdt;        // dt, dt/2
  Real gamma0, d, q, c;
  Real k0, k1, k2;     // -U'(x) + F0 = k0 + k1 cos(th) + k2 cos(th)^2
  Real th_s, th_o;     // fp32: th = th_s x + th_o [rad];  fp64: th/pi = th_s x + th_o
  Real s2;             // fp32: 2 sigma^2 (so rho^2 = s2 lambda, lambda = -ln u1, see box_muller_f32); fp64: sigma
  Real A;              // tilt amplitude
  Real L, v0, e0, sv;  // init: x0 = L u, v0, e0, sv = sqrt(D/gamma0)
  Real bm_o;           // fp32: 2 pi 2^-24 - 3 pi, offset of the Box-Muller angle (see S2)
  Real fxS;            // precise fp32 mode: 2^32 / L, length -> fixed-point units (S4)
  Real pad;
};
static_assert(sizeof(Coef<float>) == 80, "Coef<float> layout");
static_assert(sizeof(Coef<double>) == 160, "Coef<double> layout");

template <typename Real>
struct State {
  Real x, v, e;
  Real xl;       // unused
  // precise fp32 mode only (see "Precise fp32 mode" below): the position is (xc 2^32 + xf) L 2^-32 + x
  uint32_t xf;   //   fraction of a period, 32-bit fixed point
  int32_t xc;    //   whole periods
  Real thb;      //   angle of the fixed-point part, 2 pi xf 2^-32 + phase (recomputed, not stored)
};

// ---------------------------------------------------------------------------------------------
// S2  Box-Muller on a word pair -> (rho, cs, sn) with rho = sigma sqrt(-2 ln u1) and
// sigma z_even = rho cos(2 pi u2), sigma z_odd = rho sin(2 pi u2).
// fp32 uniform map ((w >> 9) + 0.5) 2^-23, built exactly as m - (1 - 2^-24) with
// m = as_float((w >> 9) + 0x3f800000) in [1, 2).
//
// fp32: the angle handed to MUFU is 2 pi u2 - pi, in [-pi, pi), where one FMA rounds to at most
// 2^-23 rad (four times finer than on [2 pi, 4 pi)); that half turn flips the sign of both
// functions, so Normal2f carries cs = -cos(2 pi u2), sn = -sin(2 pi u2) and NEGATED = true tells
// the caller to use -rho (an operand modifier of the consuming FMA, no instruction).
// ---------------------------------------------------------------------------------------------
struct Normal2f {
  float rho, cs, sn;
  static constexpr bool NEGATED = true;
};

__device__ __forceinline__ float uniform_f32(uint32_t w) {
  const float m = __uint_as_float((w >> 9) + 0x3f800000u);
  return __fadd_rn(m, -(1.0f - 0x1p-24f));  // exact
}

// The radius.  lg2.approx is accurate to 2^-22 ABSOLUTELY on (1/2, 2), so as u1 -> 1, where the logarithm goes to
// 0, its relative error -- hence that of rho -- grows without bound: 63 % at u1 = 1 - 2^-24, i.e. 2.2e-4 sigma on
// v.  The exhaustive 100-step comparison with the oracle (every trajectory of configs [1-3]) found exactly these
// draws: 3 + 2 trajectories beyond 1e-5 in configs [2], [3], each with a uniform within 10^-6 of 1.  Branch-free
// repair, three instructions per pair (a branch anywhere inside the loop trip cuts the basic block in which ptxas
// interleaves Philox rounds and floating-point work: measured +15 %; two blocks of look-ahead with the test at
// the loop boundary: +8 %): with t = 1 - u1 (exact in fp32) and lambda = -ln u1 = t + t^2/2 + ... >= t,
//     lam = max(-ln2 lg2.approx(u1) - B, t),    B = ln2 2^-22 (the error bound, so that the first term <= lambda),
// is never above lambda + 0 and never below max(t, lambda - 2B): |lam - lambda| <= min(2B, t^2/2).  The radius
// sqrt(2 lam) is then off by at most 8e-6 (at t = 8e-4, rho = 0.04) instead of 2.2e-4, by 2.7e-7 at rho = 1.2 --
// 3.6e-7 on v at the largest sigma of the configs (D = 1) against a tolerance of 1e-5.
constexpr float BM_LG2_BIAS = 0.6931471805599453f * 0x1p-22f;

__device__ __forceinline__ Normal2f box_muller_f32(uint32_t wa, uint32_t wb, float s2,
                                                   float bm_o) {
  Normal2f o;
  const float m1 = __uint_as_float((wa >> 9) + 0x3f800000u);
  const float u1 = __fadd_rn(m1, -(1.0f - 0x1p-24f));   // uniform_f32(wa), exact
  const float t = __fadd_rn(1.0f, -u1);                 // exact: (2^24 - 2k - 1) 2^-24 has 24 bits (2 - 2^-24 - m1 would
                                                        // not be: 2 - 2^-24 is no fp32 number)
  // lam <= -ln u1 whatever the sign of MUFU.LG2's error; t <= -ln u1 always: the larger of the two (see above)
  const float lam = fmaxf(__fmaf_rn(fast_lg2(u1), -0.6931471805599453f, -BM_LG2_BIAS), t);
  o.rho = fast_sqrt(__fmul_rn(lam, s2));
  // 2 pi u2 - pi = 2 pi (m - 1 + 2^-24) - pi = 2 pi m + bm_o,  bm_o = 2 pi 2^-24 - 3 pi
  const float m2 = __uint_as_float((wb >> 9) + 0x3f800000u);
  const float ang = __fmaf_rn(m2, 6.283185307179586f, bm_o);
  o.cs = fast_cos(ang);
  o.sn = fast_sin(ang);
  return o;
}

// ---------------------------------------------------------------------------------------------
// fp64 cos(pi t), sin(pi t) for the hot loop.  The CUDA math library's cospi / sincospi spend
// more issue slots on materialising 64-bit polynomial coefficients (UMOV / IMAD.MOV pairs: DFMA
// takes no 64-bit immediate), quadrant selects and special-case branches than on DFMAs, and the
// fp64 kernel was issue-bound by them.  Here: t is reduced to r = t - rint(t) in [-1/2, 1/2]
// (magic-number rounding, exact), the parity of rint(t) goes to the sign bit with two integer
// instructions, and cos(pi r), sin(pi r) / r are degree-7 polynomials in r^2 (Chebyshev fits on
// r^2 in [0, 1/4]: 2.0e-15 absolute and 2.4e-16 relative with the rounded coefficients -- chosen
// against the 1e-12 trajectory tolerance, where a function error enters multiplied by dt or sigma;
// degree 8 reached 1e-16 for one more DFMA per evaluation) whose coefficients sit in constant
// memory, which DFMA reads as an operand.
// Valid for |t| < 2^51.
// ---------------------------------------------------------------------------------------------
constexpr int N_COSPI = 8;  // terms: degree 7 in r^2
__constant__ double C_COSPI[N_COSPI] = {
    0.9999999999999981, -4.934802200543686, 4.058712126333295, -1.3352627661817635,
    0.23533058831317874, -0.025806531975921563, 0.0019278700526981333, -0.0001004164642205389};

__device__ __forceinline__ double reduce_half_turns(double t, uint32_t& sign) {
  const double magic = 6755399441055744.0;  // 1.5 * 2^52: adding it rounds to an integer
  const double tm = __dadd_rn(t, magic);
  // parity of rint(t) -> sign bit.  A funnel shift: ptxas turns a plain `<< 31` into IMAD.U32 (x 2^31) on the
  // FMA pipe, whose dispatch port the FP64 pipe shares (profiles/r02_pipe_rates.txt) -- the one this kernel is short of.
  asm("shf.l.wrap.b32 %0, 0, %1, 31;" : "=r"(sign) : "r"(__double2loint(tm)));
  return __dadd_rn(t, -__dadd_rn(tm, -magic));             // exact
}
__device__ __forceinline__ double flip_sign(double p, uint32_t sign) {
  return __hiloint2double(__double2hiint(p) ^ static_cast<int>(sign), __double2loint(p));
}
__device__ __forceinline__ double cospi_f64(double t) {
  uint32_t sign;
  const double r = reduce_half_turns(t, sign);
  const double r2 = __dmul_rn(r, r);
  double p = C_COSPI[N_COSPI - 1];
#pragma unroll
  for (int k = N_COSPI - 2; k >= 0; --k) p = __fma_rn(p, r2, C_COSPI[k]);
  return flip_sign(p, sign);
}
// ---------------------------------------------------------------------------------------------
// fp64 Box-Muller from two small tables ("fp64 arithmetic").  The FP64 pipe (64 lanes/clk/SM)
// and the FMA pipes share one dispatch port, so what this kernel is short of is FP64 operations: the
// polynomial-only versions of round 1 took 17 (sin, cos) + 18 (-2 ln u) + 8 (sqrt) + 1 of them per pair;
// these take 10 + 9 + 7 + 1, with function errors of the same size (<= 4e-16 absolute for sin / cos,
// <= 7e-16 relative for ln u, < 1 ulp for the square root) against the 1e-12 trajectory tolerance.
//
// NoiseTables<double>: built on the host in extended precision once per process, uploaded per context,
// copied to shared memory by every CTA of an fp64 step kernel (20.5 KB, ~1 us); the single-step path
// reads the same shared copy, so split launches stay bit-identical.
//   circle[i] = (cos a_i, sin a_i),  a_i = 2 pi (i + 1/2) / 1024,  i < 1024
//   logt[i]   = (rc_i, -ln rc_i - [i >= LOG_ADJ_FROM] ln 2),  rc_i = fl(1 / c_i),  c_i = 1 + i / 256,  i <= 256
// ---------------------------------------------------------------------------------------------
constexpr int CIRCLE_BITS = 10;
constexpr int CIRCLE_N = 1 << CIRCLE_BITS;
constexpr int LOG_N = 257;
constexpr int LOG_ADJ_FROM = 106;                // c_i >= 1.412 ~ sqrt 2: the mantissa is taken as m / 2
constexpr int NOISE_TABLE_N = CIRCLE_N + LOG_N;  // double2 entries: circle first, then logt

// The shared-memory copy every CTA of an fp64 step kernel makes (stage_noise_tables in abm_kernels.cuh).  A static
// array, so that a look-up is LDS [index * 16 + constant]: with the tables behind pointers every look-up paid an
// integer add, which ptxas issues as IMAD.IADD on the FMA pipe.
__shared__ double2 s_noise[NOISE_TABLE_N];
template <typename Real>
struct NoiseTables {};  // a tag: fp32 has none (MUFU), fp64 reads s_noise
// A right shift the compiler cannot merge with the scaling of the table index that follows it: index -> address
// is then one shift-and-add (LEA, ALU pipe) instead of a mask and an add that ptxas issues on the FMA pipe.
template <int N>
__device__ __forceinline__ uint32_t shr_opaque(uint32_t x) {
  uint32_t d;
  asm("shr.u32 %0, %1, %2;" : "=r"(d) : "r"(x), "n"(N));
  return d;
}

// (cos d - 1) / d^2 and sin(d) / d as linear functions of d^2 on |d| <= pi / 1024 (csrc/fit_coefficients.py:
// 1.5e-19 and 2.8e-16 absolute on cos d, sin d), the angle scale C = 2 pi 2^-32 and (1/2 - 2^21) C, and
// (log1p(r) / r - 1) / r of degree 3 on |r| <= 2^-9 (6e-16 relative to log1p r), ln 2 and 2.  In constant
// memory: a DFMA reads it as an operand (a 64-bit literal costs two moves per use).
__constant__ double C_BMTRIG[6] = {-0.4999999999999846, 0.04166665359389469, 0.9999999999999077,
                                   -0.16666658823003866, 1.4629180792671596e-09, -0.0030679608443122427};
__constant__ double C_LOG1P[6] = {-0.49999999999969563, 0.33333333333307247, -0.2500006370268452,
                                  0.20000054602306092, 0.6931471805599453, 2.0};

// cos(2 pi u), sin(2 pi u) for u = (w + 1/2) 2^-32: the top 10 bits of w pick the table angle a_i, the low
// 22 bits are the remainder d = 2 pi (low - 2^21 + 1/2) 2^-32, |d| <= pi / 1024, and
// cos(a + d) = cos a + (cos a (cos d - 1) - sin a sin d),  sin(a + d) = sin a + (sin a (cos d - 1) + cos a sin d).
__device__ __forceinline__ void sincos_2pi_u_f64(uint32_t w, double* sn, double* cs) {
  const double2 t = s_noise[shr_opaque<32 - CIRCLE_BITS>(w)];
  const uint32_t low = w & ((1u << (32 - CIRCLE_BITS)) - 1u);
  const double d = __fma_rn(static_cast<double>(low), C_BMTRIG[4], C_BMTRIG[5]);
  const double d2 = __dmul_rn(d, d);
  const double cm1 = __dmul_rn(d2, __fma_rn(d2, C_BMTRIG[1], C_BMTRIG[0]));
  const double sd = __dmul_rn(d, __fma_rn(d2, C_BMTRIG[3], C_BMTRIG[2]));
  *cs = __fma_rn(-t.y, sd, __fma_rn(t.x, cm1, t.x));
  *sn = __fma_rn(t.x, sd, __fma_rn(t.y, cm1, t.y));
}

// ln u for u = (w + 1/2) 2^-32 = k 2^-33, k = 2w + 1 = m 2^e, m in [1, 2): the table entry nearest to m gives
// r = m / c - 1 = fma(m, rc, -1), |r| <= 2^-9, and ln m = -ln rc + log1p(r), log1p(r) = r (1 + r g(r)).
// For c >= 1.412 the entry holds -ln rc - ln 2 and e counts one more (m taken as m / 2 in [0.706, 1)), so
// that e ln 2 and ln m never cancel as u -> 1; the last entry, c = 2, has rc = 1/2 and 0 exactly, and
// ln u keeps its relative accuracy where it is smallest.
__device__ __forceinline__ double ln_uniform_f64(uint32_t w) {
  const double kd = __fma_rn(static_cast<double>(w), C_LOG1P[5], 1.0);  // exact, < 2^33
  const int hi = __double2hiint(kd);
  const int mant = hi & 0x000fffff;
  const uint32_t i = shr_opaque<12>(static_cast<uint32_t>(mant) + 0x800u);  // round(256 (m - 1)), 0 .. 256
  const double m = __hiloint2double(mant | 0x3ff00000, __double2loint(kd));
  const double2 t = s_noise[CIRCLE_N + i];
  const double r = __fma_rn(m, t.x, -1.0);
  double g = C_LOG1P[3];
#pragma unroll
  for (int q = 2; q >= 0; --q) g = __fma_rn(g, r, C_LOG1P[q]);
  const double p = __fma_rn(g, r, 1.0);                                 // log1p(r) / r
  // exponent, one more where i >= LOG_ADJ_FROM, i.e. mant >= (LOG_ADJ_FROM << 12) - 0x800: as a carry out of the
  // mantissa field (three ALU instructions; the comparison cost a predicated move on the FMA pipe)
  const double E = static_cast<double>(((hi + (0x100000 - ((LOG_ADJ_FROM << 12) - 0x800))) >> 20) - (1023 + 33));
  return __fma_rn(E, C_LOG1P[4], __fma_rn(r, p, t.y));
}

__device__ __forceinline__ double rsqrt_approx_f64(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));  // MUFU.RSQ64H: ~2^-21 from the high word of x
  return y;
}
// sqrt(a) for a normal positive a: coupled Newton iteration on g -> sqrt a, h -> 1 / (2 sqrt a) from the
// hardware seed, then one residual correction; relative error < 1 ulp (2^-21 -> 3e-13 -> rounding).
__device__ __forceinline__ double sqrt_pos_f64(double a) {
  const double y = rsqrt_approx_f64(a);
  const double g0 = __dmul_rn(a, y), h0 = __dmul_rn(0.5, y);
  const double r0 = __fma_rn(-g0, h0, 0.5);
  const double g1 = __fma_rn(g0, r0, g0), h1 = __fma_rn(h0, r0, h0);
  return __fma_rn(__fma_rn(-g1, g1, a), h1, g1);
}

struct Normal2d {
  double rho, cs, sn;
  static constexpr bool NEGATED = false;
};

__device__ __forceinline__ double uniform_f64(uint32_t w) {
  return __fma_rn(static_cast<double>(w), 0x1p-32, 0x1p-33);  // (w + 0.5) 2^-32, exact
}

__device__ __forceinline__ Normal2d box_muller_f64(uint32_t wa, uint32_t wb, double sigma) {
  Normal2d o;
  o.rho = __dmul_rn(sigma, sqrt_pos_f64(__dmul_rn(-2.0, ln_uniform_f64(wa))));
  sincos_2pi_u_f64(wb, &o.sn, &o.cs);
  return o;
}

// ---------------------------------------------------------------------------------------------
// S3  force  -U'(x) + F0 (+ tilt folded into k0t by the caller):  one cosine per evaluation,
// cos 2th = 2 cos^2 th - 1  (Eq. 3).
//
// fp32: th = th_s x + th_o in radians goes to MUFU.COS through the range-scale multiply ptxas puts
// in front of it: two roundings at the magnitude of th, up to ~2.4e-6 rad for |x| ~ 3 L in fast
// mode; in precise mode x is a small offset and thb the angle of the fixed-point part (S4).
// ---------------------------------------------------------------------------------------------
template <bool PRECISE>
__device__ __forceinline__ float force(const Coef<float>& k, float x, float k0t, float thb) {
  const float c = fast_cos(__fmaf_rn(x, k.th_s, PRECISE ? thb : k.th_o));
  return __fmaf_rn(__fmaf_rn(k.k2, c, k.k1), c, k0t);
}
template <bool PRECISE>
__device__ __forceinline__ double force(const Coef<double>& k, double x, double k0t, double) {
  const double c = cospi_f64(__fma_rn(x, k.th_s, k.th_o));
  return __fma_rn(__fma_rn(k.k2, c, k.k1), c, k0t);
}

__device__ __forceinline__ float fma_(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double fma_(double a, double b, double c) { return __fma_rn(a, b, c); }
__device__ __forceinline__ float mul_(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ float add_(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ double add_(double a, double b) { return __dadd_rn(a, b); }

// ---------------------------------------------------------------------------------------------
// S4  one step.  k0t = k0 + A cos(omega t_n), k0t1 = k0 + A cos(omega t_{n+1}) (Heun only);
// (rho, cs) = noise of this step, sigma z = rho * cs.
//
// Euler-Maruyama (all right-hand sides at the old state, reading G4):
//   x' = x + dt v;  v' = v + dt a_v + sigma z;  e' = e + dt a_e
//   a_v = (d e - gamma0) v + f(x),   a_e = q - e (c + d v^2)             (Eqs. 2, 1)
// The increments are added to the state unscaled (no pre-multiplied (1 - gamma0 dt) factors):
// a rounded factor next to 1 would bias every step in the same direction.
// ---------------------------------------------------------------------------------------------
//
// Precise fp32 mode: what limits the 100-step agreement with the fp64
// oracle is rounding at the magnitude of the unwrapped position -- of the angle 2 pi (x + phi) / L
// and of x' = x + dt v (the error random-walks and is amplified each step by dt U'').  Here the
// position is split as  X L 2^-32 + x:
//   * X = xc 2^32 + xf, a 64-bit fixed-point number of periods (resolution 2.3e-10 L), changed only
//     by exact integer additions;
//   * x, a float offset that starts at 0 and collects the increments of at most four steps, so it
//     is rounded at the magnitude of a few dt v (ulp ~ 1e-9 L), not of the position.
// After every step whose global index is 3 mod 4 (the end of a Philox block on the fast path; the
// single-step path applies the same rule, so split launches stay bit-identical) fold() moves the
// offset into X: rni(x 2^32 / L) by one F2I, IADD3 + IADD3.X, and recomputes thb, the angle of the
// fraction word (I2F of the signed word: relative 2^-25 of at most half a period).  The force is
// then cos(thb + (2 pi / L) x): the same FFMA as in fast mode with thb in place of the phase.
// Cost over fast mode: 2 FP32 + 1 F2I + 1 I2F + 2 integer adds per FOUR steps, two more words of
// state.  (A float -> integer conversion per step would be cheaper on the FMA port but runs at MUFU
// rate on the pipe the cosines already keep 60 % busy.)  The conversion is 64 bits wide, so the offset of
// four steps may be any number of periods.
__device__ __forceinline__ float fixed_angle(uint32_t xf, float th_o) {
  // 2 pi 2^-32 * (signed fraction) + phase
  return __fmaf_rn(static_cast<float>(static_cast<int32_t>(xf)), 1.4629180792671596e-09f, th_o);
}
__device__ __forceinline__ void fold(State<float>& s, const Coef<float>& k) {
  // 64-bit conversion: any offset is legal (a 32-bit one would saturate silently at |offset| >= L / 2)
  const int64_t d = __float2ll_rn(__fmul_rn(s.x, k.fxS));
  const int64_t X = ((static_cast<int64_t>(s.xc) << 32) | s.xf) + d;
  s.xf = static_cast<uint32_t>(X);
  s.xc = static_cast<int32_t>(X >> 32);
  s.x = 0.0f;
  s.thb = fixed_angle(s.xf, k.th_o);
}
__device__ __forceinline__ void fold(State<double>&, const Coef<double>&) {}
// The position the ABI exposes (frames, moments, raster) in precise mode, in fp32:
// X rounded to 24 bits by the conversion, times L 2^-32, plus the offset (one FMA).
__device__ __forceinline__ float position_fixed(uint32_t xf, int32_t xc, float x, float L) {
  const long long X = (static_cast<long long>(xc) << 32) | xf;
  return __fmaf_rn(__ll2float_rn(X), __fmul_rn(L, 0x1p-32f), x);
}
// x[k] of the state arrays as a position (xl == nullptr: the x array holds positions; else the x
// array holds the offset and the xl / xh arrays the bits of xf / xc)
__device__ __forceinline__ float load_position(const float* x, const float* xl, const float* xh,
                                               uint64_t k, float L) {
  return xl ? position_fixed(__float_as_uint(xl[k]), __float_as_int(xh[k]), x[k], L) : x[k];
}
__device__ __forceinline__ double load_position(const double* x, const double*, const double*,
                                                uint64_t k, double) {
  return x[k];
}

// Order of the sums: cos -> f -> a_v -> v + dt a_v -> + noise, five dependent FMAs from the cosine to the new
// velocity.  Adding everything that does not wait for the cosine first (h = (d e - gamma0) v + k0t as the
// constant term of the force polynomial, the noise increment onto v before dt a_v) leaves three and shortens the
// recurrence v_n -> x_{n+1} -> cos -> v_{n+2} that bounds small ensembles from 27.2 to 22.9 clocks per step
// (csrc/pipe_rates.cu, last table); measured on the kernels: step_kernel_small 0.192 -> 0.185 ms per 10^4 steps
// (config[0]), but the throughput-bound loop of config[1] 22.31 -> 22.85 ms per 20,000 steps (the same
// instruction count, a worse ptxas schedule), config[2] 8.87 -> 8.99.  Both kernels must execute the same
// arithmetic (a trajectory does not depend on which kernel ran), and config[1] is the headline: not taken.
template <bool PRECISE, typename Real>
__device__ __forceinline__ void em_step(State<Real>& s, const Coef<Real>& k, Real k0t, Real rho,
                                        Real cs) {
  const Real f = force<PRECISE>(k, s.x, k0t, s.thb);
  const Real av = fma_(fma_(k.d, s.e, -k.gamma0), s.v, f);
  const Real ae = fma_(-s.e, fma_(k.d, mul_(s.v, s.v), k.c), k.q);
  s.x = fma_(k.dt, s.v, s.x);
  s.v = fma_(rho, cs, fma_(k.dt, av, s.v));
  s.e = fma_(k.dt, ae, s.e);
}

// Stochastic Heun: predictor = EM step with the full noise increment; corrector averages the
// drift at (X, t_n) and (X~, t_{n+1}); the same sigma z in both (reading G16).
// v' is rounded ONCE at the magnitude of v (the increment is summed first).  The cheaper corrector
// v' = v~ + (dt/2)(a2 - a1) on a predictor built as in em_step (two instructions less per step) rounds three
// times at that magnitude; on a stiff potential (config[3]'s model with L = 0.5: dt max U'' = 1.6) the
// instability of the dynamics amplifies the difference to 1.2e-5 after 100 steps against 8.7e-6 (measured).
template <bool PRECISE, typename Real>
__device__ __forceinline__ void heun_step(State<Real>& s, const Coef<Real>& k, Real k0t, Real k0t1,
                                          Real rho, Real cs) {
  const Real sz = mul_(rho, cs);
  const Real f1 = force<PRECISE>(k, s.x, k0t, s.thb);
  const Real av1 = fma_(fma_(k.d, s.e, -k.gamma0), s.v, f1);
  const Real ae1 = fma_(-s.e, fma_(k.d, mul_(s.v, s.v), k.c), k.q);
  const Real xp = fma_(k.dt, s.v, s.x);
  const Real vp = add_(s.v, fma_(k.dt, av1, sz));
  const Real ep = fma_(k.dt, ae1, s.e);
  const Real f2 = force<PRECISE>(k, xp, k0t1, s.thb);
  const Real av2 = fma_(fma_(k.d, ep, -k.gamma0), vp, f2);
  const Real ae2 = fma_(-ep, fma_(k.d, mul_(vp, vp), k.c), k.q);
  s.x = fma_(k.hdt, add_(s.v, vp), s.x);
  s.v = add_(s.v, fma_(k.hdt, add_(av1, av2), sz));  // one rounding at the magnitude of v
  s.e = fma_(k.hdt, add_(ae1, ae2), s.e);
}

// ---------------------------------------------------------------------------------------------
// S0  initial state from the init block: x0 = L u(w0) with the run's position map,
// v0 constant or sv * sqrt(-2 ln u(w2)) cos(2 pi u(w3)), e0 constant; w1 reserved.
// Not on the hot loop: precise functions.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ float init_x(const Coef<float>& k, uint32_t w0) {
  return __fmul_rn(k.L, __fmul_rn(static_cast<float>(w0 >> 8), 0x1p-24f));
}
__device__ __forceinline__ double init_x(const Coef<double>& k, uint32_t w0) {
  return __dmul_rn(k.L, __dmul_rn(static_cast<double>(w0), 0x1p-32));
}
__device__ __forceinline__ float init_v_thermal(const Coef<float>& k, uint32_t w2, uint32_t w3) {
  const float r = sqrtf(-2.0f * logf(uniform_f32(w2)));
  return k.sv * r * cospif(2.0f * uniform_f32(w3));
}
__device__ __forceinline__ double init_v_thermal(const Coef<double>& k, uint32_t w2, uint32_t w3) {
  const double r = sqrt(-2.0 * log(uniform_f64(w2)));
  return k.sv * r * cospi(2.0 * uniform_f64(w3));
}

}  // namespace abm
