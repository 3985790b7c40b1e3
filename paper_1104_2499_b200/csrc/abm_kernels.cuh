// abm_kernels.cuh -- the kernels of the hot path (sm_100a): init (S0), step (S1-S5, S7),
// snapshot (S5), moments (S6), tilt table and the Philox diagnostic.
#pragma once
#include "abm_device.cuh"

namespace abm {

#ifndef ABM_STEP_BLOCK
#define ABM_STEP_BLOCK 128
#endif
// Resident CTAs per SM of the step kernel (the register cap follows: 65,536 / (128 * n)), per
// kernel family.  The loop is throughput-bound from four warps per scheduler on
// (profiles/r01_scaling.md: no wave quantisation, a partly filled wave runs proportionally
// faster), so occupancy is chosen for the code ptxas produces under the cap -- no spills, few
// moves -- not for latency hiding.
// Measured on B200 (round-1 sweeps, particle-steps/s): fp32 EM one set, final loop of the round (20,000 steps of
// config[1]): 5: 22.32 ms < 3 ~ 4: 22.47 < 6 ~ 8: 22.50 < 7 ~ 10: 22.91 < 12: 23.22;
// fp32 Heun 5 ~ 4 > 6 > 8; fp32 with per-thread coefficients 4 > 6 > 8 > 12 (12 spilled 236 B);
// fp64 (final loop of the round, 2,000 steps of config[4]): 5: 27.51 ms ~ 4: 27.63 < 3: 28.17 < 7: 28.28
// < 6: 28.54 < 8: 28.75 (16 B of stack per thread in the loop); 12 spilled > 1 KB.
#ifndef ABM_MINB_F32U
#define ABM_MINB_F32U 5   // fp32 Euler-Maruyama, one parameter set (uniform coefficients): <= 96 regs (ptxas takes 62)
#endif
#ifndef ABM_MINB_F32H
#define ABM_MINB_F32H 5   // fp32 Heun, one parameter set: <= 96 regs
#endif
#ifndef ABM_MINB_F32N
#define ABM_MINB_F32N 4   // fp32, per-thread coefficient record (config[2]): <= 128 regs
#endif
#ifndef ABM_MINB_F32S
#define ABM_MINB_F32S 5   // fp32, sweep over D, q, F0, A only (config[2]): <= 96 regs
#endif
#ifndef ABM_MINB_F64
#define ABM_MINB_F64 5    // fp64: <= 96 regs (ptxas takes 86: no stack traffic in the loop)
#endif
constexpr int STEP_BLOCK = ABM_STEP_BLOCK;   // threads per CTA of the step kernel
// Where a thread's coefficient record comes from.
//   COEF_PER_THREAD   the whole record loaded per thread from the table into vector registers (any sweep)
//   COEF_PARAM        one parameter set: the record is a kernel parameter (constant-bank operands)
//   COEF_SPLIT        a sweep whose sets differ only in D, q, F0, A (noise level, pumping rate, load force, tilt
//                     amplitude: what the paper, and BASELINE.json configs[2] sweep): the
//                     coefficients those decide -- s2, q, k0, A -- are loaded per thread, all others are the
//                     kernel-parameter record of set 0, as in COEF_PARAM.  The same intrinsics on the same
//                     values as COEF_PER_THREAD: bit-identical results, fewer registers and no round-key
//                     reloads in the loop.
enum { COEF_PER_THREAD = 0, COEF_PARAM = 1, COEF_SPLIT = 2 };
template <typename Real, int INTEG, int COEF>
constexpr int step_min_blocks() {
  return sizeof(Real) == 8 ? ABM_MINB_F64
                           : (COEF == COEF_PER_THREAD ? ABM_MINB_F32N
                              : COEF == COEF_SPLIT    ? ABM_MINB_F32S
                                                      : (INTEG == 1 ? ABM_MINB_F32H : ABM_MINB_F32U));
}
constexpr int MOM_BLOCK = 256;    // threads per CTA of the moment reduction (max)
constexpr int MOM_PER_THREAD = 16;
constexpr int N_SUMS = 8;

template <typename Real>
struct StepArgs {
  Real* x;
  Real* v;
  Real* e;
  Real* xl;                      // PRECISE: bits of xf, the fraction word of the fixed-point position
  Real* xh;                      // PRECISE: bits of xc, its whole periods (else both nullptr)
  const Coef<Real>* coef_table;  // [n_sets] (used when !UNIFORM)
  const Real* tilt;              // tilt[j] = k0 + A cos(omega (tilt_base + j) dt): (k0, A) of the one set, or (0, 1);
                                 // tilt_base is a multiple of 4 and tilt + INTEG is 16-byte aligned (TiltCursor)
  void* snap;                    // bound snapshot buffer or nullptr
  uint4* rng_state;              // xorshift state per trajectory (used when XS), at a pair boundary
  uint64_t n_traj;               // local trajectories
  uint64_t n_particles;          // per set
  uint64_t traj_base, set_stride;
  uint64_t set_magic;            // ceil(2^64 / n_particles) (set_magic_of)
  uint64_t seed;
  uint64_t step0;                // first global step of this launch
  uint64_t tilt_base;            // global step of tilt[0]
  uint32_t n_steps;              // steps in this launch
  uint32_t snap_every;           // K (0 = never)
  uint32_t snap_stride;          // bytes per trajectory in snap
  uint32_t traj_hi;              // high word of every global trajectory index, if shared
  uint32_t traj_hi_shared;       // 1: all trajectories of the launch share traj_hi
  uint32_t rk0[10], rk1[10];     // Philox round keys k0 + r W0, k1 + r W1 (host-computed: constant-bank operands)
  const double2* noise_tables;   // fp64: circle and log tables of the Box-Muller transform (NoiseTables), else nullptr
  Coef<Real> coef0;              // the single set's coefficients (used when UNIFORM)
};

// ---------------------------------------------------------------------------------------------
// index helpers
// ---------------------------------------------------------------------------------------------
struct TrajId {
  uint64_t global;  // index into the random stream
  uint32_t set;
};
// global index and set of local trajectory k, with a plain division (kernels that run once)
__device__ __forceinline__ TrajId traj_id_div(uint64_t k, uint64_t n_particles, uint64_t traj_base,
                                              uint64_t set_stride, bool single_set) {
  TrajId t;
  const uint64_t s = single_set ? 0 : k / n_particles;
  t.set = static_cast<uint32_t>(s);
  t.global = traj_base + s * set_stride + (k - s * n_particles);
  return t;
}
// The step kernels: k / n_particles without the 64-bit division subroutine: set_magic = ceil(2^64 / n_particles) from the host
// (0 stands for 2^64, i.e. n_particles = 1), one high multiply and a correction (the estimate is never low and
// at most one too high).  A CALL in the step kernels' prologue makes ptxas reload every uniform register --
// round keys and coefficients -- inside the hot loop (12 LDCU per trip measured).
__host__ __device__ inline uint64_t set_magic_of(uint64_t n_particles) {
  return n_particles > 1 ? ~0ull / n_particles + 1 : 0;
}
__device__ __forceinline__ uint64_t set_of(uint64_t k, uint64_t n_particles, uint64_t set_magic) {
  if (set_magic == 0) return k;
  uint64_t s = __umul64hi(k, set_magic);
  if (s * n_particles > k) --s;
  return s;
}
__device__ __forceinline__ TrajId traj_id(uint64_t k, uint64_t n_particles, uint64_t traj_base,
                                          uint64_t set_stride, bool single_set, uint64_t set_magic) {
  TrajId t;
  if (single_set) {
    t.set = 0;
    t.global = traj_base + k;
  } else {
    const uint64_t s = set_of(k, n_particles, set_magic);
    t.set = static_cast<uint32_t>(s);
    t.global = traj_base + s * set_stride + (k - s * n_particles);
  }
  return t;
}

// ---------------------------------------------------------------------------------------------
// S5  snapshot store: float2 (x, v) / float4 (x, v, e, 1) per trajectory, thread-contiguous so
// a warp writes 256 / 512 contiguous bytes (the headless stand-in for the GL vertex buffer,
// PAPER.md:158-162).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void store_snapshot(void* snap, uint32_t stride, uint64_t k,
                                               const State<float>& s) {
  if (stride == 8) {
    reinterpret_cast<float2*>(snap)[k] = make_float2(s.x, s.v);
  } else {
    reinterpret_cast<float4*>(snap)[k] = make_float4(s.x, s.v, s.e, 1.0f);
  }
}
__device__ __forceinline__ void store_snapshot(void* snap, uint32_t stride, uint64_t k,
                                               const State<double>& s) {
  if (stride == 16) {
    reinterpret_cast<double2*>(snap)[k] = make_double2(s.x, s.v);
  } else {
    reinterpret_cast<double4*>(snap)[k] = make_double4(s.x, s.v, s.e, 1.0);
  }
}

template <typename Real>
__global__ void snapshot_kernel(const Real* __restrict__ x, const Real* __restrict__ v,
                                const Real* __restrict__ e, const Real* __restrict__ xl,
                                const Real* __restrict__ xh,
                                const Coef<Real>* __restrict__ coef_table, uint64_t n_traj,
                                uint64_t n_particles, uint32_t n_sets, void* snap, uint32_t stride) {
  const uint64_t k = static_cast<uint64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (k >= n_traj) return;
  const uint32_t set = n_sets == 1 ? 0u : static_cast<uint32_t>(k / n_particles);
  State<Real> s{load_position(x, xl, xh, k, coef_table[set].L), v[k], e[k], Real(0), 0u, 0, Real(0)};
  store_snapshot(snap, stride, k, s);
}

// ---------------------------------------------------------------------------------------------
// S0  init
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void store_fixed(float* xl, float* xh, uint64_t k, uint32_t xf, int32_t xc) {
  xl[k] = __uint_as_float(xf);
  xh[k] = __int_as_float(xc);
}
__device__ __forceinline__ void store_fixed(double*, double*, uint64_t, uint32_t, int32_t) {}

template <typename Real>
__global__ void init_kernel(Real* __restrict__ x, Real* __restrict__ v, Real* __restrict__ e,
                            const Coef<Real>* __restrict__ coef_table, uint64_t n_traj,
                            uint64_t n_particles, uint64_t traj_base, uint64_t set_stride,
                            uint64_t seed, uint32_t n_sets, uint32_t init_v,
                            uint4* __restrict__ rng_state, Real* __restrict__ xl,
                            Real* __restrict__ xh) {
  const uint64_t k = static_cast<uint64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (k >= n_traj) return;
  const TrajId id = traj_id_div(k, n_particles, traj_base, set_stride, n_sets == 1);
  if (rng_state) rng_state[k] = xorshift_seed(seed, id.global);
  const Coef<Real> c = coef_table[id.set];
  const uint4 w = philox_block(seed, id.global, INIT_BLOCK);
  if (xl) {  // precise fp32 mode: X = x0 2^32 / L = (w0 >> 8) << 8 exactly, offset 0
    store_fixed(xl, xh, k, w.x & 0xffffff00u, 0);
    x[k] = Real(0);
  } else {
    x[k] = init_x(c, w.x);
  }
  v[k] = init_v ? init_v_thermal(c, w.z, w.w) : c.v0;
  e[k] = c.e0;
}

// ---------------------------------------------------------------------------------------------
// tilt table: tilt[j] = k0 + A cos(omega * ((base + j) * dt)), evaluated in fp64 (reading G15).
// Single-set runs pass the set's (k0, A): the table then holds the whole time-dependent constant of
// the force and the step kernel adds nothing; sweeps pass (0, 1) and apply each set's A, k0 themselves.
// ---------------------------------------------------------------------------------------------
template <typename Real>
__global__ void tilt_kernel(Real* __restrict__ tilt, uint64_t base, uint32_t n, double omega,
                            double dt, double k0, double A) {
  const uint32_t j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  const double t = static_cast<double>(base + j) * dt;
  tilt[j] = static_cast<Real>(k0 + A * cos(omega * t));  // (k0, A) = (0, 1): the cosine itself
}

// ---------------------------------------------------------------------------------------------
// The step kernel.  One trajectory per thread; the state lives in registers for the whole
// launch ("fill local memory with parameters ... for i = 0 to T ... assign local
// parameters to global memory").  One Philox block feeds four steps: words (0,1) -> steps
// 4b, 4b+1 (cos, sin), words (2,3) -> steps 4b+2, 4b+3.
// ---------------------------------------------------------------------------------------------
template <typename Real>
struct Noise4;
template <>
struct Noise4<float> {
  static constexpr float SIGN = Normal2f::NEGATED ? -1.0f : 1.0f;
  Normal2f a, b;
  __device__ __forceinline__ Noise4(const uint4& w, const Coef<float>& k, const NoiseTables<float>& = {})
      : a(box_muller_f32(w.x, w.y, k.s2, k.bm_o)), b(box_muller_f32(w.z, w.w, k.s2, k.bm_o)) {}
  __device__ __forceinline__ Noise4(const Normal2f& a_, const Normal2f& b_) : a(a_), b(b_) {}
};
template <>
struct Noise4<double> {
  static constexpr double SIGN = Normal2d::NEGATED ? -1.0 : 1.0;
  Normal2d a, b;
  __device__ __forceinline__ Noise4(const uint4& w, const Coef<double>& k, const NoiseTables<double>&)
      : a(box_muller_f64(w.x, w.y, k.s2)), b(box_muller_f64(w.z, w.w, k.s2)) {}
};

template <typename Real, int INTEG, int TILT, bool PRECISE>
__device__ __forceinline__ void one_step(State<Real>& s, const Coef<Real>& k, Real rho, Real cs,
                                         Real t0, Real t1) {
  // TILT == 2: the table holds k0 + A cos(omega t) itself (single-set runs, fp64 on the host side of
  // the rounding); TILT == 1: it holds cos(omega t) and the set's A, k0 are applied here.
  const Real k0t = TILT == 2 ? t0 : (TILT ? fma_(k.A, t0, k.k0) : k.k0);
  if (INTEG == 0) {
    em_step<PRECISE>(s, k, k0t, rho, cs);
  } else {
    const Real k0t1 = TILT == 2 ? t1 : (TILT ? fma_(k.A, t1, k.k0) : k.k0);
    heun_step<PRECISE>(s, k, k0t, k0t1, rho, cs);
  }
}

// The tilt values of the coming four steps (TILT != 0): t_n ... t_{n+3} for Euler-Maruyama, and t_{n+4} too for
// Heun, whose corrector evaluates the force at t_{n+1}.  One 16-byte load per Philox block (fp64: two) from an
// address every thread of the launch shares: the host places the table so that what a block loads is 16-byte
// aligned whenever n is a multiple of 4 (step_impl: the table starts at a multiple of four steps, shifted by one
// element for Heun, whose first value of a block is the last one of the block before and is carried in a register).
template <typename Real, int INTEG>
struct TiltCursor {
  const Real* p = nullptr;
  Real carry = 0;
  __device__ __forceinline__ void start(const Real* q) {
    p = q;
    if (INTEG == 1) carry = q[0];
  }
  __device__ __forceinline__ void next4(Real& t0, Real& t1, Real& t2, Real& t3, Real& t4) {
    if constexpr (sizeof(Real) == 4) {
      const float4 q = *reinterpret_cast<const float4*>(p + INTEG);
      if (INTEG == 1) { t0 = carry; t1 = q.x; t2 = q.y; t3 = q.z; t4 = q.w; carry = q.w; }
      else { t0 = q.x; t1 = q.y; t2 = q.z; t3 = q.w; }
    } else {
      const double2 q = *reinterpret_cast<const double2*>(p + INTEG);
      const double2 r = *reinterpret_cast<const double2*>(p + INTEG + 2);
      if (INTEG == 1) { t0 = carry; t1 = q.x; t2 = q.y; t3 = r.x; t4 = r.y; carry = r.y; }
      else { t0 = q.x; t1 = q.y; t2 = r.x; t3 = r.y; }
    }
    p += 4;
  }
};
// elements in front of the table so that (table + INTEG) is 16-byte aligned
template <typename Real>
__host__ __device__ constexpr uint32_t tilt_table_shift(int integ) {
  return integ == 1 ? (sizeof(Real) == 4 ? 3u : 1u) : 0u;
}

// Four steps from the noise of one Philox block.
template <typename Real, int INTEG, int TILT, bool PRECISE>
__device__ __forceinline__ void four_steps_z(State<Real>& s, const Coef<Real>& cf,
                                             const Noise4<Real>& z, TiltCursor<Real, INTEG>& tl) {
  Real t0 = 0, t1 = 0, t2 = 0, t3 = 0, t4 = 0;
  if (TILT) tl.next4(t0, t1, t2, t3, t4);
  const Real ra = Noise4<Real>::SIGN * z.a.rho, rb = Noise4<Real>::SIGN * z.b.rho;
  one_step<Real, INTEG, TILT, PRECISE>(s, cf, ra, z.a.cs, t0, t1);
  one_step<Real, INTEG, TILT, PRECISE>(s, cf, ra, z.a.sn, t1, t2);
  one_step<Real, INTEG, TILT, PRECISE>(s, cf, rb, z.b.cs, t2, t3);
  one_step<Real, INTEG, TILT, PRECISE>(s, cf, rb, z.b.sn, t3, t4);
  if constexpr (PRECISE) fold(s, cf);  // after the step with global index 3 mod 4
}
// Four steps from one Philox block.
template <typename Real, int INTEG, int TILT, bool PRECISE>
__device__ __forceinline__ void four_steps(State<Real>& s, const Coef<Real>& cf, const uint4& w,
                                           TiltCursor<Real, INTEG>& tl, const NoiseTables<Real>& nt) {
  const Noise4<Real> z(w, cf, nt);
  four_steps_z<Real, INTEG, TILT, PRECISE>(s, cf, z, tl);
}

// The state as a frame shows it: in precise mode x is the remainder, the frame wants the position.
template <bool PRECISE, typename Real>
__device__ __forceinline__ State<Real> frame_state(const State<Real>& s, const Coef<Real>& cf) {
  State<Real> o = s;
  if constexpr (PRECISE) o.x = position_fixed(s.xf, s.xc, s.x, cf.L);
  return o;
}

// The step loop of one trajectory.
//
// TABLE (the whole launch shares traj_hi, the high word of the global trajectory index = Philox
// counter word 3): the half of the first two Philox rounds that depends only on the block index --
// two of the 20 multiplies -- is the same for every trajectory, so each CTA computes it once per
// block into a shared-memory table (PHILOX_CHUNK blocks per refill, one entry per thread, double
// buffered: one __syncthreads per refill) and every thread fetches its entry with one broadcast
// LDS.128.  Two more multiplies depend only on the trajectory and are done once per run.  16
// IMAD.WIDE per block remain per thread.  IMAD.WIDE runs at a quarter of the FFMA rate on the
// FFMA dispatch port (profiles/r01_pipe_rates.txt), so multiplies are what this loop is short of.
// All threads of a CTA execute the same loop (bounds are launch-uniform); threads past the end of
// the ensemble integrate a copy of the last trajectory and store nothing (`active`).
//
// Software pipeline: the Philox block of the NEXT four steps is computed next to the
// floating-point work of the current four, so every warp issues a steady mix of IMAD.WIDE / LOP3
// and FFMA / MUFU instead of an integer phase followed by a floating-point phase.  The block
// after the last one of a run is computed and dropped (its counter may wrap: harmless).
constexpr int PHILOX_CHUNK = STEP_BLOCK;  // table entries per refill = threads per CTA
#ifndef ABM_UNROLL2
#define ABM_UNROLL2 1
#endif
#ifndef ABM_UNROLL2_F64
#define ABM_UNROLL2_F64 1
#endif
#ifndef ABM_RK_CONST
#define ABM_RK_CONST 1
#endif
#if ABM_RK_CONST
#define PHILOX_FINISH(pt, u, a, k0, k1) philox_finish_rk(pt, (u).x, (u).y, (u).z, (a).rk0, (a).rk1)
#else
#define PHILOX_FINISH(pt, u, a, k0, k1) philox_finish(pt, (u).x, (u).y, (u).z, k0, k1)
#endif

//
// XS (generator variant, NEXT-4): the words come from the trajectory's xorshift state S instead.
// S always sits at a pair boundary -- before output 2 (n >> 1) -- when a step starts: whole blocks
// draw four outputs; a single even step draws its pair from a copy, the odd step after it commits.
//
// BODY: what is done with the words.  The step kernels integrate (Integrate: four steps per block, one step
// on the slow path, a frame where one is due); the stream diagnostic (philox_loop_kernel, abm_philox_blocks_loop)
// stores them (DumpWords) -- it instantiates THIS function, so the words it shows are produced by the
// instructions the step kernels execute: philox_traj, the double-buffered block-head table, philox_finish_rk
// with the host-computed round keys, two blocks per trip in fp32.
template <typename Real, int INTEG, int TILT, bool PRECISE>
struct Integrate {
  const StepArgs<Real>& a;
  const Coef<Real>& cf;
  State<Real>& s;
  const uint64_t k;
  const bool active;
  const NoiseTables<Real> nt;
  TiltCursor<Real, INTEG> tl;
  __device__ __forceinline__ Integrate(const StepArgs<Real>& a_, const Coef<Real>& cf_, State<Real>& s_,
                                       uint64_t k_, bool active_, const NoiseTables<Real>& nt_)
      : a(a_), cf(cf_), s(s_), k(k_), active(active_), nt(nt_) {}
  // a run of whole blocks starts at step n (a multiple of 4)
  __device__ __forceinline__ void start(uint64_t n) {
    if (TILT) tl.start(a.tilt + (n - a.tilt_base));
  }
  __device__ __forceinline__ void block(const uint4& w) {
    four_steps<Real, INTEG, TILT, PRECISE>(s, cf, w, tl, nt);
  }
  // step n alone; w holds the words of its pair where the block layout has them
  __device__ __forceinline__ void single(const uint4& w, uint64_t n) {
    const Noise4<Real> z(w, cf, nt);
    const bool second = (n >> 1) & 1u;
    const Real rho = Noise4<Real>::SIGN * (second ? z.b.rho : z.a.rho);
    const Real cs = (n & 1u) ? (second ? z.b.sn : z.a.sn) : (second ? z.b.cs : z.a.cs);
    Real t0 = 0, t1 = 0;
    if (TILT) {
      t0 = a.tilt[n - a.tilt_base];
      if (INTEG == 1) t1 = a.tilt[n - a.tilt_base + 1];
    }
    one_step<Real, INTEG, TILT, PRECISE>(s, cf, rho, cs, t0, t1);
    if constexpr (PRECISE) {
      if ((n & 3u) == 3u) fold(s, cf);  // the same rule as four_steps
    }
  }
  __device__ __forceinline__ void frame() {
    if (active) store_snapshot(a.snap, a.snap_stride, k, frame_state<PRECISE>(s, cf));
  }
};
struct DumpWords {
  uint4* out;  // the next block of this thread's trajectory (nullptr: a shadowing thread, stores nothing)
  __device__ __forceinline__ void start(uint64_t) {}
  __device__ __forceinline__ void block(const uint4& w) {
    if (out) *out++ = w;
  }
  __device__ __forceinline__ void single(const uint4& w, uint64_t n) {
    if (out && (n & 3u) == 0) *out++ = w;
  }
  __device__ __forceinline__ void frame() {}
};

template <typename Real, bool TABLE, bool XS, typename Body>
__device__ __forceinline__ void run_steps(const StepArgs<Real>& a, const uint32_t traj_lo,
                                          const uint32_t traj_hi, Body& body, uint4& S) {
  __shared__ uint4 tab[TABLE ? 2 : 1][TABLE ? PHILOX_CHUNK : 1];
  uint32_t par = 0;
  const uint32_t k0 = static_cast<uint32_t>(a.seed), k1 = static_cast<uint32_t>(a.seed >> 32);
  uint64_t n = a.step0;
  const uint64_t n_end = a.step0 + a.n_steps;
  const uint32_t K = a.snap != nullptr ? a.snap_every : 0u;
  uint64_t next_snap = ~0ull;
  if (K) next_snap = (n / K + 1) * static_cast<uint64_t>(K);

  // Frames fall on Philox-block boundaries when K is a multiple of 4 (n is a multiple of 4 on the
  // fast path): they are then stored from inside the block loop and the software pipeline
  // runs through them.  Otherwise a run of whole blocks ends at the next frame.
  const bool snap_aligned = (K & 3u) == 0;
  while (n < n_end) {
    const uint64_t lim = (snap_aligned || next_snap > n_end) ? n_end : next_snap;
    if ((n & 3u) == 0 && lim - n >= 4) {
      // ---- fast path: whole Philox blocks, four steps each ----
      uint64_t b = n >> 2;
      uint64_t nb64 = (lim - n) >> 2;
      const uint64_t to_wrap = 0x100000000ull - (b & 0xffffffffull);  // keep b's high word fixed
      if (nb64 > to_wrap) nb64 = to_wrap;
      const uint32_t nb = static_cast<uint32_t>(nb64 > 0x40000000ull ? 0x40000000ull : nb64);
      const uint32_t b_hi = static_cast<uint32_t>(b >> 32);
      uint32_t b_lo = static_cast<uint32_t>(b);
      body.start(n);
      uint64_t to_snap = (K && snap_aligned) ? (next_snap - n) >> 2 : ~0ull;  // blocks to the frame
      uint32_t left = nb;
      if (XS) {
        // The look-ahead block is drawn for every block but the last of the run, so that exactly
        // 4 nb outputs are consumed.
        uint4 w = xorshift128_x4(S);
        do {
          const uint32_t seg = left < to_snap ? left : static_cast<uint32_t>(to_snap);  // >= 1
          const bool last = seg == left;
          uint32_t ahead = last ? seg - 1u : seg;  // blocks of this segment with a look-ahead draw
          if constexpr ((sizeof(Real) == 4 || ABM_UNROLL2_F64 != 0) && ABM_UNROLL2 != 0) {  // two blocks per trip, as for Philox
            if (ahead & 1u) {
              const uint4 w_next = xorshift128_x4(S);
              body.block(w);
              w = w_next;
            }
#pragma unroll 1
            for (ahead >>= 1; ahead; --ahead) {
              const uint4 wa = xorshift128_x4(S);
              body.block(w);
              w = xorshift128_x4(S);
              body.block(wa);
            }
          } else {
#pragma unroll 1
            for (; ahead; --ahead) {
              const uint4 w_next = xorshift128_x4(S);
              body.block(w);
              w = w_next;
            }
          }
          if (last) body.block(w);
          left -= seg;
          if (seg == to_snap) {  // a frame is due after this block
            body.frame();
            to_snap = K >> 2;
          } else {
            to_snap -= seg;
          }
        } while (left);
        n += static_cast<uint64_t>(nb) << 2;
        // aligned K: the frames of this run were stored above.  Otherwise the run ended at or before
        // the next frame, which the check at the bottom of the loop stores.
        if (K && snap_aligned) next_snap = (n / K + 1) * static_cast<uint64_t>(K);
      } else {
      uint4 w = philox4x32_10(b_lo, b_hi, traj_lo, traj_hi, k0, k1);
      if (TABLE) {
        const PhiloxTraj pt = philox_traj(traj_lo, b_hi, k0);
        do {
          // refill: entry j belongs to block b_lo + 1 + j (the block the pipeline computes in
          // iteration j of this chunk)
          const PhiloxBlockHead h = philox_block_head(b_lo + 1u + threadIdx.x, traj_hi, k0, k1);
          tab[par][threadIdx.x] = make_uint4(h.u0, h.u1, h.u2, 0u);
          __syncthreads();
          const uint32_t in_chunk = left < static_cast<uint32_t>(PHILOX_CHUNK)
                                        ? left : static_cast<uint32_t>(PHILOX_CHUNK);
          const uint4* tp = tab[par];
          uint32_t done = 0;
          do {
            const uint32_t rest = in_chunk - done;
            const uint32_t seg = rest < to_snap ? rest : static_cast<uint32_t>(to_snap);  // >= 1
            // fp32: two blocks per loop trip -- the look-ahead words alternate between two register
            // sets, so no moves rotate them and the loop overhead is halved (fp64 too since round 2:
            // ABM_UNROLL2_F64 = 1; the one-block branch below is compiled only with -DABM_UNROLL2_F64=0).
            if constexpr ((sizeof(Real) == 4 || ABM_UNROLL2_F64 != 0) && ABM_UNROLL2 != 0) {
              if (seg & 1u) {
                const uint4 u = *tp++;
                const uint4 w_next = PHILOX_FINISH(pt, u, a, k0, k1);
                body.block(w);
                w = w_next;
              }
              const uint4* const tp_end = tp + (seg & ~1u);
#pragma unroll 1
              while (tp != tp_end) {
                const uint4 ua = tp[0];
                const uint4 wa = PHILOX_FINISH(pt, ua, a, k0, k1);
                body.block(w);
                const uint4 ub = tp[1];
                w = PHILOX_FINISH(pt, ub, a, k0, k1);
                body.block(wa);
                tp += 2;
              }
            } else {
              const uint4* const tp_end = tp + seg;
#pragma unroll 1
              do {
                const uint4 u = *tp;
                const uint4 w_next = PHILOX_FINISH(pt, u, a, k0, k1);
                body.block(w);
                w = w_next;
              } while (++tp != tp_end);
            }
            done += seg;
            if (seg == to_snap) {  // a frame is due after this block
              body.frame();
              to_snap = K >> 2;
            } else {
              to_snap -= seg;
            }
          } while (done != in_chunk);
          left -= in_chunk;
          b_lo += in_chunk;
          par ^= 1u;
        } while (left);
      } else {
        do {
          const uint32_t seg = left < to_snap ? left : static_cast<uint32_t>(to_snap);  // >= 1
          const uint32_t seg_end = b_lo + seg;  // may wrap to 0: the loop runs until equality
#pragma unroll 1
          do {
            const uint4 w_next = philox4x32_10(b_lo + 1u, b_hi, traj_lo, traj_hi, k0, k1);
            body.block(w);
            w = w_next;
          } while (++b_lo != seg_end);
          left -= seg;
          if (seg == to_snap) {  // a frame is due after this block
            body.frame();
            to_snap = K >> 2;
          } else {
            to_snap -= seg;
          }
        } while (left);
      }
      n += static_cast<uint64_t>(nb) << 2;
      if (K && snap_aligned) next_snap = (n / K + 1) * static_cast<uint64_t>(K);
      }
    } else {
      // ---- slow path: one step (unaligned head / tail, or K not a multiple of 4) ----
      uint4 w;
      if (XS) {
        // the pair of steps (n & ~1, n | 1) from a copy of S; the odd step commits the advance.
        // The pair is placed where the Philox code below expects the pair of step n.
        uint4 T = S;
        const uint32_t wa = xorshift128(T), wb = xorshift128(T);
        w = make_uint4(wa, wb, wa, wb);
        if (n & 1u) S = T;
      } else {
        w = philox_block(a.seed, (static_cast<uint64_t>(traj_hi) << 32) | traj_lo, n >> 2);
      }
      body.single(w, n);
      ++n;
    }
    if (n == next_snap) {
      body.frame();
      next_snap += K;
    }
  }
}

#ifndef ABM_PHILOX_TABLE
#define ABM_PHILOX_TABLE 1
#endif

// fp64: every CTA copies the Box-Muller tables (1281 x 16 B = 20.5 KB) from global to shared memory once per launch.
__device__ __forceinline__ NoiseTables<float> stage_noise_tables(const StepArgs<float>&) { return {}; }
__device__ __forceinline__ NoiseTables<double> stage_noise_tables(const StepArgs<double>& a) {
  for (int i = threadIdx.x; i < NOISE_TABLE_N; i += STEP_BLOCK) s_noise[i] = a.noise_tables[i];
  __syncthreads();
  return {};
}

template <typename Real, int INTEG, bool TILT, int COEF, bool PRECISE, bool XS>
__global__ void __launch_bounds__(STEP_BLOCK, step_min_blocks<Real, INTEG, COEF>())
step_kernel(const __grid_constant__ StepArgs<Real> a) {
  constexpr bool UNIFORM = COEF == COEF_PARAM;
  const uint64_t k_raw = static_cast<uint64_t>(blockIdx.x) * STEP_BLOCK + threadIdx.x;
  const bool active = k_raw < a.n_traj;
  const uint64_t k = active ? k_raw : a.n_traj - 1;  // idle threads shadow the last trajectory
  const TrajId id = traj_id(k, a.n_particles, a.traj_base, a.set_stride, UNIFORM, a.set_magic);
  Coef<Real> cf = COEF == COEF_PER_THREAD ? a.coef_table[id.set] : a.coef0;
  if (COEF != COEF_PER_THREAD) {
    // Kernel-parameter coefficients are uniform operands and an FMA takes at most one of those.
    // One operand of each uniform pair -- (d, c), (d, gamma0), (k2, k1), (th_s, th_o) -- and the
    // Box-Muller angle offset are therefore read from the table in global memory instead: a
    // loaded value stays in a register for the whole loop, whereas ptxas re-materialises
    // constant-bank values with an LDC / MOV per use.
    const Coef<Real>* g = a.coef_table;
    cf.d = g->d;
    cf.k1 = g->k1;
    cf.th_o = g->th_o;
    cf.bm_o = g->bm_o;
  }
  if (COEF == COEF_SPLIT) {  // what differs between the sets of this sweep
    const Coef<Real>* g = a.coef_table + id.set;
    cf.s2 = g->s2;
    cf.q = g->q;
    cf.k0 = g->k0;
    cf.A = g->A;
  }

  State<Real> s{a.x[k], a.v[k], a.e[k], Real(0), 0u, 0, Real(0)};
  if constexpr (PRECISE) {  // x is the offset; the xl / xh arrays hold the fixed-point words
    s.xf = __float_as_uint(a.xl[k]);
    s.xc = __float_as_int(a.xh[k]);
    s.thb = fixed_angle(s.xf, cf.th_o);
  }

  // High word of the global trajectory index (Philox counter word 3): the host passes it as a
  // kernel parameter when the whole launch shares one value (always, unless the index range
  // straddles a multiple of 2^32); the block-head table of run_steps needs that.
  uint4 S = make_uint4(0u, 0u, 0u, 0u);
  constexpr int TL = TILT ? (UNIFORM ? 2 : 1) : 0;  // what the tilt table holds (one_step)
  Integrate<Real, INTEG, TL, PRECISE> body(a, cf, s, k, active, stage_noise_tables(a));
  if (XS) {
    S = a.rng_state[k];
    run_steps<Real, false, true>(a, 0u, 0u, body, S);
  } else if (a.traj_hi_shared) {
    run_steps<Real, ABM_PHILOX_TABLE != 0, false>(a, static_cast<uint32_t>(id.global), a.traj_hi, body, S);
  } else {
    run_steps<Real, false, false>(a, static_cast<uint32_t>(id.global),
                                  static_cast<uint32_t>(id.global >> 32), body, S);
  }

  if (active) {
    if constexpr (PRECISE) store_fixed(a.xl, a.xh, k, s.xf, s.xc);
    a.x[k] = s.x;
    a.v[k] = s.v;
    a.e[k] = s.e;
    if (XS) a.rng_state[k] = S;
  }
}

// ---------------------------------------------------------------------------------------------
// The step kernel for SMALL ensembles (the paper's own regime: 2^0 ... 2^14 work items, PAPER.md:100,
// where a launch is as slow as one warp's dependent chain, profiles/r01_scaling.md).  With fewer
// warps than schedulers there is nothing to hide latency behind, so the work of one trajectory is
// split between warps instead: a CTA is four warps around 32 trajectories -- warp 0 integrates
// (force, update: the sequential part), warps 1-3 draw the noise of the coming Philox blocks
// (Philox4x32-10 + Box-Muller: 60 % of the instructions, independent of the state) into a
// double-buffered shared-memory ring of SMALL_CHUNK blocks; one __syncthreads per chunk.
// The arithmetic is the same code as in step_kernel (four_steps_z on the same Noise4 values), so the
// result is bit-identical to it -- trajectory i does not depend on which kernel ran.
// fp32, Philox, launches made of whole Philox blocks with frames on block boundaries; everything
// else goes to step_kernel.
// ---------------------------------------------------------------------------------------------
constexpr int SMALL_CHUNK = 16;    // Philox blocks per chunk (64 steps)
constexpr int SMALL_TRAJ = 32;     // trajectories per CTA (one integrating warp)
#ifndef ABM_SMALL_UNROLL
#define ABM_SMALL_UNROLL 4
#endif
constexpr int SMALL_UNROLL = ABM_SMALL_UNROLL;  // Philox blocks per trip of the integrating warp's loop
#ifndef ABM_SMALL_PRODUCERS
#define ABM_SMALL_PRODUCERS 3
#endif
constexpr int SMALL_PRODUCERS = ABM_SMALL_PRODUCERS;            // noise warps per CTA
constexpr int SMALL_BLOCK = 32 * (1 + SMALL_PRODUCERS);  // threads per CTA: 1 integrating warp + the noise warps

template <int INTEG, bool TILT, bool UNIFORM, bool PRECISE>
__global__ void __launch_bounds__(SMALL_BLOCK)
step_kernel_small(const __grid_constant__ StepArgs<float> a) {
  __shared__ float ring[2][SMALL_CHUNK][6][SMALL_TRAJ];
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;  // warp w issues from scheduler w
  const uint64_t k_raw = static_cast<uint64_t>(blockIdx.x) * SMALL_TRAJ + lane;
  const bool active = k_raw < a.n_traj;
  const uint64_t k = active ? k_raw : a.n_traj - 1;  // idle lanes shadow the last trajectory
  const TrajId id = traj_id(k, a.n_particles, a.traj_base, a.set_stride, UNIFORM, a.set_magic);
  const Coef<float> cf = UNIFORM ? a.coef0 : a.coef_table[id.set];
  constexpr int TL = TILT ? (UNIFORM ? 2 : 1) : 0;

  const uint32_t n_blocks = a.n_steps >> 2;         // the host sends whole blocks only
  const uint64_t b0 = a.step0 >> 2;
  const uint32_t n_chunks = (n_blocks + SMALL_CHUNK - 1) / SMALL_CHUNK;

  auto produce = [&](uint32_t chunk, uint32_t buf) {  // warp w >= 1: blocks j = w - 1, w - 1 + SMALL_PRODUCERS, ...
    const uint32_t first = chunk * SMALL_CHUNK;
    const uint32_t cnt = n_blocks - first < SMALL_CHUNK ? n_blocks - first : SMALL_CHUNK;
    for (uint32_t j = warp - 1u; j < cnt; j += SMALL_PRODUCERS) {
      const Noise4<float> z(philox_block(a.seed, id.global, b0 + first + j), cf);
      float(*slot)[SMALL_TRAJ] = ring[buf][j];
      slot[0][lane] = z.a.rho; slot[1][lane] = z.a.cs; slot[2][lane] = z.a.sn;
      slot[3][lane] = z.b.rho; slot[4][lane] = z.b.cs; slot[5][lane] = z.b.sn;
    }
  };

  State<float> s{0.f, 0.f, 0.f, 0.f, 0u, 0, 0.f};
  TiltCursor<float, INTEG> tl;
  uint32_t to_snap = 0xffffffffu;  // blocks until the next frame (a launch has fewer than 2^30 steps)
  const uint32_t K = a.snap != nullptr ? a.snap_every : 0u;
  if (warp == 0) {
    s.x = a.x[k]; s.v = a.v[k]; s.e = a.e[k];
    if constexpr (PRECISE) {
      s.xf = __float_as_uint(a.xl[k]);
      s.xc = __float_as_int(a.xh[k]);
      s.thb = fixed_angle(s.xf, cf.th_o);
    }
    if (TILT) tl.start(a.tilt + (a.step0 - a.tilt_base));
    if (K) to_snap = static_cast<uint32_t>(((a.step0 / K + 1) * static_cast<uint64_t>(K) - a.step0) >> 2);
  } else {
    produce(0u, 0u);
  }
  __syncthreads();
  uint32_t buf = 0;
  for (uint32_t c = 0; c < n_chunks; ++c) {
    if (warp == 0) {
      const uint32_t first = c * SMALL_CHUNK;
      const uint32_t cnt = n_blocks - first < SMALL_CHUNK ? n_blocks - first : SMALL_CHUNK;
#pragma unroll SMALL_UNROLL
      for (uint32_t j = 0; j < cnt; ++j) {
        float(*slot)[SMALL_TRAJ] = ring[buf][j];
        Normal2f za, zb;
        za.rho = slot[0][lane]; za.cs = slot[1][lane]; za.sn = slot[2][lane];
        zb.rho = slot[3][lane]; zb.cs = slot[4][lane]; zb.sn = slot[5][lane];
        const Noise4<float> z(za, zb);
        four_steps_z<float, INTEG, TL, PRECISE>(s, cf, z, tl);
        if (--to_snap == 0) {
          if (active) store_snapshot(a.snap, a.snap_stride, k, frame_state<PRECISE>(s, cf));
          to_snap = K >> 2;
        }
      }
    } else if (c + 1 < n_chunks) {
      produce(c + 1, buf ^ 1u);
    }
    __syncthreads();
    buf ^= 1u;
  }
  if (warp == 0 && active) {
    if constexpr (PRECISE) store_fixed(a.xl, a.xh, k, s.xf, s.xc);
    a.x[k] = s.x;
    a.v[k] = s.v;
    a.e[k] = s.e;
  }
}

// ---------------------------------------------------------------------------------------------
// S6  moments.  Pass 1: each CTA reduces a contiguous slice of one set (fp64 accumulators,
// fixed order: per-thread serial, xor-shuffle tree, serial over warps).  Pass 2: one thread
// per set adds the CTA partials in index order and finalises.  No atomics: reproducible.
// sums = { N, sum x, sum x^2, sum v, sum v^2, sum e, sum dx, sum dx^2 }, dx = x - x(0).
// ---------------------------------------------------------------------------------------------
template <typename Real>
__global__ void __launch_bounds__(MOM_BLOCK)
moments_partial_kernel(const Real* __restrict__ x, const Real* __restrict__ v,
                       const Real* __restrict__ e, const Real* __restrict__ xl,
                       const Real* __restrict__ xh, const Coef<Real>* __restrict__ coef_table,
                       uint64_t n_particles, uint64_t traj_base, uint64_t set_stride, uint64_t seed,
                       uint32_t blocks_per_set, uint32_t slice, double* __restrict__ partial) {
  const uint32_t set = blockIdx.x / blocks_per_set;
  const uint32_t blk = blockIdx.x - set * blocks_per_set;
  const uint64_t r0 = static_cast<uint64_t>(blk) * slice;
  uint64_t r1 = r0 + slice;
  if (r1 > n_particles) r1 = n_particles;
  const Coef<Real> c = coef_table[set];
  double acc[N_SUMS - 1] = {0, 0, 0, 0, 0, 0, 0};
  for (uint64_t r = r0 + threadIdx.x; r < r1; r += blockDim.x) {
    const uint64_t k = static_cast<uint64_t>(set) * n_particles + r;
    const uint64_t g = traj_base + static_cast<uint64_t>(set) * set_stride + r;
    const uint4 w = philox_block(seed, g, INIT_BLOCK);
    const double xi = static_cast<double>(load_position(x, xl, xh, k, c.L));
    const double vi = static_cast<double>(v[k]);
    const double dx = xi - static_cast<double>(init_x(c, w.x));
    acc[0] += xi;
    acc[1] += xi * xi;
    acc[2] += vi;
    acc[3] += vi * vi;
    acc[4] += static_cast<double>(e[k]);
    acc[5] += dx;
    acc[6] += dx * dx;
  }
  __shared__ double sm[MOM_BLOCK / 32][N_SUMS - 1];
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
#pragma unroll
  for (int q = 0; q < N_SUMS - 1; ++q) {
    double t = acc[q];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) t += __shfl_xor_sync(0xffffffffu, t, off);
    if (lane == 0) sm[warp][q] = t;
  }
  __syncthreads();
  if (threadIdx.x < N_SUMS - 1) {
    double t = 0;
    const uint32_t n_warps = (blockDim.x + 31u) >> 5;
    for (uint32_t wq = 0; wq < n_warps; ++wq) t += sm[wq][threadIdx.x];
    partial[(static_cast<uint64_t>(blockIdx.x)) * (N_SUMS - 1) + threadIdx.x] = t;
  }
}

struct MomentRec {  // mirrors abm_moment (include/abm.h)
  uint64_t n, step;
  double mean_x, var_x, mean_v, var_v, mean_e, mean_dx, mean_dx2, mean_x2;
};

__host__ __device__ inline void finalize_moment(const double* s, uint64_t step, MomentRec* m) {
  const double N = s[0];
  m->n = static_cast<uint64_t>(N);
  m->step = step;
  const double mx = s[1] / N, mv = s[3] / N;
  // no FMA contraction: the device record and abm_moments_from_sums (host) agree bit for bit
#ifdef __CUDA_ARCH__
  const double mx2 = __dmul_rn(mx, mx), mv2 = __dmul_rn(mv, mv);
  m->var_x = __dsub_rn(s[2] / N, mx2);
  m->var_v = __dsub_rn(s[4] / N, mv2);
#else
  volatile double mx2 = mx * mx, mv2 = mv * mv;
  m->var_x = s[2] / N - mx2;
  m->var_v = s[4] / N - mv2;
#endif
  m->mean_x = mx;
  m->mean_v = mv;
  m->mean_e = s[5] / N;
  m->mean_dx = s[6] / N;
  m->mean_dx2 = s[7] / N;
  m->mean_x2 = s[2] / N;
}

// One warp per set: lane l adds the CTA partials l, l + 32, ... in index order, then a fixed
// xor-shuffle tree; lane 0 finalises.
__global__ void __launch_bounds__(128)
moments_final_kernel(const double* __restrict__ partial, uint32_t n_sets, uint32_t blocks_per_set,
                     uint64_t n_particles, uint64_t step, double* __restrict__ sums,
                     MomentRec* __restrict__ out) {
  const uint32_t set = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const uint32_t lane = threadIdx.x & 31u;
  if (set >= n_sets) return;  // whole warps leave together
  double s[N_SUMS];
  s[0] = static_cast<double>(n_particles);
  const double* p = partial + static_cast<uint64_t>(set) * blocks_per_set * (N_SUMS - 1);
#pragma unroll
  for (int q = 0; q < N_SUMS - 1; ++q) {
    double t = 0;
    for (uint32_t b = lane; b < blocks_per_set; b += 32)
      t += p[static_cast<uint64_t>(b) * (N_SUMS - 1) + q];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) t += __shfl_xor_sync(0xffffffffu, t, off);
    s[q + 1] = t;
  }
  if (lane == 0) {
    for (int q = 0; q < N_SUMS; ++q) sums[static_cast<uint64_t>(set) * N_SUMS + q] = s[q];
    finalize_moment(s, step, &out[set]);
  }
}

// ---------------------------------------------------------------------------------------------
// Headless presentation: the paper draws every work item as one vertex of
// the shared buffer; with no graphics API the frame is rasterised here into a
// 2-D histogram of (x mod L, v) -- a point splat with additive blending -- and colour-mapped to
// RGBA8.  The bin of a point is decided in fp64 with individually rounded operations (include/abm.h
// states the rule), so that the CPU oracle takes the same decision bit for bit.
//
// Points are unsorted, so every CTA scatters over the whole image: small images (<= RASTER_SMEM_BINS
// bins) are privatised in shared memory (shared atomics, then one global reduction per CTA and
// bin); larger ones use fire-and-forget global reductions (RED.ADD), which the 126 MB L2 absorbs
// (a 1024 x 1024 image is 4 MB).
// ---------------------------------------------------------------------------------------------
constexpr int RASTER_BLOCK = 256;
constexpr uint32_t RASTER_SMEM_BINS = 12288;  // 48 KB of uint32

// -> bin index, or 0xffffffff if the point is outside the velocity window (or not finite)
__device__ __forceinline__ uint32_t raster_bin(double x, double v, double L, double v_min,
                                               double v_range, uint32_t W, uint32_t H) {
  const double xi = __ddiv_rn(x, L);
  const double f = __dsub_rn(xi, floor(xi));                 // in [0, 1]
  const double eta = __ddiv_rn(__dsub_rn(v, v_min), v_range);
  if (!(eta >= 0.0) || !(eta < 1.0) || !(f >= 0.0)) return 0xffffffffu;  // also drops NaN
  uint32_t ix = static_cast<uint32_t>(floor(__dmul_rn(f, static_cast<double>(W))));
  uint32_t iy = static_cast<uint32_t>(floor(__dmul_rn(eta, static_cast<double>(H))));
  if (ix >= W) ix = W - 1;  // f == 1 after rounding (x a hair below a multiple of L)
  if (iy >= H) iy = H - 1;
  return iy * W + ix;
}

template <typename Real, bool SMEM>
__global__ void __launch_bounds__(RASTER_BLOCK)
raster_kernel(const Real* __restrict__ x, const Real* __restrict__ v, const Real* __restrict__ xl,
              const Real* __restrict__ xh, const Coef<Real>* __restrict__ coef_table, uint64_t n_traj, uint64_t n_particles,
              uint32_t n_sets, uint32_t W, uint32_t H, double v_min, double v_range,
              uint32_t* __restrict__ counts) {
  extern __shared__ uint32_t hist[];
  const uint32_t n_bins = W * H;
  if (SMEM) {
    for (uint32_t b = threadIdx.x; b < n_bins; b += RASTER_BLOCK) hist[b] = 0;
    __syncthreads();
  }
  const uint64_t stride = static_cast<uint64_t>(gridDim.x) * RASTER_BLOCK;
  for (uint64_t k = static_cast<uint64_t>(blockIdx.x) * RASTER_BLOCK + threadIdx.x; k < n_traj;
       k += stride) {
    const uint32_t set = n_sets == 1 ? 0u : static_cast<uint32_t>(k / n_particles);
    const Real Lr = coef_table[set].L;
    const double L = static_cast<double>(Lr);
    const uint32_t bin = raster_bin(static_cast<double>(load_position(x, xl, xh, k, Lr)),
                                    static_cast<double>(v[k]), L, v_min,
                                    v_range, W, H);
    if (bin != 0xffffffffu) {
      if (SMEM) atomicAdd(&hist[bin], 1u);
      else atomicAdd(&counts[bin], 1u);  // result unused: compiles to RED.E.ADD
    }
  }
  if (SMEM) {
    __syncthreads();
    for (uint32_t b = threadIdx.x; b < n_bins; b += RASTER_BLOCK) {
      const uint32_t c = hist[b];
      if (c) atomicAdd(&counts[b], c);
    }
  }
}

// counts -> RGBA8 grey ramp: level = min(255, floor(255 c / saturation)), alpha 255.
__global__ void __launch_bounds__(256)
colormap_kernel(const uint32_t* __restrict__ counts, uint32_t n_bins, uint32_t saturation,
                uchar4* __restrict__ rgba) {
  const uint32_t b = blockIdx.x * 256u + threadIdx.x;
  if (b >= n_bins) return;
  const uint64_t c = counts[b];
  const uint64_t lv = c >= saturation ? 255ull : (255ull * c) / saturation;
  const unsigned char l = static_cast<unsigned char>(lv);
  rgba[b] = make_uchar4(l, l, l, 255);
}

// ---------------------------------------------------------------------------------------------
// Diagnostic: raw Philox blocks of the stream
// ---------------------------------------------------------------------------------------------
__global__ void philox_blocks_kernel(uint64_t seed, uint64_t traj_first, uint64_t n_traj,
                                     uint64_t block_first, uint64_t n_blocks, uint4* out) {
  const uint64_t t = static_cast<uint64_t>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (t >= n_traj * n_blocks) return;
  const uint64_t k = t / n_blocks, j = t - k * n_blocks;
  out[t] = philox_block(seed, traj_first + k, block_first + j);
}

// The same words as the block loop of the step kernels produces them: this kernel has step_kernel's launch
// geometry and thread <-> trajectory assignment and instantiates the SAME run_steps (above) with a body that
// stores each block's words instead of integrating with them.  a.step0 = 4 * first block, a.n_steps = 4 *
// blocks, a.snap_every = frame period in steps (segments the loop as frames do; nothing is stored for them),
// a.snap any non-null pointer if a.snap_every != 0.  out[k * n_blocks + j] = block step0 / 4 + j of trajectory k.
// Real only selects the loop shape (float: two blocks per trip; double: one).
template <typename Real>
__global__ void __launch_bounds__(STEP_BLOCK)
philox_loop_kernel(const __grid_constant__ StepArgs<Real> a, uint4* __restrict__ out) {
  const uint64_t k_raw = static_cast<uint64_t>(blockIdx.x) * STEP_BLOCK + threadIdx.x;
  const bool active = k_raw < a.n_traj;
  const uint64_t k = active ? k_raw : a.n_traj - 1;
  const uint64_t g = a.traj_base + k;
  DumpWords body{active ? out + k * (a.n_steps >> 2) : nullptr};
  uint4 S = make_uint4(0u, 0u, 0u, 0u);
  if (a.traj_hi_shared)
    run_steps<Real, ABM_PHILOX_TABLE != 0, false>(a, static_cast<uint32_t>(g), a.traj_hi, body, S);
  else
    run_steps<Real, false, false>(a, static_cast<uint32_t>(g), static_cast<uint32_t>(g >> 32), body, S);
}

}  // namespace abm
