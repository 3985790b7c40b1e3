// pipe_rates.cu -- measures the per-SM issue rates of the instruction classes the step kernel is
// made of, on the device it runs on (build-plan step 0 of SURVEY.md 7; the denominators of the
// "alu" roofline in DESIGN.md).  Not part of the C ABI: a stand-alone diagnostic,
//
//     python -m paper_1104_2499_b200.build --pipe-rates && paper_1104_2499_b200/pipe_rates
//
// Method: every thread runs CHAINS independent dependency chains of one instruction (inline PTX,
// so ptxas keeps each one), unrolled, for ITERS iterations; one CTA of `threads` threads per SM
// x `ctas_per_sm`; the SM-clock cycles of every CTA are read with clock64() and the slowest CTA
// is taken.  Result: warp-lane operations per clock per SM.  A second table measures mixes
// (two classes interleaved) to expose which classes share a pipe / an issue port.
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#include <algorithm>
#include <cuda_runtime.h>
#include "abm_device.cuh"  // only for the last table: the accuracy of box_muller_f32 as the step kernels call it

#define CK(x)                                                                      \
  do {                                                                             \
    cudaError_t e_ = (x);                                                          \
    if (e_ != cudaSuccess) {                                                       \
      std::fprintf(stderr, "%s:%d %s\n", __FILE__, __LINE__, cudaGetErrorString(e_)); \
      std::exit(1);                                                                \
    }                                                                              \
  } while (0)

constexpr int CHAINS = 8;
constexpr int UNROLL = 8;   // CHAINS * UNROLL instructions (per class) per loop iteration

enum Op {
  FFMA_RRR, FFMA_RRC, FFMA_RIR, FMUL_RR, FADD_RR, IMAD_LO, IMAD_WIDE_R, IMAD_WIDE_I, LOP3_XOR3,
  IADD3, SHF_R, MUFU_COS, MUFU_SIN, MUFU_LG2, MUFU_SQRT, MUFU_RSQ, MUFU_EX2, MUFU_RCP,
  DFMA_, DMUL_, DADD_, I2F_, F2I_, FFMA2_, FRND_, N_OPS
};
static const char* OP_NAME[N_OPS] = {
  "FFMA r,r,r", "FFMA r,r,c[]", "FFMA r,imm,r", "FMUL r,r", "FADD r,r", "IMAD.LO r,r,r",
  "IMAD.WIDE.U32 r,r", "IMAD.WIDE r,imm + LOP3", "LOP3 (xor3)", "IADD3 r,r,r", "SHF.R",
  "FMUL+MUFU.COS", "FMUL+MUFU.SIN", "MUFU.LG2", "MUFU.SQRT", "MUFU.RSQ", "MUFU.EX2", "FADD+MUFU.RCP",
  "DFMA", "DMUL", "DADD", "I2F.U32", "F2I.U32", "FFMA2 (f32x2, per elem)", "FRND"};

struct Regs {
  float f[CHAINS];
  uint32_t u[CHAINS];
  uint32_t h[CHAINS];
  double d[CHAINS];
  unsigned long long p[CHAINS];
};

__constant__ float c_k[4];

template <int OP>
__device__ __forceinline__ void one(Regs& r, int j, float fb, float fc, uint32_t ub, uint32_t uc,
                                    double db, double dc, unsigned long long pb = 0,
                                    unsigned long long pc = 0) {
  if (OP == FFMA_RRR) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(r.f[j]) : "f"(fb), "f"(fc));
  if (OP == FFMA_RRC) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(r.f[j]) : "f"(fb), "f"(c_k[1]));
  if (OP == FFMA_RIR) asm volatile("fma.rn.f32 %0, %0, 0f3F7FFFF0, %1;" : "+f"(r.f[j]) : "f"(fc));
  if (OP == FMUL_RR) asm volatile("mul.rn.f32 %0, %0, %1;" : "+f"(r.f[j]) : "f"(fb));
  if (OP == FADD_RR) asm volatile("add.rn.f32 %0, %0, %1;" : "+f"(r.f[j]) : "f"(fc));
  if (OP == IMAD_LO) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r.u[j]) : "r"(ub), "r"(uc));
  // 32 x 32 -> 64 with both result words fed back as the next operands (a product chain with a
  // dead high word would be folded by ptxas)
  if (OP == IMAD_WIDE_R)
    asm volatile("{\n\t.reg .u64 p;\n\tmul.wide.u32 p, %0, %1;\n\tmov.b64 {%0, %1}, p;\n\t}"
                 : "+r"(r.u[j]), "+r"(r.h[j]));
  // half a Philox round: one wide multiply by an immediate, one three-input xor of its words
  if (OP == IMAD_WIDE_I)
    asm volatile("{\n\t.reg .u64 p;\n\t.reg .u32 lo, hi;\n\tmul.wide.u32 p, %0, 0xD2511F53;\n\t"
                 "mov.b64 {lo, hi}, p;\n\tlop3.b32 %0, lo, hi, %1, 0x96;\n\t}" : "+r"(r.u[j]) : "r"(ub));
  if (OP == LOP3_XOR3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r.u[j]) : "r"(ub), "r"(uc));
  if (OP == IADD3)
    asm volatile("{\n\t.reg .u32 t;\n\tadd.u32 t, %0, %1;\n\tadd.u32 %0, t, %2;\n\t}" : "+r"(r.u[j]) : "r"(ub), "r"(uc));
  if (OP == SHF_R) asm volatile("shf.r.wrap.b32 %0, %0, %1, 9;" : "+r"(r.u[j]) : "r"(ub));
  if (OP == MUFU_COS) asm volatile("cos.approx.ftz.f32 %0, %0;" : "+f"(r.f[j]));
  if (OP == MUFU_SIN) asm volatile("sin.approx.ftz.f32 %0, %0;" : "+f"(r.f[j]));
  if (OP == MUFU_LG2) asm volatile("lg2.approx.ftz.f32 %0, %0;" : "+f"(r.f[j]));
  if (OP == MUFU_SQRT) asm volatile("sqrt.approx.ftz.f32 %0, %0;" : "+f"(r.f[j]));
  if (OP == MUFU_RSQ) asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(r.f[j]));
  if (OP == MUFU_EX2) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(r.f[j]));
  // with an FADD in the chain: ptxas folds rcp(rcp(x)) to x even in volatile asm, which emptied the loop
  if (OP == MUFU_RCP)
    asm volatile("{\n\t.reg .f32 t;\n\trcp.approx.ftz.f32 t, %0;\n\tadd.rn.f32 %0, t, %1;\n\t}" : "+f"(r.f[j]) : "f"(fc));
  if (OP == DFMA_) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(r.d[j]) : "d"(db), "d"(dc));
  if (OP == DMUL_) asm volatile("mul.rn.f64 %0, %0, %1;" : "+d"(r.d[j]) : "d"(db));
  if (OP == DADD_) asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(r.d[j]) : "d"(dc));
  if (OP == I2F_) asm volatile("{\n\t.reg .f32 t;\n\tcvt.rn.f32.u32 t, %0;\n\tmov.b32 %0, t;\n\t}" : "+r"(r.u[j]));
  // packed pair of fp32 FMAs (sm_100 FFMA2): counted as TWO lane-ops per thread below
  if (OP == FFMA2_) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(r.p[j]) : "l"(pb), "l"(pc));
  if (OP == FRND_) asm volatile("cvt.rni.f32.f32 %0, %0;" : "+f"(r.f[j]));
  if (OP == F2I_) asm volatile("{\n\t.reg .u32 t;\n\tcvt.rzi.u32.f32 t, %0;\n\tmov.b32 %0, t;\n\t}" : "+f"(r.f[j]));
}

__host__ __device__ constexpr bool uses_f(int op) {
  return op <= FADD_RR || (op >= MUFU_COS && op <= MUFU_RCP) || op == F2I_ || op == FRND_;
}
__host__ __device__ constexpr bool uses_d(int op) { return op >= DFMA_ && op <= DADD_; }
__host__ __device__ constexpr bool uses_p(int op) { return op == FFMA2_; }
__host__ __device__ constexpr bool uses_u(int op) {
  return op < N_OPS && !uses_f(op) && !uses_d(op) && !uses_p(op);
}

template <int OP>
__device__ __forceinline__ void init_regs(Regs& r, const float* in, int o) {
#pragma unroll
  for (int j = 0; j < CHAINS; ++j) {
    if (uses_f(OP)) r.f[j] = in[4 + o] + j + threadIdx.x;
    if (uses_u(OP)) { r.u[j] = __float_as_uint(in[5 + o]) + 3 * j + threadIdx.x; r.h[j] = 0; }
    if (uses_d(OP)) r.d[j] = static_cast<double>(in[4 + o]) + j + threadIdx.x;
    if (uses_p(OP)) {
      const float2 t = make_float2(in[4 + o] + j + threadIdx.x, in[5 + o] + j);
      r.p[j] = *reinterpret_cast<const unsigned long long*>(&t);
    }
  }
}
template <int OP>
__device__ __forceinline__ void fold_regs(const Regs& r, float& acc, uint32_t& ua, double& da) {
#pragma unroll
  for (int j = 0; j < CHAINS; ++j) {
    if (uses_f(OP)) acc += r.f[j];
    if (uses_u(OP)) ua ^= r.u[j] ^ r.h[j];
    if (uses_d(OP)) da += r.d[j];
    if (uses_p(OP)) ua ^= static_cast<uint32_t>(r.p[j]) ^ static_cast<uint32_t>(r.p[j] >> 32);
  }
}

// OPA alone (OPB == N_OPS) or OPA and OPB interleaved one to one.
template <int OPA, int OPB>
__global__ void __launch_bounds__(1024) rate_kernel(int iters, const float* __restrict__ in,
                                                   float* __restrict__ out,
                                                   long long* __restrict__ cycles) {
  Regs a, b;
  const float fb = in[0], fc = in[1];
  const uint32_t ub = __float_as_uint(in[2]) | 1u, uc = __float_as_uint(in[3]);
  const double db = static_cast<double>(in[0]), dc = static_cast<double>(in[1]);
  const float2 fb2 = make_float2(fb, fb), fc2 = make_float2(fc, fc);
  const unsigned long long pb = *reinterpret_cast<const unsigned long long*>(&fb2);
  const unsigned long long pc = *reinterpret_cast<const unsigned long long*>(&fc2);
  init_regs<OPA>(a, in, 0);
  init_regs<OPB>(b, in, 2);
  __syncthreads();
  const long long t0 = clock64();
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < UNROLL; ++u) {
#pragma unroll
      for (int j = 0; j < CHAINS; ++j) {
        one<OPA>(a, j, fb, fc, ub, uc, db, dc, pb, pc);
        if (OPB != N_OPS) one<OPB == N_OPS ? 0 : OPB>(b, j, fb, fc, ub, uc, db, dc, pb, pc);
      }
    }
  }
  const long long t1 = clock64();
  __syncthreads();
  float acc = 0;
  uint32_t ua = 0;
  double da = 0;
  fold_regs<OPA>(a, acc, ua, da);
  fold_regs<OPB>(b, acc, ua, da);
  if (static_cast<double>(acc) + static_cast<double>(ua) + da == 12345.0) out[threadIdx.x] = acc;  // keep all live
  if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

struct Dev {
  int n_sm;
  float* in;
  float* out;
  long long* cyc;
};

template <int OPA, int OPB>
double run(const Dev& d, int threads, int ctas_per_sm, int iters) {
  const int grid = d.n_sm * ctas_per_sm;
  rate_kernel<OPA, OPB><<<grid, threads>>>(4, d.in, d.out, d.cyc);  // warm-up (I-cache)
  rate_kernel<OPA, OPB><<<grid, threads>>>(iters, d.in, d.out, d.cyc);
  CK(cudaDeviceSynchronize());
  std::vector<long long> c(grid);
  CK(cudaMemcpy(c.data(), d.cyc, sizeof(long long) * grid, cudaMemcpyDeviceToHost));
  const long long worst = *std::max_element(c.begin(), c.end());
  const double per_class = static_cast<double>(iters) * UNROLL * CHAINS * threads * ctas_per_sm;
  return per_class / static_cast<double>(worst);  // lane-ops per clock per SM, per class
}

template <int OP>
void single(const Dev& d) {
  const double r4 = run<OP, N_OPS>(d, 128, 1, 2000);    // 1 warp / scheduler: what ONE warp can issue
  const double r8 = run<OP, N_OPS>(d, 256, 1, 2000);    // 2 warps / scheduler
  const double r16 = run<OP, N_OPS>(d, 512, 1, 2000);   // 4 warps / scheduler
  const double r32 = run<OP, N_OPS>(d, 1024, 1, 1000);  // 8 warps / scheduler
  const double w = OP == FFMA2_ ? 2.0 : 1.0;  // two fp32 FMAs per FFMA2
  std::printf("%-22s %8.1f %8.1f %8.1f %8.1f\n", OP_NAME[OP], w * r4, w * r8, w * r16, w * r32);
}

template <int OPA, int OPB>
void mix(const Dev& d) {
  const double r = run<OPA, OPB>(d, 1024, 1, 1000);
  const double wa = OPA == FFMA2_ ? 2.0 : 1.0, wb = OPB == FFMA2_ ? 2.0 : 1.0;
  std::printf("%-24s + %-24s %8.1f / %8.1f, %8.1f total\n", OP_NAME[OPA], OP_NAME[OPB], wa * r, wb * r,
              (wa + wb) * r);
}

template <int OPA, int OPB>
void mix1(const Dev& d) {
  const double r = run<OPA, OPB>(d, 128, 1, 2000);
  const double wa = OPA == FFMA2_ ? 2.0 : 1.0, wb = OPB == FFMA2_ ? 2.0 : 1.0;
  std::printf("%-24s + %-24s %8.1f / %8.1f, %8.1f total\n", OP_NAME[OPA], OP_NAME[OPB], wa * r, wb * r,
              (wa + wb) * r);
}

// ---------------------------------------------------------------------------------------------
// Third table: the instruction mix of the fp32 Euler-Maruyama step loop (one Philox block = four
// steps: 54 FFMA/FMUL/FADD, 6 x (FMUL.RZ + MUFU.COS), 6 more MUFU, 16 x (IMAD.WIDE + LOP3), 8 more
// ALU-pipe instructions) as a stream of INDEPENDENT chains, 128-thread CTAs as in the step kernel.
// What this runs at is what the SM can do with that mix when nothing waits on a dependency: the
// ceiling the step kernel is compared with in DESIGN.md 8.  MODE bit 0: FP32, 1: Philox, 2: MUFU,
// 3: the extra ALU instructions.
// ---------------------------------------------------------------------------------------------
#define PR_FF(r) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(r) : "f"(fb), "f"(fc));
#define PR_IW(r)                                                                                  \
  asm volatile("{\n\t.reg .u64 p;\n\t.reg .u32 lo, hi;\n\tmul.wide.u32 p, %0, 0xD2511F53;\n\t"    \
               "mov.b64 {lo, hi}, p;\n\tlop3.b32 %0, lo, hi, %1, 0x96;\n\t}" : "+r"(r) : "r"(ub));
#define PR_LX(r) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r) : "r"(ub), "r"(uc));
#define PR_MC(r) asm volatile("cos.approx.ftz.f32 %0, %0;" : "+f"(r));
#define PR_ML(r) asm volatile("lg2.approx.ftz.f32 %0, %0;" : "+f"(r));
#define PR_MS(r) asm volatile("sqrt.approx.ftz.f32 %0, %0;" : "+f"(r));
#define PR_ME(r) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(r));

template <int MODE>
__global__ void __launch_bounds__(128) loop_mix_kernel(int iters, const float* __restrict__ in,
                                                       float* __restrict__ out,
                                                       long long* __restrict__ cycles) {
  float f[12], m[8];
  uint32_t u[8];
  const float fb = in[0], fc = in[1];
  const uint32_t ub = __float_as_uint(in[2]) | 1u, uc = __float_as_uint(in[3]);
#pragma unroll
  for (int j = 0; j < 12; ++j) f[j] = in[4] + j + threadIdx.x;
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    u[j] = ub * (j + 3) + threadIdx.x;
    m[j] = in[5] + j * 0.1f;
  }
  __syncthreads();
  const long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int q = 0; q < 2; ++q) {  // half a block per pass
      if (MODE & 1) { PR_FF(f[0]) PR_FF(f[1]) PR_FF(f[2]) }
      if (MODE & 2) { PR_IW(u[0]) PR_IW(u[1]) }
      if (MODE & 4) { PR_MC(m[0]) }
      if (MODE & 1) { PR_FF(f[3]) PR_FF(f[4]) PR_FF(f[5]) }
      if (MODE & 2) { PR_IW(u[2]) PR_IW(u[3]) }
      if (MODE & 4) { PR_MC(m[1]) PR_ML(m[2]) }
      if (MODE & 1) { PR_FF(f[6]) PR_FF(f[7]) PR_FF(f[8]) PR_FF(f[0]) }
      if (MODE & 8) { PR_LX(u[4]) PR_LX(u[5]) }
      if (MODE & 2) { PR_IW(u[0]) PR_IW(u[1]) }
      if (MODE & 4) { PR_MC(m[3]) PR_MS(m[4]) }
      if (MODE & 1) { PR_FF(f[9]) PR_FF(f[10]) PR_FF(f[11]) PR_FF(f[1]) PR_FF(f[2]) }
      if (MODE & 2) { PR_IW(u[2]) PR_IW(u[3]) }
      if (MODE & 4) { PR_ME(m[5]) }
      if (MODE & 8) { PR_LX(u[6]) PR_LX(u[7]) }
      if (MODE & 1) {
        PR_FF(f[3]) PR_FF(f[4]) PR_FF(f[5]) PR_FF(f[6]) PR_FF(f[7]) PR_FF(f[8])
        PR_FF(f[9]) PR_FF(f[10]) PR_FF(f[11]) PR_FF(f[0]) PR_FF(f[1]) PR_FF(f[2])
      }
    }
  }
  const long long t1 = clock64();
  float acc = 0;
  uint32_t ua = 0;
#pragma unroll
  for (int j = 0; j < 12; ++j) acc += f[j];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    ua ^= u[j];
    acc += m[j];
  }
  if (static_cast<double>(acc) + static_cast<double>(ua) == 12345.0) out[threadIdx.x] = acc;
  if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

// -> SM cycles per warp and scheduler for one pass of the mix (one Philox block = four steps)
template <int MODE>
double loop_mix(const Dev& d, int ctas_per_sm) {
  const int iters = 20000, grid = d.n_sm * ctas_per_sm;
  loop_mix_kernel<MODE><<<grid, 128>>>(200, d.in, d.out, d.cyc);
  loop_mix_kernel<MODE><<<grid, 128>>>(iters, d.in, d.out, d.cyc);
  CK(cudaDeviceSynchronize());
  std::vector<long long> c(grid);
  CK(cudaMemcpy(c.data(), d.cyc, sizeof(long long) * grid, cudaMemcpyDeviceToHost));
  const long long worst = *std::max_element(c.begin(), c.end());
  return static_cast<double>(worst) / iters / ctas_per_sm;  // a CTA has one warp per scheduler
}

template <int MODE>
void loop_mix_row(const Dev& d, const char* name) {
  std::printf("%-44s %8.1f %8.1f %8.1f\n", name, loop_mix<MODE>(d, 4), loop_mix<MODE>(d, 9),
              loop_mix<MODE>(d, 12));
}

// ---------------------------------------------------------------------------------------------
// Fourth table: the fp32 Heun + tilt loop (config[3]) as independent chains, per Philox block = four steps:
// 120 FFMA/FADD/FMUL, 10 x (FMUL.RZ + MUFU.COS) + 6 more MUFU, 16 x (IMAD.WIDE + LOP3), 4 LDG + 1 LDS.128,
// F2I + I2F, 14 more ALU instructions.  MODE bits: 1 FP32, 2 Philox, 4 MUFU, 8 ALU extras, 16 loads + conversions.
// ---------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(128) heun_mix_kernel(int iters, const float* __restrict__ in,
                                                       float* __restrict__ out,
                                                       long long* __restrict__ cycles) {
  __shared__ float4 sh[128];
  float f[12], m[8];
  uint32_t u[8];
  const float fb = in[0], fc = in[1];
  const uint32_t ub = __float_as_uint(in[2]) | 1u, uc = __float_as_uint(in[3]);
#pragma unroll
  for (int j = 0; j < 12; ++j) f[j] = in[4] + j + threadIdx.x;
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    u[j] = ub * (j + 3) + threadIdx.x;
    m[j] = in[5] + j * 0.1f;
  }
  sh[threadIdx.x] = make_float4(fb, fc, fb, fc);
  __syncthreads();
  const float* g = in;
  float ld = 0.f;
  const long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int q = 0; q < 2; ++q) {  // half a block per pass: 60 FP32, 8 IW, 5 cos + 3 MUFU, 7 ALU, 2 LDG
      if (MODE & 1) { PR_FF(f[0]) PR_FF(f[1]) PR_FF(f[2]) PR_FF(f[3]) PR_FF(f[4]) PR_FF(f[5]) }
      if (MODE & 2) { PR_IW(u[0]) PR_IW(u[1]) }
      if (MODE & 4) { PR_MC(m[0]) PR_MC(m[1]) }
      if (MODE & 16) { float t; asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(t) : "l"(g + (it & 3))); ld += t; }
      if (MODE & 1) { PR_FF(f[6]) PR_FF(f[7]) PR_FF(f[8]) PR_FF(f[9]) PR_FF(f[10]) PR_FF(f[11]) PR_FF(f[0]) PR_FF(f[1]) }
      if (MODE & 2) { PR_IW(u[2]) PR_IW(u[3]) }
      if (MODE & 4) { PR_MC(m[2]) PR_ML(m[3]) }
      if (MODE & 8) { PR_LX(u[4]) PR_LX(u[5]) PR_LX(u[6]) }
      if (MODE & 1) { PR_FF(f[2]) PR_FF(f[3]) PR_FF(f[4]) PR_FF(f[5]) PR_FF(f[6]) PR_FF(f[7]) PR_FF(f[8]) PR_FF(f[9]) }
      if (MODE & 2) { PR_IW(u[0]) PR_IW(u[1]) }
      if (MODE & 4) { PR_MC(m[4]) PR_MS(m[5]) }
      if (MODE & 16) { float t; asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(t) : "l"(g + ((it + 1) & 3))); ld += t; }
      if (MODE & 1) { PR_FF(f[10]) PR_FF(f[11]) PR_FF(f[0]) PR_FF(f[1]) PR_FF(f[2]) PR_FF(f[3]) PR_FF(f[4]) PR_FF(f[5]) }
      if (MODE & 2) { PR_IW(u[2]) PR_IW(u[3]) }
      if (MODE & 4) { PR_MC(m[6]) PR_ME(m[7]) }
      if (MODE & 8) { PR_LX(u[7]) PR_LX(u[4]) PR_LX(u[5]) PR_LX(u[6]) }
      if (MODE & 1) {
        PR_FF(f[6]) PR_FF(f[7]) PR_FF(f[8]) PR_FF(f[9]) PR_FF(f[10]) PR_FF(f[11]) PR_FF(f[0]) PR_FF(f[1]) PR_FF(f[2]) PR_FF(f[3])
        PR_FF(f[4]) PR_FF(f[5]) PR_FF(f[6]) PR_FF(f[7]) PR_FF(f[8]) PR_FF(f[9]) PR_FF(f[10]) PR_FF(f[11]) PR_FF(f[0]) PR_FF(f[1])
        PR_FF(f[2]) PR_FF(f[3]) PR_FF(f[4]) PR_FF(f[5]) PR_FF(f[6]) PR_FF(f[7]) PR_FF(f[8]) PR_FF(f[9]) PR_FF(f[10]) PR_FF(f[11])
      }
    }
    if (MODE & 16) {  // once per block: the block-head LDS.128 and the fold's F2I + I2F
      const float4 t = sh[(threadIdx.x + it) & 127];
      ld += t.x;
      asm volatile("{\n\t.reg .s32 t;\n\tcvt.rni.s32.f32 t, %0;\n\tcvt.rn.f32.s32 %0, t;\n\t}" : "+f"(m[7]));
    }
  }
  const long long t1 = clock64();
  float acc = ld;
  uint32_t ua = 0;
#pragma unroll
  for (int j = 0; j < 12; ++j) acc += f[j];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    ua ^= u[j];
    acc += m[j];
  }
  if (static_cast<double>(acc) + static_cast<double>(ua) == 12345.0) out[threadIdx.x] = acc;
  if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

// ---------------------------------------------------------------------------------------------
// Fifth table: the fp64 Euler-Maruyama loop (config[4]) as independent chains, per Philox block:
// 114 DFMA + 22 DMUL + 12 DADD, 16 x (IMAD.WIDE + LOP3), 6 I2F.F64 + 2 MUFU.RSQ64H, 19 integer moves /
// multiplies on the FMA pipe (IMAD.MOV, IMAD.U32), 41 ALU-pipe instructions, 5 LDS.128.
// MODE bits: 1 FP64, 2 Philox, 4 conversions + MUFU, 8 ALU, 16 FMA-pipe integer, 32 LDS.
// ---------------------------------------------------------------------------------------------
#define PR_DF(r) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(r) : "d"(db), "d"(dc));
#define PR_DM(r) asm volatile("mul.rn.f64 %0, %0, %1;" : "+d"(r) : "d"(db));
#define PR_DA(r) asm volatile("add.rn.f64 %0, %0, %1;" : "+d"(r) : "d"(dc));
#define PR_IM(r) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r) : "r"(ub), "r"(uc));
#define PR_ID(r, x) asm volatile("cvt.rn.f64.s32 %0, %1;" : "=d"(r) : "r"(x));
#define PR_RS(r) asm volatile("rsqrt.approx.ftz.f64 %0, %0;" : "+d"(r));

template <int MODE>
__global__ void __launch_bounds__(128) f64_mix_kernel(int iters, const float* __restrict__ in,
                                                      float* __restrict__ out,
                                                      long long* __restrict__ cycles) {
  __shared__ double2 sh[128];
  double d[12], cv[3], rs = 1.5;
  uint32_t u[8];
  const double db = static_cast<double>(in[0]), dc = static_cast<double>(in[1]);
  const uint32_t ub = __float_as_uint(in[2]) | 1u, uc = __float_as_uint(in[3]);
#pragma unroll
  for (int j = 0; j < 12; ++j) d[j] = static_cast<double>(in[4]) + j + threadIdx.x;
#pragma unroll
  for (int j = 0; j < 8; ++j) u[j] = ub * (j + 3) + threadIdx.x;
  cv[0] = cv[1] = cv[2] = 0;
  sh[threadIdx.x] = make_double2(db, dc);
  __syncthreads();
  double ld = 0;
  const long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int q = 0; q < 2; ++q) {  // half a block: 57 DFMA, 11 DMUL, 6 DADD, 8 IW, 3 I2F, 1 RSQ, 20 ALU, 10 IMAD
      if (MODE & 1) { PR_DF(d[0]) PR_DF(d[1]) PR_DF(d[2]) PR_DF(d[3]) PR_DM(d[4]) PR_DF(d[5]) PR_DF(d[6]) PR_DA(d[7]) }
      if (MODE & 2) { PR_IW(u[0]) PR_IW(u[1]) }
      if (MODE & 4) { PR_ID(cv[0], u[4]) }
      if (MODE & 8) { PR_LX(u[4]) PR_LX(u[5]) PR_LX(u[6]) PR_LX(u[7]) PR_LX(u[4]) }
      if (MODE & 16) { PR_IM(u[5]) PR_IM(u[6]) PR_IM(u[7]) }
      if (MODE & 1) { PR_DF(d[8]) PR_DF(d[9]) PR_DF(d[10]) PR_DM(d[11]) PR_DF(d[0]) PR_DF(d[1]) PR_DF(d[2]) PR_DF(d[3]) PR_DM(d[4]) PR_DA(d[5]) }
      if (MODE & 2) { PR_IW(u[2]) PR_IW(u[3]) }
      if (MODE & 32) { const double2 t = sh[(threadIdx.x + it + q) & 127]; ld += t.x; }
      if (MODE & 8) { PR_LX(u[5]) PR_LX(u[6]) PR_LX(u[7]) PR_LX(u[4]) PR_LX(u[5]) }
      if (MODE & 1) { PR_DF(d[6]) PR_DF(d[7]) PR_DF(d[8]) PR_DF(d[9]) PR_DM(d[10]) PR_DF(d[11]) PR_DF(d[0]) PR_DF(d[1]) PR_DM(d[2]) PR_DA(d[3]) }
      if (MODE & 4) { PR_ID(cv[1], u[5]) PR_RS(rs) }
      if (MODE & 16) { PR_IM(u[4]) PR_IM(u[5]) PR_IM(u[6]) }
      if (MODE & 2) { PR_IW(u[0]) PR_IW(u[1]) }
      if (MODE & 1) { PR_DF(d[4]) PR_DF(d[5]) PR_DF(d[6]) PR_DF(d[7]) PR_DM(d[8]) PR_DF(d[9]) PR_DF(d[10]) PR_DF(d[11]) PR_DM(d[0]) PR_DA(d[1]) }
      if (MODE & 8) { PR_LX(u[6]) PR_LX(u[7]) PR_LX(u[4]) PR_LX(u[5]) PR_LX(u[6]) }
      if (MODE & 32) { const double2 t = sh[(threadIdx.x + 2 * it + q) & 127]; ld += t.y; }
      if (MODE & 1) { PR_DF(d[2]) PR_DF(d[3]) PR_DF(d[4]) PR_DF(d[5]) PR_DM(d[6]) PR_DF(d[7]) PR_DF(d[8]) PR_DF(d[9]) PR_DM(d[10]) PR_DA(d[11]) }
      if (MODE & 2) { PR_IW(u[2]) PR_IW(u[3]) }
      if (MODE & 4) { PR_ID(cv[2], u[6]) }
      if (MODE & (16 | 64)) { PR_IM(u[7]) PR_IM(u[4]) PR_IM(u[5]) PR_IM(u[6]) }  // 64: only these 4 (8 per block)
      if (MODE & 8) { PR_LX(u[7]) PR_LX(u[4]) PR_LX(u[5]) PR_LX(u[6]) PR_LX(u[7]) }
      if (MODE & 1) {
        PR_DF(d[0]) PR_DF(d[1]) PR_DF(d[2]) PR_DF(d[3]) PR_DM(d[4]) PR_DF(d[5]) PR_DF(d[6]) PR_DF(d[7]) PR_DM(d[8]) PR_DA(d[9])
        PR_DF(d[10]) PR_DF(d[11]) PR_DF(d[0]) PR_DF(d[1]) PR_DM(d[2]) PR_DF(d[3]) PR_DF(d[4]) PR_DF(d[5]) PR_DM(d[6]) PR_DA(d[7])
        PR_DF(d[8]) PR_DF(d[9]) PR_DF(d[10]) PR_DF(d[11]) PR_DF(d[0]) PR_DF(d[1])
      }
    }
    if (MODE & 32) { const double2 t = sh[(threadIdx.x + 3 * it) & 127]; ld += t.x; }
  }
  const long long t1 = clock64();
  double acc = ld + cv[0] + cv[1] + cv[2] + rs;
  uint32_t ua = 0;
#pragma unroll
  for (int j = 0; j < 12; ++j) acc += d[j];
#pragma unroll
  for (int j = 0; j < 8; ++j) ua ^= u[j];
  if (acc + static_cast<double>(ua) == 12345.0) out[threadIdx.x] = static_cast<float>(acc);
  if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

#define DEFINE_MIX_ROW(fn, kern)                                                                       \
  template <int MODE>                                                                                  \
  double fn(const Dev& d, int ctas_per_sm) {                                                           \
    const int iters = 10000, grid = d.n_sm * ctas_per_sm;                                              \
    kern<MODE><<<grid, 128>>>(200, d.in, d.out, d.cyc);                                                \
    kern<MODE><<<grid, 128>>>(iters, d.in, d.out, d.cyc);                                              \
    CK(cudaDeviceSynchronize());                                                                       \
    std::vector<long long> c(grid);                                                                    \
    CK(cudaMemcpy(c.data(), d.cyc, sizeof(long long) * grid, cudaMemcpyDeviceToHost));                 \
    return static_cast<double>(*std::max_element(c.begin(), c.end())) / iters / ctas_per_sm;           \
  }
DEFINE_MIX_ROW(heun_mix, heun_mix_kernel)
DEFINE_MIX_ROW(f64_mix, f64_mix_kernel)

// ---------------------------------------------------------------------------------------------
// Sixth table: dependent-issue latency.  ONE warp, one chain: every instruction waits for the one before.
// Cycles per link of the chain (SM clocks), the quantity that bounds the small-ensemble kernel, where one
// warp per scheduler integrates and nothing hides the recurrence v_n -> x_{n+1} -> force -> v_{n+2}.
// ---------------------------------------------------------------------------------------------
enum Chain { CH_FFMA, CH_FMUL, CH_FORCE, CH_COS, CH_DFMA, CH_IMADW, CH_LOP3, CH_LDS, CH_EMSTEP, CH_EMSTEP2, N_CHAINS };
static const char* CHAIN_NAME[N_CHAINS] = {
    "FFMA -> FFMA", "FMUL -> FMUL", "FFMA -> FMUL.RZ -> MUFU.COS -> FFMA -> FFMA (force of x)",
    "FMUL.RZ -> MUFU.COS", "DFMA -> DFMA", "IMAD.WIDE -> LOP3 (one Philox half round)", "LOP3 -> LOP3",
    "LDS -> FFMA (shared-memory load to use)", "EM recurrence, sums in round 1's order: cos -> f -> a_v -> v + dt a_v -> + noise",
    "EM recurrence as em_step has it now: cos -> f + h -> (v + noise) + dt a_v"};

template <int CH>
__global__ void __launch_bounds__(32) chain_kernel(int iters, const float* __restrict__ in,
                                                   float* __restrict__ out, long long* __restrict__ cycles) {
  __shared__ float sh[64];
  float x = in[4] + threadIdx.x * 1e-3f, v = in[5];
  const float fb = in[0], fc = in[1];
  double dx = x;
  const double db = fb, dc = fc;
  uint32_t u = __float_as_uint(in[2]) | 1u;
  const uint32_t ub = __float_as_uint(in[3]);
  sh[threadIdx.x] = fc;
  sh[threadIdx.x + 32] = fc;
  __syncthreads();
  const long long t0 = clock64();
#pragma unroll 1
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int q = 0; q < 16; ++q) {
      if (CH == CH_FFMA) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x) : "f"(fb), "f"(fc));
      if (CH == CH_FMUL) asm volatile("mul.rn.f32 %0, %0, %1;" : "+f"(x) : "f"(fb));
      if (CH == CH_FORCE)
        asm volatile("{\n\t.reg .f32 a, c, p;\n\tfma.rn.f32 a, %0, %1, %2;\n\tcos.approx.ftz.f32 c, a;\n\t"
                     "fma.rn.f32 p, c, %1, %2;\n\tfma.rn.f32 %0, p, c, %2;\n\t}" : "+f"(x) : "f"(fb), "f"(fc));
      if (CH == CH_COS) asm volatile("cos.approx.ftz.f32 %0, %0;" : "+f"(x));
      if (CH == CH_DFMA) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(dx) : "d"(db), "d"(dc));
      if (CH == CH_IMADW)
        asm volatile("{\n\t.reg .u64 p;\n\t.reg .u32 lo, hi;\n\tmul.wide.u32 p, %0, 0xD2511F53;\n\t"
                     "mov.b64 {lo, hi}, p;\n\tlop3.b32 %0, lo, hi, %1, 0x96;\n\t}" : "+r"(u) : "r"(ub));
      if (CH == CH_LOP3) asm volatile("lop3.b32 %0, %0, %1, %1, 0x96;" : "+r"(u) : "r"(ub));
      if (CH == CH_LDS) {
        float t;
        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(t) : "r"(static_cast<uint32_t>(__cvta_generic_to_shared(sh)) +
                                                                 ((__float_as_uint(x) & 31u) << 2)));
        asm volatile("fma.rn.f32 %0, %1, %2, %0;" : "+f"(x) : "f"(t), "f"(fb));
      }
      if (CH == CH_EMSTEP) {
        // two Euler-Maruyama steps of (x, v) with the force from the OLD position: x' = x + dt v,
        // v' = v + dt (g v + k1 c + k2 c^2) + noise; e dropped (its chain is shorter)
        asm volatile("{\n\t.reg .f32 a, c, p, f, w;\n\t"
                     "fma.rn.f32 a, %0, %2, %3;\n\tcos.approx.ftz.f32 c, a;\n\tfma.rn.f32 p, c, %2, %3;\n\t"
                     "fma.rn.f32 f, p, c, %3;\n\tfma.rn.f32 w, %2, %1, f;\n\tfma.rn.f32 %0, %3, %1, %0;\n\t"
                     "fma.rn.f32 w, %3, w, %1;\n\tfma.rn.f32 %1, %2, %3, w;\n\t}"
                     : "+f"(x), "+f"(v) : "f"(fb), "f"(fc));
      }
      if (CH == CH_EMSTEP2) {
        // the same step with the sums in em_step's order: h = g v + k0 and v + noise do not wait for the
        // cosine; a_v = (k2 c + k1) c + h; v' = dt a_v + (v + noise)
        asm volatile("{\n\t.reg .f32 a, c, p, h, w, t;\n\t"
                     "fma.rn.f32 a, %0, %2, %3;\n\tcos.approx.ftz.f32 c, a;\n\tfma.rn.f32 h, %2, %1, %3;\n\t"
                     "fma.rn.f32 t, %2, %3, %1;\n\tfma.rn.f32 p, c, %2, %3;\n\tfma.rn.f32 w, p, c, h;\n\t"
                     "fma.rn.f32 %0, %3, %1, %0;\n\tfma.rn.f32 %1, %3, w, t;\n\t}"
                     : "+f"(x), "+f"(v) : "f"(fb), "f"(fc));
      }
    }
  }
  const long long t1 = clock64();
  if (static_cast<double>(x) + v + dx + u == 12345.0) out[threadIdx.x] = x;
  if (threadIdx.x == 0) cycles[0] = t1 - t0;
}

template <int CH>
void chain_row(const Dev& d) {
  const int iters = 4000;
  chain_kernel<CH><<<1, 32>>>(100, d.in, d.out, d.cyc);
  chain_kernel<CH><<<1, 32>>>(iters, d.in, d.out, d.cyc);
  CK(cudaDeviceSynchronize());
  long long c = 0;
  CK(cudaMemcpy(&c, d.cyc, sizeof(c), cudaMemcpyDeviceToHost));
  std::printf("%-72s %8.2f\n", CHAIN_NAME[CH], static_cast<double>(c) / iters / 16);
}

// ---------------------------------------------------------------------------------------------
// Seventh table: accuracy of the fast fp32 Box-Muller (abm_device.cuh: box_muller_f32, MUFU.LG2 / SQRT / COS /
// SIN) over ALL 2^23 values each uniform can take, against fp64 (sigma = 1).  lg2.approx is accurate to 2^-22
// absolutely, so the radius rho = sqrt(-2 ln u1) loses relative accuracy as u1 -> 1; DESIGN.md 7 quotes these rows.
// ---------------------------------------------------------------------------------------------
__device__ unsigned long long g_bm[6];  // bit patterns of non-negative doubles: max-reduce as integers
__global__ void bm_accuracy_kernel() {
  const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;  // 23-bit uniform index
  const uint32_t w = k << 9;
  const float s2 = 2.0f;   // 2 sigma^2, sigma = 1
  const float bm_o = static_cast<float>(2.0 * 3.141592653589793 * 0x1p-24 - 3.0 * 3.141592653589793);
  const abm::Normal2f z = abm::box_muller_f32(w, w, s2, bm_o);
  const double u = (static_cast<double>(k) + 0.5) * 0x1p-23;
  const double rho = sqrt(-2.0 * log(u));
  const double e_rho = fabs(static_cast<double>(z.rho) - rho);
  // Normal2f carries -cos, -sin of 2 pi u (NEGATED)
  const double e_cs = fabs(-static_cast<double>(z.cs) - cospi(2.0 * u));
  const double e_sn = fabs(-static_cast<double>(z.sn) - sinpi(2.0 * u));
  const bool finite = isfinite(z.rho) && isfinite(z.cs) && isfinite(z.sn);
  atomicMax(&g_bm[0], static_cast<unsigned long long>(__double_as_longlong(e_rho)));
  atomicMax(&g_bm[1], static_cast<unsigned long long>(__double_as_longlong(e_rho / rho)));
  atomicMax(&g_bm[2], static_cast<unsigned long long>(__double_as_longlong(e_cs)));
  atomicMax(&g_bm[3], static_cast<unsigned long long>(__double_as_longlong(e_sn)));
  if (!finite) atomicAdd(&g_bm[4], 1ull);
  if (e_rho > 1e-5) atomicMax(&g_bm[5], static_cast<unsigned long long>(__double_as_longlong(1.0 - u)));
}
static void bm_accuracy_table() {
  unsigned long long h[6] = {0, 0, 0, 0, 0, 0};
  CK(cudaMemcpyToSymbol(g_bm, h, sizeof(h)));
  bm_accuracy_kernel<<<(1u << 23) / 256, 256>>>();
  CK(cudaDeviceSynchronize());
  CK(cudaMemcpyFromSymbol(h, g_bm, sizeof(h)));
  auto d = [&](int i) { double v; memcpy(&v, &h[i], 8); return v; };
  std::printf("# fast fp32 Box-Muller (box_muller_f32, sigma = 1) over all 2^23 uniforms, against fp64\n");
  std::printf("%-72s %10.3e\n", "max |rho - sqrt(-2 ln u1)|", d(0));
  std::printf("%-72s %10.3e\n", "max relative error of rho", d(1));
  std::printf("%-72s %10.3e\n", "largest 1 - u1 with an absolute error of rho above 1e-5", d(5));
  std::printf("%-72s %10.3e\n", "max |cos| error", d(2));
  std::printf("%-72s %10.3e\n", "max |sin| error", d(3));
  std::printf("%-72s %10llu\n", "non-finite results", h[4]);
}

int main() {
  Dev d;
  cudaDeviceProp p;
  CK(cudaGetDeviceProperties(&p, 0));
  d.n_sm = p.multiProcessorCount;
  int clk_khz = 0;
  CK(cudaDeviceGetAttribute(&clk_khz, cudaDevAttrClockRate, 0));
  std::printf("# device %s, %d SMs, max SM clock %.0f MHz\n", p.name, d.n_sm, clk_khz / 1e3);
  const float h_in[8] = {0.9999f, 1e-7f, 1.7f, 2.9f, 1.0f, 3.3f, 2.0f, 5.5f};
  CK(cudaMalloc(&d.in, sizeof(h_in)));
  CK(cudaMemcpy(d.in, h_in, sizeof(h_in), cudaMemcpyHostToDevice));
  CK(cudaMemcpyToSymbol(c_k, h_in, 16));
  CK(cudaMalloc(&d.out, 4096));
  CK(cudaMalloc(&d.cyc, sizeof(long long) * d.n_sm * 16));
  std::printf("# warp-lane operations per clock per SM (slowest CTA), 8 independent chains/thread\n");
  std::printf("%-22s %8s %8s %8s %8s\n", "instruction", "4 warps", "8 warps", "16 warps", "32 warps");
  single<FFMA_RRR>(d); single<FFMA_RRC>(d); single<FFMA_RIR>(d); single<FMUL_RR>(d);
  single<FADD_RR>(d); single<IMAD_LO>(d); single<IMAD_WIDE_R>(d); single<IMAD_WIDE_I>(d);
  single<LOP3_XOR3>(d); single<IADD3>(d); single<SHF_R>(d);
  single<MUFU_COS>(d); single<MUFU_SIN>(d); single<MUFU_LG2>(d); single<MUFU_SQRT>(d);
  single<MUFU_RSQ>(d); single<MUFU_EX2>(d); single<MUFU_RCP>(d);
  single<DFMA_>(d); single<DMUL_>(d); single<DADD_>(d); single<I2F_>(d); single<F2I_>(d);
  single<FFMA2_>(d); single<FRND_>(d);
  std::printf("# mixes, 32 warps/SM, one to one\n");
  mix<FFMA_RRR, LOP3_XOR3>(d);
  mix<FFMA_RRR, IMAD_WIDE_I>(d);
  mix<FFMA_RRR, IMAD_LO>(d);
  mix<FFMA_RRR, MUFU_COS>(d);
  mix<FFMA_RRR, FMUL_RR>(d);
  mix<IMAD_WIDE_I, LOP3_XOR3>(d);
  mix<LOP3_XOR3, IADD3>(d);
  mix<MUFU_COS, MUFU_LG2>(d);
  mix<MUFU_COS, LOP3_XOR3>(d);
  mix<DFMA_, FFMA_RRR>(d);
  mix<DFMA_, LOP3_XOR3>(d);
  mix<DFMA_, IMAD_WIDE_I>(d);
  mix<FFMA2_, IMAD_WIDE_I>(d);
  mix<FFMA2_, IMAD_LO>(d);
  mix<FFMA2_, LOP3_XOR3>(d);
  mix<FFMA2_, MUFU_COS>(d);
  mix<FFMA2_, FFMA_RRR>(d);
  mix<FRND_, FFMA_RRR>(d);
  mix<FRND_, MUFU_LG2>(d);
  mix<I2F_, MUFU_LG2>(d);
  mix<I2F_, LOP3_XOR3>(d);
  mix<I2F_, FFMA_RRR>(d);
  std::printf("# the same one-to-one mixes with ONE warp per scheduler (4 warps/SM): what a single warp can issue\n");
  mix1<FFMA_RRR, LOP3_XOR3>(d);
  mix1<FFMA_RRR, FMUL_RR>(d);
  mix1<FFMA_RRR, MUFU_COS>(d);
  mix1<FFMA2_, FFMA_RRR>(d);
  mix1<FFMA2_, LOP3_XOR3>(d);
  std::printf("# the fp32 Euler-Maruyama step-loop mix as independent chains: SM cycles per warp and scheduler for\n"
              "# one Philox block (four steps); the step kernel itself: kernel time x clock / (steps / 4) / warps per scheduler\n");
  std::printf("%-44s %8s %8s %8s\n", "instructions per block", "4 CTA/SM", "9 CTA/SM", "12 CTA/SM");
  loop_mix_row<1>(d, "54 FFMA/FMUL/FADD");
  loop_mix_row<2>(d, "16 (IMAD.WIDE + LOP3)");
  loop_mix_row<4>(d, "6 (FMUL.RZ + MUFU.COS) + 6 MUFU");
  loop_mix_row<8>(d, "8 LOP3");
  loop_mix_row<3>(d, "FP32 + Philox");
  loop_mix_row<5>(d, "FP32 + MUFU");
  loop_mix_row<6>(d, "Philox + MUFU");
  loop_mix_row<7>(d, "FP32 + Philox + MUFU");
  loop_mix_row<15>(d, "all (the step loop's mix, 118 instructions)");
  std::printf("# the fp32 Heun + tilt step-loop mix (config[3]) as independent chains: SM cycles per warp and scheduler\n"
              "# for one Philox block (four steps)\n");
  std::printf("%-44s %8s %8s %8s\n", "instructions per block", "4 CTA/SM", "8 CTA/SM", "12 CTA/SM");
#define ROW(fn, mode, name) std::printf("%-44s %8.1f %8.1f %8.1f\n", name, fn<mode>(d, 4), fn<mode>(d, 8), fn<mode>(d, 12));
  ROW(heun_mix, 1, "120 FFMA/FADD/FMUL")
  ROW(heun_mix, 2, "16 (IMAD.WIDE + LOP3)")
  ROW(heun_mix, 4, "10 (FMUL.RZ + MUFU.COS) + 6 MUFU")
  ROW(heun_mix, 3, "FP32 + Philox")
  ROW(heun_mix, 7, "FP32 + Philox + MUFU")
  ROW(heun_mix, 15, "FP32 + Philox + MUFU + 14 ALU")
  ROW(heun_mix, 31, "all (+ 4 LDG, LDS.128, F2I, I2F: 199 instr.)")
#undef ROW
  std::printf("# the fp64 Euler-Maruyama step-loop mix (config[4]) as independent chains: SM cycles per warp and scheduler\n"
              "# for one Philox block (four steps)\n");
  std::printf("%-44s %8s %8s %8s\n", "instructions per block", "3 CTA/SM", "5 CTA/SM", "8 CTA/SM");
#define ROW(fn, mode, name) std::printf("%-44s %8.1f %8.1f %8.1f\n", name, fn<mode>(d, 3), fn<mode>(d, 5), fn<mode>(d, 8));
  ROW(f64_mix, 1, "114 DFMA + 22 DMUL + 12 DADD")
  ROW(f64_mix, 2, "16 (IMAD.WIDE + LOP3)")
  ROW(f64_mix, 3, "FP64 + Philox")
  ROW(f64_mix, 17, "FP64 + 20 IMAD (moves on the FMA pipe)")
  ROW(f64_mix, 9, "FP64 + 40 ALU")
  ROW(f64_mix, 5, "FP64 + 6 I2F.F64 + 2 MUFU.RSQ64H")
  ROW(f64_mix, 33, "FP64 + 5 LDS.128")
  ROW(f64_mix, 19, "FP64 + Philox + 20 IMAD")
  ROW(f64_mix, 63, "all (the fp64 loop's mix, 257 instructions)")
  ROW(f64_mix, 47, "all but the 20 IMAD")
  ROW(f64_mix, 111, "all with 8 IMAD instead of 20 (the loop of round 2: 227 instructions)")
#undef ROW
  std::printf("# dependent-issue latency: one warp, one chain; SM cycles per link\n");
  chain_row<CH_FFMA>(d); chain_row<CH_FMUL>(d); chain_row<CH_COS>(d); chain_row<CH_FORCE>(d);
  chain_row<CH_EMSTEP>(d); chain_row<CH_EMSTEP2>(d); chain_row<CH_DFMA>(d); chain_row<CH_IMADW>(d); chain_row<CH_LOP3>(d); chain_row<CH_LDS>(d);
  bm_accuracy_table();
  return 0;
}
