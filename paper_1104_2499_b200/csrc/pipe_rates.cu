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
#include <vector>
#include <algorithm>
#include <cuda_runtime.h>

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
  "FMUL+MUFU.COS", "FMUL+MUFU.SIN", "MUFU.LG2", "MUFU.SQRT", "MUFU.RSQ", "MUFU.EX2", "MUFU.RCP",
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
  if (OP == MUFU_RCP) asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(r.f[j]));
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
  const double r8 = run<OP, N_OPS>(d, 256, 1, 2000);    // 2 warps / scheduler
  const double r16 = run<OP, N_OPS>(d, 512, 1, 2000);   // 4 warps / scheduler
  const double r32 = run<OP, N_OPS>(d, 1024, 1, 1000);  // 8 warps / scheduler
  const double w = OP == FFMA2_ ? 2.0 : 1.0;  // two fp32 FMAs per FFMA2
  std::printf("%-22s %8.1f %8.1f %8.1f\n", OP_NAME[OP], w * r8, w * r16, w * r32);
}

template <int OPA, int OPB>
void mix(const Dev& d) {
  const double r = run<OPA, OPB>(d, 1024, 1, 1000);
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
  std::printf("%-22s %8s %8s %8s\n", "instruction", "8 warps", "16 warps", "32 warps");
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
  return 0;
}
