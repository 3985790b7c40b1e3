// abm.cu -- host side of the C ABI declared in include/abm.h.
//
// Owns the context (state arrays, coefficient table, reduction scratch), precomputes the
// per-set coefficients in fp64, and enqueues the kernels of abm_kernels.cuh on the caller's
// stream.  There is no CPU fallback: every step of the path runs in those kernels.
#include "abm.h"

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <thread>
#include <unordered_set>
#include <vector>

#include "abm_kernels.cuh"

namespace {

using namespace abm;

constexpr uint32_t CTX_MAGIC = 0x41424d31u;      // "ABM1"
constexpr uint32_t MAX_LAUNCH_STEPS = 1u << 30;  // steps per launch without a tilt table
constexpr uint32_t TILT_CHUNK = 1u << 16;        // steps per launch with a tilt table

static_assert(sizeof(abm_moment) == 80, "abm_moment is 80 bytes (include/abm.h)");
static_assert(sizeof(MomentRec) == sizeof(abm_moment), "MomentRec mirrors abm_moment");
static_assert(N_SUMS == ABM_N_SUMS, "sum count");

}  // namespace

struct abm_ctx {
  uint32_t magic;
  int device;
  cudaStream_t stream;
  uint32_t precision, integrator, init_v, snap_every, rng;
  uint32_t n_sets;
  bool tilt;
  bool precise;         // fp32 accuracy mode resolved at create (include/abm.h, abm_params.accuracy)
  bool split_coefs;     // several sets that differ only in D, q, F0, A, v0, e0: COEF_SPLIT step kernel
  bool beyond_tolerance;  // some set is stiffer than that mode is good for (ABM_ACCURACY_BEYOND_TOLERANCE)
  uint64_t n_particles, n_traj, seed, step, traj_base, set_stride;
  double dt, omega;
  uint64_t small_max_traj;  // ensembles up to this size run step_kernel_small (abm_params.step_kernel)
  double tilt_k0, tilt_A;  // what the tilt table holds: k0 + A cos(omega t) of the one set, or (0, 1)
  size_t real_size;
  void *x, *v, *e;      // state, SoA, Real[n_traj]
  void* xl;             // precise fp32 mode only: fraction word of the fixed-point position, [n_traj]
  void* xh;             //   and its whole periods (the x array then holds the float offset)
  uint4* rng_state;     // xorshift state per trajectory (ABM_RNG_XORSHIFT128 only)
  void* coef_table;     // Coef<Real>[n_sets]
  void* tilt_table;     // Real[TILT_CHUNK + 8]: 3 elements of alignment shift, 3 of lead-in, the chunk, t_{n+1} of its last step
  double2* noise_tables;  // fp64 only: Box-Muller circle and log tables (NoiseTables), [NOISE_TABLE_N]
  double* partial;      // [n_sets * blocks_per_set][7]
  double* sums;         // [n_sets][8]
  MomentRec* moments;   // [n_sets]
  void* host_coefs;     // host copy of the coefficient table (source of the async upload)
  void* frame;          // staging frame for abm_snapshot_host (lazily allocated)
  size_t frame_bytes;
  uint32_t mom_block, mom_slice, blocks_per_set;
  void* snap;
  uint32_t snap_stride;
  int sticky;           // first CUDA error seen
  Coef<float> coef0_f;  // set 0 (kernel-parameter copy for single-set runs)
  Coef<double> coef0_d;
};

namespace {

#define ABM_CK(ctx, call)                                   \
  do {                                                      \
    cudaError_t err__ = (call);                             \
    if (err__ != cudaSuccess) {                             \
      if (ctx) (ctx)->sticky = static_cast<int>(err__);     \
      return err__ == cudaErrorMemoryAllocation ? ABM_ENOMEM : ABM_ECUDA; \
    }                                                       \
  } while (0)

template <typename Real>
Coef<Real> make_coef(const abm_params& p) {
  const double two_pi = 6.283185307179586476925286766559;
  Coef<Real> c;
  std::memset(&c, 0, sizeof(c));
  c.dt = static_cast<Real>(p.dt);
  c.hdt = static_cast<Real>(0.5 * p.dt);
  c.gamma0 = static_cast<Real>(p.gamma0);
  c.d = static_cast<Real>(p.d);
  c.q = static_cast<Real>(p.q);
  c.c = static_cast<Real>(p.c);
  // -U'(x) = -(2pi/L) (A1 cos th + 2 A2 cos 2th) = (2pi/L) (2 A2 - A1 cos th - 4 A2 cos^2 th)
  const double g = two_pi / p.L;
  c.k0 = static_cast<Real>(g * 2.0 * p.A2 + p.F0);
  c.k1 = static_cast<Real>(-g * p.A1);
  c.k2 = static_cast<Real>(-g * 4.0 * p.A2);
  if (sizeof(Real) == 4) {
    c.th_s = static_cast<Real>(g);                      // radians
    c.th_o = static_cast<Real>(g * p.phi);
    c.s2 = static_cast<Real>(2.0 * (2.0 * p.D * p.dt));  // 2 sigma^2
  } else {
    c.th_s = static_cast<Real>(2.0 / p.L);              // half-turns (cospi)
    c.th_o = static_cast<Real>(2.0 * p.phi / p.L);
    c.s2 = static_cast<Real>(std::sqrt(2.0 * p.D * p.dt));  // sigma
  }
  c.bm_o = static_cast<Real>(two_pi * 0x1p-24 - 1.5 * two_pi);
  c.fxS = static_cast<Real>(4294967296.0 / p.L);
  c.A = static_cast<Real>(p.A);
  c.L = static_cast<Real>(p.L);
  c.v0 = static_cast<Real>(p.v0);
  c.e0 = static_cast<Real>(p.e0);
  c.sv = static_cast<Real>(p.init_v ? std::sqrt(p.D / p.gamma0) : 0.0);
  return c;
}

// dt * max|U''(x)| <= dt (2 pi / L)^2 (|A1| + 4 |A2|): the factor by which one step turns a
// position error into a velocity error.  The 100-step fp32-vs-fp64 deviation grows in proportion
// to it (3.6e-6 at 0.079 = configs[0-2], 8e-6..1e-5 at 0.39 =
// config[3], against the 1e-5 of BASELINE.json), so ABM_ACCURACY_AUTO switches to the precise
// kernels above PRECISE_ABOVE.
constexpr double PRECISE_ABOVE = 0.15;
// ... and beyond PRECISE_GOOD_TO even the precise kernels may miss 1e-5 (include/abm.h, "What the modes promise")
constexpr double PRECISE_GOOD_TO = 0.3;
double stiffness(const abm_params& p) {
  const double g = 6.283185307179586476925286766559 / p.L;
  return p.dt * g * g * (std::fabs(p.A1) + 4.0 * std::fabs(p.A2));
}

// Host loops over parameter sets (validation, coefficient precomputation): a sweep has up to 2^16 sets
// and the device idles meanwhile, so large tables are split over a few host threads.
template <typename F>
void parallel_sets(uint32_t n_sets, F&& body) {
  unsigned n_thr = std::thread::hardware_concurrency();
  if (n_thr > 8) n_thr = 8;
  if (n_sets < 8192 || n_thr < 2) {
    body(0u, n_sets);
    return;
  }
  std::vector<std::thread> pool;
  const uint32_t chunk = (n_sets + n_thr - 1) / n_thr;
  try {
    for (uint32_t s0 = chunk; s0 < n_sets; s0 += chunk)
      pool.emplace_back([&body, s0, chunk, n_sets] { body(s0, s0 + chunk < n_sets ? s0 + chunk : n_sets); });
  } catch (...) {  // could not start (more) threads: the rest runs here
    const uint32_t started = static_cast<uint32_t>(pool.size());
    for (auto& t : pool) t.join();
    body(0u, chunk < n_sets ? chunk : n_sets);
    if ((started + 1) * chunk < n_sets) body((started + 1) * chunk, n_sets);
    return;
  }
  body(0u, chunk < n_sets ? chunk : n_sets);
  for (auto& t : pool) t.join();
}

bool finite_all(const abm_params& p) {
  const double v[] = {p.dt, p.gamma0, p.q, p.c, p.d, p.D, p.F0, p.A, p.omega,
                      p.L,  p.A1,     p.A2, p.phi, p.v0, p.e0};
  for (double t : v)
    if (!std::isfinite(t)) return false;
  return true;
}

// What the one pass over the parameter sets finds besides validity.
struct SetFlags {
  std::atomic<int> tilt{0};   // some set has A != 0
  std::atomic<int> stiff{0};  // some set's stiffness() exceeds PRECISE_ABOVE
  std::atomic<int> very_stiff{0};  // ... exceeds PRECISE_GOOD_TO
  std::atomic<int> shape_differs{0};  // some set differs from set 0 in more than D, q, F0, A, v0, e0
};

int validate(const abm_params* params, uint64_t n_particles, uint32_t n_sets, SetFlags* flags) {
  if (!params || n_particles == 0 || n_sets == 0) return ABM_EINVAL;
  const abm_params& p0 = params[0];
  if (p0.struct_size != sizeof(abm_params)) return ABM_EINVAL;
  if (p0.precision > ABM_FP64 || p0.integrator > ABM_HEUN || p0.init_v > ABM_INIT_V_THERMAL ||
      p0.accuracy > ABM_ACCURACY_PRECISE || p0.rng > ABM_RNG_XORSHIFT128 ||
      p0.step_kernel > ABM_STEP_KERNEL_SPLIT_WARPS)
    return ABM_EINVAL;
  std::atomic<int> bad{0};
  parallel_sets(n_sets, [&](uint32_t s0, uint32_t s1) {
    bool tilt = false, stiff = false, very_stiff = false, shape_differs = false;
    for (uint32_t s = s0; s < s1; ++s) {
      const abm_params& p = params[s];
      bool ok = p.struct_size == sizeof(abm_params) && p.step_kernel == p0.step_kernel;
      ok = ok && p.precision == p0.precision && p.integrator == p0.integrator && p.init_v == p0.init_v &&
           p.accuracy == p0.accuracy && p.rng == p0.rng && p.snapshot_every == p0.snapshot_every &&
           p.dt == p0.dt && p.omega == p0.omega && p.traj_base == p0.traj_base &&
           p.traj_set_stride == p0.traj_set_stride && p.stream == p0.stream;
      ok = ok && finite_all(p) && p.dt > 0.0 && p.L > 0.0 && !(p.D < 0.0);
      ok = ok && !(p.init_v == ABM_INIT_V_THERMAL && !(p.gamma0 > 0.0));
      if (!ok) {
        bad.store(1, std::memory_order_relaxed);
        return;
      }
      tilt = tilt || p.A != 0.0;
      shape_differs = shape_differs || p.gamma0 != p0.gamma0 || p.c != p0.c || p.d != p0.d || p.L != p0.L ||
                      p.A1 != p0.A1 || p.A2 != p0.A2 || p.phi != p0.phi;
      const double S = stiffness(p);
      stiff = stiff || S > PRECISE_ABOVE;
      very_stiff = very_stiff || S > PRECISE_GOOD_TO;
    }
    if (tilt) flags->tilt.store(1, std::memory_order_relaxed);
    if (stiff) flags->stiff.store(1, std::memory_order_relaxed);
    if (very_stiff) flags->very_stiff.store(1, std::memory_order_relaxed);
    if (shape_differs) flags->shape_differs.store(1, std::memory_order_relaxed);
  });
  if (bad.load()) return ABM_EINVAL;
  // total trajectory count must fit the kernels' 64-bit indexing and 31-bit grids
  const uint64_t max_traj = static_cast<uint64_t>(0x7fffffffu) * STEP_BLOCK;
  if (n_particles > max_traj / n_sets) return ABM_EINVAL;
  if (p0.traj_set_stride != 0 && p0.traj_set_stride < n_particles) return ABM_EINVAL;
  // the global index range traj_base + (n_sets - 1) stride + n_particles - 1 must not wrap 2^64 (the
  // kernels derive the shared high word of the Philox counter from its two ends)
  const uint64_t stride = p0.traj_set_stride ? p0.traj_set_stride : n_particles;
  const uint64_t span_sets = static_cast<uint64_t>(n_sets - 1);
  if (span_sets != 0 && stride > (~0ull - (n_particles - 1)) / span_sets) return ABM_EINVAL;
  const uint64_t span = span_sets * stride + (n_particles - 1);
  if (p0.traj_base > ~0ull - span) return ABM_EINVAL;
  return ABM_OK;
}

// Device memory comes from a stream-ordered pool owned by the library (one per device, kept for
// the life of the process): after the first context of a given size, abm_create / abm_destroy cost
// microseconds and do not serialise against other users of the driver.  The pool keeps at most
// POOL_KEEP_BYTES of freed memory across synchronisation points (every BASELINE.json config fits);
// what a larger context leaves behind goes back to the driver -- and so to PyTorch's allocator, which
// cannot see into this pool -- at the next synchronisation, and abm_trim() releases the rest.
constexpr int MAX_DEVICES = 64;
constexpr uint64_t POOL_KEEP_BYTES = 1ull << 30;
std::mutex g_pool_mutex;
cudaMemPool_t g_pools[MAX_DEVICES] = {};

cudaError_t pool_for(int device, cudaMemPool_t* out) {
  if (device < 0 || device >= MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_pool_mutex);
  if (!g_pools[device]) {
    cudaMemPoolProps props;
    std::memset(&props, 0, sizeof(props));
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = device;
    cudaMemPool_t pool = nullptr;
    cudaError_t e = cudaMemPoolCreate(&pool, &props);
    if (e != cudaSuccess) return e;
    uint64_t keep = POOL_KEEP_BYTES;
    e = cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
    if (e != cudaSuccess) {
      cudaMemPoolDestroy(pool);
      return e;
    }
    g_pools[device] = pool;
  }
  *out = g_pools[device];
  return cudaSuccess;
}

cudaError_t dev_alloc(abm_ctx* c, void** p, size_t bytes) {
  cudaMemPool_t pool = nullptr;
  cudaError_t e = pool_for(c->device, &pool);
  if (e != cudaSuccess) return e;
  return cudaMallocFromPoolAsync(p, bytes ? bytes : 1, pool, c->stream);
}

void dev_free(abm_ctx* c, void* p) {
  if (p) cudaFreeAsync(p, c->stream);
}

void free_all(abm_ctx* c) {
  void* all[] = {c->x, c->v, c->e, c->xl, c->xh, c->rng_state, c->coef_table, c->tilt_table, c->noise_tables,
                 c->partial, c->sums, c->moments, c->frame};
  for (void* p : all) dev_free(c, p);
  std::free(c->host_coefs);
  c->host_coefs = nullptr;
}

// Pinned staging buffer for large coefficient tables (a sweep of 2^16 sets uploads 5 MB at every
// abm_create): one per device, kept for the life of the process, so that the table is written
// straight into page-locked memory and goes to the device by DMA instead of through a pageable
// copy (0.8 ms -> 0.2 ms for config[2]).  `done` marks the last upload that read the buffer; a
// second abm_create waits for it before overwriting.  If the buffer is taken (another thread is
// inside abm_create on the same device) or cannot be allocated, the caller falls back to malloc.
struct Staging {
  void* p = nullptr;
  size_t cap = 0;
  cudaEvent_t done = nullptr;
  bool in_use = false;
};
std::mutex g_stage_mutex;
Staging g_stage[MAX_DEVICES];
constexpr size_t STAGING_MIN_BYTES = 256 * 1024;

void* stage_acquire(int device, size_t bytes) {
  if (device < 0 || device >= MAX_DEVICES || bytes < STAGING_MIN_BYTES) return nullptr;
  std::lock_guard<std::mutex> lock(g_stage_mutex);
  Staging& st = g_stage[device];
  if (st.in_use) return nullptr;
  if (!st.done && cudaEventCreateWithFlags(&st.done, cudaEventDisableTiming) != cudaSuccess) {
    st.done = nullptr;
    cudaGetLastError();
    return nullptr;
  }
  if (cudaEventSynchronize(st.done) != cudaSuccess) {  // the previous upload has read the buffer
    cudaGetLastError();
    return nullptr;
  }
  if (st.cap < bytes) {
    if (st.p) cudaFreeHost(st.p);
    st.p = nullptr;
    st.cap = 0;
    if (cudaHostAlloc(&st.p, bytes, cudaHostAllocDefault) != cudaSuccess) {
      st.p = nullptr;
      cudaGetLastError();
      return nullptr;
    }
    st.cap = bytes;
  }
  st.in_use = true;
  return st.p;
}
void stage_release(int device, cudaStream_t stream) {
  std::lock_guard<std::mutex> lock(g_stage_mutex);
  Staging& st = g_stage[device];
  if (cudaEventRecord(st.done, stream) != cudaSuccess) {  // cannot mark: wait here instead
    cudaGetLastError();
    cudaStreamSynchronize(stream);
  }
  st.in_use = false;
}

// The fp64 Box-Muller tables (abm_device.cuh, NoiseTables<double>), computed once per process in extended
// precision (long double: 64-bit mantissa on x86-64, 113 on aarch64) and rounded to double.  An entry may
// therefore differ in its last bit between host architectures / libm versions: fp64 trajectories are bit-identical
// across runs and launch splits on one host, and agree to ~1e-16 (not bit for bit) between hosts of different kinds
// (include/abm.h says so).
const double2* host_noise_tables() {
  static const std::vector<double2>* tab = [] {
    auto* t = new std::vector<double2>(NOISE_TABLE_N);
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int i = 0; i < CIRCLE_N; ++i) {
      const long double a = two_pi * (static_cast<long double>(2 * i + 1) / (2 * CIRCLE_N));
      (*t)[i] = make_double2(static_cast<double>(cosl(a)), static_cast<double>(sinl(a)));
    }
    const long double ln2 = 0.693147180559945309417232121458176568L;
    for (int i = 0; i < LOG_N; ++i) {
      // -ln of the ROUNDED reciprocal: ln m = -ln rc + log1p(m rc - 1) holds for whatever rc is
      const double rc = static_cast<double>(1.0L / (1.0L + i / 256.0L));
      long double lnc = -logl(static_cast<long double>(rc));
      if (i >= LOG_ADJ_FROM) lnc -= ln2;
      (*t)[CIRCLE_N + i] = make_double2(rc, (i == 0 || i == LOG_N - 1) ? 0.0 : static_cast<double>(lnc));
    }
    return t;
  }();
  return tab->data();
}

template <typename Real>
int upload_coefs_and_init(abm_ctx* c, const abm_params* params) {
  // malloc path: the host copy lives as long as the context (the upload is asynchronous)
  const size_t tab_bytes = sizeof(Coef<Real>) * c->n_sets;
  Coef<Real>* tab = static_cast<Coef<Real>*>(stage_acquire(c->device, tab_bytes));
  const bool staged = tab != nullptr;
  if (!staged) {
    tab = static_cast<Coef<Real>*>(std::malloc(tab_bytes));
    if (!tab) return ABM_ENOMEM;
    c->host_coefs = tab;
  }
  parallel_sets(c->n_sets, [&](uint32_t s0, uint32_t s1) {
    for (uint32_t s = s0; s < s1; ++s) tab[s] = make_coef<Real>(params[s]);
  });
  cudaError_t up = dev_alloc(c, &c->coef_table, tab_bytes);
  if (up == cudaSuccess)
    up = cudaMemcpyAsync(c->coef_table, tab, tab_bytes, cudaMemcpyHostToDevice, c->stream);
  if (staged) stage_release(c->device, c->stream);  // also on failure: the buffer is free again
  ABM_CK(c, up);
  const uint32_t grid = static_cast<uint32_t>((c->n_traj + 255) / 256);
  init_kernel<Real><<<grid, 256, 0, c->stream>>>(
      static_cast<Real*>(c->x), static_cast<Real*>(c->v), static_cast<Real*>(c->e),
      static_cast<const Coef<Real>*>(c->coef_table), c->n_traj, c->n_particles, c->traj_base,
      c->set_stride, c->seed, c->n_sets, c->init_v, c->rng_state, static_cast<Real*>(c->xl),
      static_cast<Real*>(c->xh));
  ABM_CK(c, cudaGetLastError());
  return ABM_OK;
}

// Ensembles of at most this many CTAs of step_kernel_small PER SM run that kernel (AUTO): measured on the B200 per
// 10^4 iterations, 0.19 / 0.236 / 0.277 / 0.339 ms at up to 1 / 2 / 3 / 4 CTAs per SM against 0.297 ms for the
// one-trajectory-per-thread kernel, which is flat up to one warp per scheduler (18,944 trajectories).  148 SMs x 3
// CTAs x 32 trajectories = 14,208 trajectories.
#ifndef ABM_SMALL_MAX_CTAS_PER_SM
#define ABM_SMALL_MAX_CTAS_PER_SM 3
#endif

template <typename Real, int INTEG, bool TILT, bool PRECISE, bool XS>
cudaError_t launch_step_p(const abm_ctx* c, const StepArgs<Real>& a) {
  if constexpr (sizeof(Real) == 4 && !XS) {
    const bool frames_ok = a.snap == nullptr || a.snap_every == 0 || (a.snap_every & 3u) == 0;
    if (c->n_traj <= c->small_max_traj && (a.step0 & 3u) == 0 && (a.n_steps & 3u) == 0 &&
        a.n_steps >= 4 && frames_ok) {
      const uint32_t g = static_cast<uint32_t>((c->n_traj + SMALL_TRAJ - 1) / SMALL_TRAJ);
      if (c->n_sets == 1)
        step_kernel_small<INTEG, TILT, true, PRECISE><<<g, SMALL_BLOCK, 0, c->stream>>>(a);
      else
        step_kernel_small<INTEG, TILT, false, PRECISE><<<g, SMALL_BLOCK, 0, c->stream>>>(a);
      return cudaGetLastError();
    }
  }
  const uint32_t grid = static_cast<uint32_t>((c->n_traj + STEP_BLOCK - 1) / STEP_BLOCK);
  if (c->n_sets == 1)
    step_kernel<Real, INTEG, TILT, COEF_PARAM, PRECISE, XS><<<grid, STEP_BLOCK, 0, c->stream>>>(a);
  else if (c->split_coefs)  // the sets differ only in D, q, F0, A (config[2])
    step_kernel<Real, INTEG, TILT, COEF_SPLIT, PRECISE, XS><<<grid, STEP_BLOCK, 0, c->stream>>>(a);
  else
    step_kernel<Real, INTEG, TILT, COEF_PER_THREAD, PRECISE, XS><<<grid, STEP_BLOCK, 0, c->stream>>>(a);
  return cudaGetLastError();
}

template <typename Real, int INTEG, bool TILT, bool PRECISE>
cudaError_t launch_step_r(const abm_ctx* c, const StepArgs<Real>& a) {
  return c->rng == ABM_RNG_XORSHIFT128 ? launch_step_p<Real, INTEG, TILT, PRECISE, true>(c, a)
                                       : launch_step_p<Real, INTEG, TILT, PRECISE, false>(c, a);
}

template <typename Real, int INTEG, bool TILT>
cudaError_t launch_step_u(const abm_ctx* c, const StepArgs<Real>& a) {
  if constexpr (sizeof(Real) == 4) {  // the accuracy modes exist in fp32 only
    if (c->precise) return launch_step_r<Real, INTEG, TILT, true>(c, a);
  }
  return launch_step_r<Real, INTEG, TILT, false>(c, a);
}

template <typename Real>
cudaError_t launch_step(const abm_ctx* c, const StepArgs<Real>& a) {
  if (c->integrator == ABM_EULER_MARUYAMA)
    return c->tilt ? launch_step_u<Real, 0, true>(c, a) : launch_step_u<Real, 0, false>(c, a);
  return c->tilt ? launch_step_u<Real, 1, true>(c, a) : launch_step_u<Real, 1, false>(c, a);
}

template <typename Real>
const Coef<Real>& coef0(const abm_ctx* c);
template <>
const Coef<float>& coef0<float>(const abm_ctx* c) { return c->coef0_f; }
template <>
const Coef<double>& coef0<double>(const abm_ctx* c) { return c->coef0_d; }

// Philox round keys k0 + r W0, k1 + r W1 of the launch record (constant-bank operands of the LOP3s)
template <typename Real>
void fill_round_keys(StepArgs<Real>& a, uint64_t seed) {
  for (uint32_t r = 0; r < 10; ++r) {
    a.rk0[r] = static_cast<uint32_t>(seed) + PHILOX_W0 * r;
    a.rk1[r] = static_cast<uint32_t>(seed >> 32) + PHILOX_W1 * r;
  }
}

template <typename Real>
int step_impl(abm_ctx* c, uint64_t n_steps) {
  StepArgs<Real> a;
  a.x = static_cast<Real*>(c->x);
  a.v = static_cast<Real*>(c->v);
  a.e = static_cast<Real*>(c->e);
  a.xl = static_cast<Real*>(c->xl);
  a.xh = static_cast<Real*>(c->xh);
  a.coef_table = static_cast<const Coef<Real>*>(c->coef_table);
  a.tilt = static_cast<const Real*>(c->tilt_table);
  a.noise_tables = c->noise_tables;
  a.snap = c->snap;
  a.rng_state = c->rng_state;
  a.n_traj = c->n_traj;
  a.n_particles = c->n_particles;
  a.traj_base = c->traj_base;
  a.set_stride = c->set_stride;
  a.set_magic = set_magic_of(c->n_particles);
  a.seed = c->seed;
  fill_round_keys(a, c->seed);
  a.snap_every = c->snap_every;
  a.snap_stride = c->snap_stride;
  a.coef0 = coef0<Real>(c);
  const uint64_t g_first = c->traj_base;
  const uint64_t g_last = c->traj_base + (c->n_sets - 1) * c->set_stride + (c->n_particles - 1);
  a.traj_hi = static_cast<uint32_t>(g_first >> 32);
  a.traj_hi_shared = (g_first >> 32) == (g_last >> 32) ? 1u : 0u;
  const uint32_t chunk_max = c->tilt ? TILT_CHUNK : MAX_LAUNCH_STEPS;
  // Small ensembles: step_kernel_small takes launches of whole Philox blocks that start on a block
  // boundary, so a call is cut into [steps up to the boundary] [whole blocks] [rest]; split launches
  // are bit-identical to one launch, whichever kernel runs them.
  const bool small = sizeof(Real) == 4 && c->rng == ABM_RNG_PHILOX && c->n_traj <= c->small_max_traj &&
                     (c->snap == nullptr || c->snap_every == 0 || (c->snap_every & 3u) == 0);
  while (n_steps > 0) {
    uint32_t chunk = static_cast<uint32_t>(n_steps < chunk_max ? n_steps : chunk_max);
    if (small) {
      const uint32_t mis = static_cast<uint32_t>(c->step & 3u);
      if (mis) chunk = chunk < 4u - mis ? chunk : 4u - mis;
      else if (chunk >= 4u) chunk &= ~3u;
    }
    a.step0 = c->step;
    a.n_steps = chunk;
    if (c->tilt) {
      // The table starts at a multiple of four steps and is shifted so that the 16-byte loads of the block
      // loop (TiltCursor) are aligned.
      a.tilt_base = c->step & ~3ull;
      Real* const tab = static_cast<Real*>(c->tilt_table) +
                        tilt_table_shift<Real>(c->integrator == ABM_EULER_MARUYAMA ? 0 : 1);
      a.tilt = tab;
      const uint32_t n_tab = static_cast<uint32_t>(c->step - a.tilt_base) + chunk + 1;  // Heun reads t_{n+1} of the last step
      tilt_kernel<Real><<<(n_tab + 255) / 256, 256, 0, c->stream>>>(tab, a.tilt_base, n_tab, c->omega, c->dt,
                                                                   c->tilt_k0, c->tilt_A);
      ABM_CK(c, cudaGetLastError());
    }
    ABM_CK(c, launch_step<Real>(c, a));
    c->step += chunk;
    n_steps -= chunk;
  }
  return ABM_OK;
}

template <typename Real>
int reduce_moments(abm_ctx* c) {
  const uint32_t grid = c->n_sets * c->blocks_per_set;
  moments_partial_kernel<Real><<<grid, c->mom_block, 0, c->stream>>>(
      static_cast<const Real*>(c->x), static_cast<const Real*>(c->v),
      static_cast<const Real*>(c->e), static_cast<const Real*>(c->xl),
      static_cast<const Real*>(c->xh), static_cast<const Coef<Real>*>(c->coef_table),
      c->n_particles, c->traj_base, c->set_stride, c->seed, c->blocks_per_set, c->mom_slice,
      c->partial);
  ABM_CK(c, cudaGetLastError());
  moments_final_kernel<<<(c->n_sets + 3) / 4, 128, 0, c->stream>>>(  // one warp per set
      c->partial, c->n_sets, c->blocks_per_set, c->n_particles, c->step, c->sums, c->moments);
  ABM_CK(c, cudaGetLastError());
  return ABM_OK;
}

// Live contexts.  A handle is looked up here before it is dereferenced, so a call on a destroyed (or
// never created) handle answers ABM_ESTATE instead of reading freed memory.
std::mutex g_live_mutex;
std::unordered_set<const abm_ctx*>& live_set() {
  static std::unordered_set<const abm_ctx*>* s = new std::unordered_set<const abm_ctx*>;  // never destroyed
  return *s;
}
bool is_live(const abm_ctx* c) {
  if (!c) return false;
  std::lock_guard<std::mutex> lock(g_live_mutex);
  return live_set().count(c) != 0;
}
bool register_ctx(const abm_ctx* c) {
  std::lock_guard<std::mutex> lock(g_live_mutex);
  try {
    live_set().insert(c);
  } catch (...) {
    return false;
  }
  return true;
}
bool unregister_ctx(const abm_ctx* c) {  // true: it was live (the caller now owns its destruction)
  std::lock_guard<std::mutex> lock(g_live_mutex);
  return live_set().erase(c) != 0;
}

int check_ctx(const abm_ctx* c) {
  if (!is_live(c) || c->magic != CTX_MAGIC) return ABM_ESTATE;
  if (c->sticky) return ABM_ECUDA;
  return ABM_OK;
}

// Makes the context's device current for the duration of an API call and restores the caller's
// device afterwards, so that a process driving several GPUs may call with any device current.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  explicit DeviceGuard(const abm_ctx* c) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != c->device)
      switched = cudaSetDevice(c->device) == cudaSuccess;
  }
  ~DeviceGuard() {
    if (switched) cudaSetDevice(prev);
  }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};

bool stride_ok(const abm_ctx* c, size_t stride) {
  return c->precision == ABM_FP32 ? (stride == 8 || stride == 16) : (stride == 16 || stride == 32);
}

int write_frame(abm_ctx* c, void* dev_ptr, uint32_t stride) {
  const uint32_t grid = static_cast<uint32_t>((c->n_traj + 255) / 256);
  if (c->precision == ABM_FP32)
    snapshot_kernel<float><<<grid, 256, 0, c->stream>>>(
        static_cast<const float*>(c->x), static_cast<const float*>(c->v),
        static_cast<const float*>(c->e), static_cast<const float*>(c->xl),
        static_cast<const float*>(c->xh), static_cast<const Coef<float>*>(c->coef_table), c->n_traj, c->n_particles, c->n_sets, dev_ptr,
        stride);
  else
    snapshot_kernel<double><<<grid, 256, 0, c->stream>>>(
        static_cast<const double*>(c->x), static_cast<const double*>(c->v),
        static_cast<const double*>(c->e), nullptr, nullptr,
        static_cast<const Coef<double>*>(c->coef_table),
        c->n_traj, c->n_particles, c->n_sets, dev_ptr, stride);
  ABM_CK(c, cudaGetLastError());
  return ABM_OK;
}

}  // namespace

extern "C" {

int abm_create(const abm_params* params, uint64_t n_particles, uint32_t n_param_sets,
               uint64_t seed, abm_ctx** out) {
  if (!out) return ABM_EINVAL;
  SetFlags flags;
  const int vs = validate(params, n_particles, n_param_sets, &flags);
  if (vs != ABM_OK) return vs;
  int device = -1;
  if (cudaGetDevice(&device) != cudaSuccess) return ABM_ECUDA;  // no device: fail loudly
  abm_ctx* c = new (std::nothrow) abm_ctx;
  if (!c) return ABM_ENOMEM;
  std::memset(static_cast<void*>(c), 0, sizeof(*c));
  const abm_params& p0 = params[0];
  c->magic = CTX_MAGIC;
  c->device = device;
  c->stream = static_cast<cudaStream_t>(p0.stream);
  c->precision = p0.precision;
  c->integrator = p0.integrator;
  c->init_v = p0.init_v;
  c->snap_every = p0.snapshot_every;
  c->rng = p0.rng;
  c->n_sets = n_param_sets;
  c->n_particles = n_particles;
  c->n_traj = n_particles * n_param_sets;
  c->seed = seed;
  c->step = 0;
  c->traj_base = p0.traj_base;
  c->set_stride = p0.traj_set_stride ? p0.traj_set_stride : n_particles;
  c->dt = p0.dt;
  c->omega = p0.omega;
  c->tilt = flags.tilt.load() != 0;
  // single set: the tilt table holds k0 + A cos(omega t) (k0 = (2 pi / L) 2 A2 + F0 as in make_coef)
  c->tilt_k0 = n_param_sets == 1 ? (6.283185307179586476925286766559 / p0.L) * 2.0 * p0.A2 + p0.F0 : 0.0;
  c->tilt_A = n_param_sets == 1 ? p0.A : 1.0;
  c->real_size = c->precision == ABM_FP32 ? 4 : 8;
  // which step kernel (abm_params.step_kernel; results do not depend on it)
  int n_sm_small = 0;
  if (cudaDeviceGetAttribute(&n_sm_small, cudaDevAttrMultiProcessorCount, c->device) != cudaSuccess || n_sm_small <= 0) {
    cudaGetLastError();
    delete c;
    return ABM_ECUDA;
  }
  // SPLIT_WARPS forced: wherever its grid of 32-trajectory CTAs fits the 2^31 - 1 limit; beyond it step_kernel runs
  c->small_max_traj = p0.step_kernel == ABM_STEP_KERNEL_PER_THREAD    ? 0
                      : p0.step_kernel == ABM_STEP_KERNEL_SPLIT_WARPS ? static_cast<uint64_t>(0x7fffffffu) * SMALL_TRAJ
                      : static_cast<uint64_t>(n_sm_small) * ABM_SMALL_MAX_CTAS_PER_SM * SMALL_TRAJ;
  c->split_coefs = n_param_sets > 1 && flags.shape_differs.load() == 0;
  c->precise = false;
  if (c->precision == ABM_FP32) {
    if (p0.accuracy == ABM_ACCURACY_PRECISE) c->precise = true;
    if (p0.accuracy == ABM_ACCURACY_AUTO && flags.stiff.load() != 0) c->precise = true;
    c->beyond_tolerance = c->precise ? flags.very_stiff.load() != 0 : flags.stiff.load() != 0;
  }
  c->coef0_f = make_coef<float>(p0);
  c->coef0_d = make_coef<double>(p0);

  // moment reduction geometry: one CTA per slice of a set
  uint32_t mb = MOM_BLOCK;
  if (n_particles < MOM_BLOCK) mb = static_cast<uint32_t>((n_particles + 31) / 32 * 32);
  c->mom_block = mb;
  c->mom_slice = mb * MOM_PER_THREAD;
  const uint64_t bps = (n_particles + c->mom_slice - 1) / c->mom_slice;
  if (bps * n_param_sets > 0x7fffffffull) {
    delete c;
    return ABM_EINVAL;
  }
  c->blocks_per_set = static_cast<uint32_t>(bps);

  int rc = ABM_OK;
  auto fail = [&](int code) {
    free_all(c);
    c->magic = 0;
    delete c;
    return code;
  };
  auto alloc = [&](void** p, size_t bytes) {
    cudaError_t e = dev_alloc(c, p, bytes);
    if (e != cudaSuccess) {
      rc = e == cudaErrorMemoryAllocation ? ABM_ENOMEM : ABM_ECUDA;
      cudaGetLastError();
      return false;
    }
    return true;
  };
  const size_t state_bytes = c->real_size * c->n_traj;
  if (!alloc(&c->x, state_bytes) || !alloc(&c->v, state_bytes) || !alloc(&c->e, state_bytes) ||
      (c->precise && (!alloc(&c->xl, state_bytes) || !alloc(&c->xh, state_bytes))) ||
      (c->rng == ABM_RNG_XORSHIFT128 &&
       !alloc(reinterpret_cast<void**>(&c->rng_state), sizeof(uint4) * c->n_traj)) ||
      !alloc(reinterpret_cast<void**>(&c->partial),
             sizeof(double) * (N_SUMS - 1) * bps * n_param_sets) ||
      !alloc(reinterpret_cast<void**>(&c->sums), sizeof(double) * N_SUMS * n_param_sets) ||
      !alloc(reinterpret_cast<void**>(&c->moments), sizeof(MomentRec) * n_param_sets) ||
      (c->tilt && !alloc(&c->tilt_table, c->real_size * (TILT_CHUNK + 8))) ||
      (c->precision == ABM_FP64 &&
       !alloc(reinterpret_cast<void**>(&c->noise_tables), sizeof(double2) * NOISE_TABLE_N)))
    return fail(rc);
  if (c->noise_tables) {
    const cudaError_t e = cudaMemcpyAsync(c->noise_tables, host_noise_tables(), sizeof(double2) * NOISE_TABLE_N,
                                          cudaMemcpyHostToDevice, c->stream);
    if (e != cudaSuccess) {
      cudaGetLastError();
      return fail(ABM_ECUDA);
    }
  }
  rc = c->precision == ABM_FP32 ? upload_coefs_and_init<float>(c, params)
                                : upload_coefs_and_init<double>(c, params);
  if (rc != ABM_OK) return fail(rc);
  if (!register_ctx(c)) {
    cudaStreamSynchronize(c->stream);
    return fail(ABM_ENOMEM);
  }
  *out = c;
  return ABM_OK;
}

int abm_step(abm_ctx* c, uint64_t n_steps) {
  const int st = check_ctx(c);
  if (st != ABM_OK) return st;
  const DeviceGuard on_device(c);
  if (n_steps == 0) return ABM_OK;
  return c->precision == ABM_FP32 ? step_impl<float>(c, n_steps) : step_impl<double>(c, n_steps);
}

int abm_snapshot(abm_ctx* c, void* dev_ptr, size_t stride_bytes) {
  const int st = check_ctx(c);
  if (st != ABM_OK) return st;
  const DeviceGuard on_device(c);
  if (!dev_ptr) {
    c->snap = nullptr;
    c->snap_stride = 0;
    return ABM_OK;
  }
  if (!stride_ok(c, stride_bytes)) return ABM_EINVAL;
  if (reinterpret_cast<uintptr_t>(dev_ptr) % stride_bytes != 0) return ABM_EINVAL;
  const int rc = write_frame(c, dev_ptr, static_cast<uint32_t>(stride_bytes));
  if (rc != ABM_OK) return rc;
  c->snap = dev_ptr;
  c->snap_stride = static_cast<uint32_t>(stride_bytes);
  return ABM_OK;
}

int abm_snapshot_host(abm_ctx* c, void* host_ptr, size_t stride_bytes) {
  const int st = check_ctx(c);
  if (st != ABM_OK) return st;
  const DeviceGuard on_device(c);
  if (!host_ptr || !stride_ok(c, stride_bytes)) return ABM_EINVAL;
  const size_t bytes = stride_bytes * c->n_traj;
  if (c->frame_bytes < bytes) {
    dev_free(c, c->frame);
    c->frame = nullptr;
    c->frame_bytes = 0;
    ABM_CK(c, dev_alloc(c, &c->frame, bytes));
    c->frame_bytes = bytes;
  }
  const int rc = write_frame(c, c->frame, static_cast<uint32_t>(stride_bytes));
  if (rc != ABM_OK) return rc;
  ABM_CK(c, cudaMemcpyAsync(host_ptr, c->frame, bytes, cudaMemcpyDeviceToHost, c->stream));
  ABM_CK(c, cudaStreamSynchronize(c->stream));
  return ABM_OK;
}

int abm_moments(abm_ctx* c, abm_moment* out) {
  const int st = check_ctx(c);
  if (st != ABM_OK) return st;
  const DeviceGuard on_device(c);
  if (!out) return ABM_EINVAL;
  const int rc = c->precision == ABM_FP32 ? reduce_moments<float>(c) : reduce_moments<double>(c);
  if (rc != ABM_OK) return rc;
  ABM_CK(c, cudaMemcpyAsync(out, c->moments, sizeof(abm_moment) * c->n_sets,
                            cudaMemcpyDeviceToHost, c->stream));
  ABM_CK(c, cudaStreamSynchronize(c->stream));
  return ABM_OK;
}

int abm_moments_async(abm_ctx* c, abm_moment* out) {
  const int st = check_ctx(c);
  if (st != ABM_OK) return st;
  const DeviceGuard on_device(c);
  if (!out) return ABM_EINVAL;
  const int rc = c->precision == ABM_FP32 ? reduce_moments<float>(c) : reduce_moments<double>(c);
  if (rc != ABM_OK) return rc;
  ABM_CK(c, cudaMemcpyAsync(out, c->moments, sizeof(abm_moment) * c->n_sets,
                            cudaMemcpyDeviceToHost, c->stream));
  return ABM_OK;
}

int abm_moment_sums(abm_ctx* c, double* out) {
  const int st = check_ctx(c);
  if (st != ABM_OK) return st;
  const DeviceGuard on_device(c);
  if (!out) return ABM_EINVAL;
  const int rc = c->precision == ABM_FP32 ? reduce_moments<float>(c) : reduce_moments<double>(c);
  if (rc != ABM_OK) return rc;
  ABM_CK(c, cudaMemcpyAsync(out, c->sums, sizeof(double) * N_SUMS * c->n_sets,
                            cudaMemcpyDeviceToHost, c->stream));
  ABM_CK(c, cudaStreamSynchronize(c->stream));
  return ABM_OK;
}

int abm_moment_sums_dev(abm_ctx* c, double* dev_out) {
  const int st = check_ctx(c);
  if (st != ABM_OK) return st;
  const DeviceGuard on_device(c);
  if (!dev_out || reinterpret_cast<uintptr_t>(dev_out) % 8 != 0) return ABM_EINVAL;
  const int rc = c->precision == ABM_FP32 ? reduce_moments<float>(c) : reduce_moments<double>(c);
  if (rc != ABM_OK) return rc;
  ABM_CK(c, cudaMemcpyAsync(dev_out, c->sums, sizeof(double) * N_SUMS * c->n_sets,
                            cudaMemcpyDeviceToDevice, c->stream));
  return ABM_OK;
}

int abm_raster(abm_ctx* c, uint32_t* dev_counts, uint32_t width, uint32_t height, double v_min,
               double v_max, uint8_t* dev_rgba, uint32_t saturation) {
  const int st = check_ctx(c);
  if (st != ABM_OK) return st;
  const DeviceGuard on_device(c);
  if (!dev_counts || width == 0 || height == 0 || !(v_max > v_min) || !std::isfinite(v_min) ||
      !std::isfinite(v_max))
    return ABM_EINVAL;
  if (static_cast<uint64_t>(width) * height > 0x40000000ull) return ABM_EINVAL;  // 2^30 bins
  if (reinterpret_cast<uintptr_t>(dev_counts) % 4 != 0) return ABM_EINVAL;
  if (dev_rgba && (saturation == 0 || reinterpret_cast<uintptr_t>(dev_rgba) % 4 != 0))
    return ABM_EINVAL;
  const uint32_t n_bins = width * height;
  ABM_CK(c, cudaMemsetAsync(dev_counts, 0, sizeof(uint32_t) * n_bins, c->stream));
  int n_sm = 148;
  cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, c->device);
  const uint64_t want = (c->n_traj + RASTER_BLOCK - 1) / RASTER_BLOCK;
  const bool smem = n_bins <= RASTER_SMEM_BINS;
  // shared-memory path: few, long-lived CTAs (each pays n_bins zeroing + merging); global path: one pass
  const uint64_t cap = static_cast<uint64_t>(n_sm) * (smem ? 4 : 8);
  const uint32_t grid = static_cast<uint32_t>(want < cap ? want : cap);
  const double v_range = v_max - v_min;
  auto launch = [&](auto real_tag) {
    using Real = decltype(real_tag);
    const Real* x = static_cast<const Real*>(c->x);
    const Real* v = static_cast<const Real*>(c->v);
    const Real* xl = static_cast<const Real*>(c->xl);
    const Real* xh = static_cast<const Real*>(c->xh);
    const Coef<Real>* tab = static_cast<const Coef<Real>*>(c->coef_table);
    if (smem)
      raster_kernel<Real, true><<<grid, RASTER_BLOCK, sizeof(uint32_t) * n_bins, c->stream>>>(
          x, v, xl, xh, tab, c->n_traj, c->n_particles, c->n_sets, width, height, v_min, v_range,
          dev_counts);
    else
      raster_kernel<Real, false><<<grid, RASTER_BLOCK, 0, c->stream>>>(
          x, v, xl, xh, tab, c->n_traj, c->n_particles, c->n_sets, width, height, v_min, v_range,
          dev_counts);
  };
  if (c->precision == ABM_FP32) launch(float{}); else launch(double{});
  ABM_CK(c, cudaGetLastError());
  if (dev_rgba) {
    colormap_kernel<<<(n_bins + 255) / 256, 256, 0, c->stream>>>(dev_counts, n_bins, saturation,
                                                                 reinterpret_cast<uchar4*>(dev_rgba));
    ABM_CK(c, cudaGetLastError());
  }
  return ABM_OK;
}

int abm_time_averaged_velocity(abm_ctx* c, double* out) {
  const int st = check_ctx(c);
  if (st != ABM_OK) return st;
  if (!out || c->step == 0) return ABM_EINVAL;
  std::vector<double> sums;
  try {
    sums.resize(static_cast<size_t>(N_SUMS) * c->n_sets);
  } catch (const std::bad_alloc&) {
    return ABM_ENOMEM;
  }
  const int rc = abm_moment_sums(c, sums.data());
  if (rc != ABM_OK) return rc;
  const double t = static_cast<double>(c->step) * c->dt;
  for (uint32_t s = 0; s < c->n_sets; ++s)
    out[s] = sums[static_cast<size_t>(s) * N_SUMS + 6] / sums[static_cast<size_t>(s) * N_SUMS] / t;
  return ABM_OK;
}

int abm_moments_from_sums(const double* sums, uint32_t n_param_sets, uint64_t step,
                          abm_moment* out_moments) {
  if (!sums || !out_moments || n_param_sets == 0) return ABM_EINVAL;
  for (uint32_t s = 0; s < n_param_sets; ++s) {
    if (!(sums[static_cast<size_t>(s) * N_SUMS] >= 1.0)) return ABM_EINVAL;
    MomentRec m;
    finalize_moment(sums + static_cast<size_t>(s) * N_SUMS, step, &m);
    std::memcpy(&out_moments[s], &m, sizeof(m));
  }
  return ABM_OK;
}

int abm_get_step(const abm_ctx* c, uint64_t* out_step) {
  if (!is_live(c)) return ABM_ESTATE;
  if (!out_step) return ABM_EINVAL;
  *out_step = c->step;
  return ABM_OK;
}

int abm_get_accuracy(const abm_ctx* c, uint32_t* out_mode) {
  if (!is_live(c)) return ABM_ESTATE;
  if (!out_mode) return ABM_EINVAL;
  *out_mode = (c->precise ? ABM_ACCURACY_PRECISE : ABM_ACCURACY_FAST) |
              (c->beyond_tolerance ? ABM_ACCURACY_BEYOND_TOLERANCE : 0u);
  return ABM_OK;
}

int abm_destroy(abm_ctx* c) {
  if (!unregister_ctx(c)) return ABM_ESTATE;  // null, never created, or destroyed before
  {
    const DeviceGuard on_device(c);
    cudaStreamSynchronize(c->stream);
    free_all(c);
  }
  c->magic = 0;
  delete c;
  return ABM_OK;
}

int abm_philox_blocks(uint64_t seed, uint64_t traj_first, uint64_t n_traj, uint64_t block_first,
                      uint64_t n_blocks, uint32_t* dev_out, void* stream) {
  if (!dev_out || n_traj == 0 || n_blocks == 0) return ABM_EINVAL;
  if (reinterpret_cast<uintptr_t>(dev_out) % 16 != 0) return ABM_EINVAL;
  if (n_traj > (0x7fffffffull * 256) / n_blocks) return ABM_EINVAL;
  const uint64_t total = n_traj * n_blocks;
  philox_blocks_kernel<<<static_cast<uint32_t>((total + 255) / 256), 256, 0,
                         static_cast<cudaStream_t>(stream)>>>(
      seed, traj_first, n_traj, block_first, n_blocks, reinterpret_cast<uint4*>(dev_out));
  return cudaGetLastError() == cudaSuccess ? ABM_OK : ABM_ECUDA;
}

int abm_philox_blocks_loop(uint64_t seed, uint64_t traj_first, uint64_t n_traj, uint64_t block_first,
                           uint64_t n_blocks, uint32_t loop_shape, uint32_t frame_every_blocks,
                           uint32_t* dev_out, void* stream) {
  if (!dev_out || n_traj == 0 || n_blocks == 0 || loop_shape > 1) return ABM_EINVAL;
  if (reinterpret_cast<uintptr_t>(dev_out) % 16 != 0) return ABM_EINVAL;
  if (n_blocks > (MAX_LAUNCH_STEPS >> 2) || block_first > (~0ull >> 2) - n_blocks) return ABM_EINVAL;
  if (frame_every_blocks > (1u << 28)) return ABM_EINVAL;
  if (n_traj > static_cast<uint64_t>(0x7fffffffu) * STEP_BLOCK || traj_first > ~0ull - (n_traj - 1))
    return ABM_EINVAL;
  // the same launch record abm_step builds (step_impl): round keys on the host, shared high word of the
  // trajectory index when the range does not straddle a multiple of 2^32
  auto launch = [&](auto real_tag) {
    using Real = decltype(real_tag);
    StepArgs<Real> a;
    std::memset(static_cast<void*>(&a), 0, sizeof(a));
    a.n_traj = n_traj;
    a.n_particles = n_traj;
    a.traj_base = traj_first;
    a.set_stride = n_traj;
    a.set_magic = set_magic_of(n_traj);
    a.seed = seed;
    fill_round_keys(a, seed);
    a.step0 = block_first << 2;
    a.tilt_base = a.step0;
    a.n_steps = static_cast<uint32_t>(n_blocks << 2);
    a.snap_every = frame_every_blocks << 2;
    a.snap = frame_every_blocks ? static_cast<void*>(dev_out) : nullptr;  // only compared with null
    const uint64_t g_last = traj_first + (n_traj - 1);
    a.traj_hi = static_cast<uint32_t>(traj_first >> 32);
    a.traj_hi_shared = (traj_first >> 32) == (g_last >> 32) ? 1u : 0u;
    const uint32_t grid = static_cast<uint32_t>((n_traj + STEP_BLOCK - 1) / STEP_BLOCK);
    philox_loop_kernel<Real><<<grid, STEP_BLOCK, 0, static_cast<cudaStream_t>(stream)>>>(
        a, reinterpret_cast<uint4*>(dev_out));
  };
  if (loop_shape == 0) launch(float{}); else launch(double{});
  return cudaGetLastError() == cudaSuccess ? ABM_OK : ABM_ECUDA;
}

int abm_trim(void) {
  int device = -1;
  if (cudaGetDevice(&device) != cudaSuccess || device < 0 || device >= MAX_DEVICES) return ABM_ECUDA;
  cudaMemPool_t pool = nullptr;
  {
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    pool = g_pools[device];
  }
  if (!pool) return ABM_OK;  // nothing was ever allocated on this device
  if (cudaDeviceSynchronize() != cudaSuccess) return ABM_ECUDA;
  return cudaMemPoolTrimTo(pool, 0) == cudaSuccess ? ABM_OK : ABM_ECUDA;
}

const char* abm_strerror(int status) {
  switch (status) {
    case ABM_OK: return "ok";
    case ABM_EINVAL: return "invalid argument";
    case ABM_ENOMEM: return "out of memory";
    case ABM_ECUDA: return "CUDA error (no usable device, or a launch/copy failed)";
    case ABM_ESTATE: return "null or destroyed context";
    case ABM_ELIMIT: return "job exceeds the library's fixed built-in scratch (abm_frame_moment_sums_static)";
    default: return "unknown status";
  }
}

uint32_t abm_abi_version(void) { return 6; }

}  // extern "C"

// =================================================================================================
// abm_frame_moment_sums_static -- the moment sums of a caller-owned frame, for callers that may not
// allocate (include/abm.h says who they are).  Nothing in this section calls cudaMalloc, cudaFree, a
// memory pool or any other allocating routine; the two-pass reduction's intermediate records live in
// the file-scope array below, which belongs to the library image and therefore exists, once per GPU
// that loads the image, from load to process exit.
//
// The array is shared by every call on a GPU.  It is never cleared: pass 1 writes records
// [0, n_sets * blocks_per_set) in full and pass 2 reads exactly those, so stale contents of an
// earlier, larger call are never looked at.  Two calls whose kernels overlap on one GPU would write the
// same records -- the header tells callers to keep them on one stream.
// =================================================================================================
namespace {

constexpr uint32_t STATIC_RECORD = N_SUMS - 1;  // doubles per partial record (N is not summed)
static_assert(ABM_STATIC_SCRATCH_BYTES == ABM_STATIC_MAX_SLICES * STATIC_RECORD * sizeof(double),
              "ABM_STATIC_SCRATCH_BYTES in include/abm.h is the size of g_static_partial");

// In HOST code this name is only a handle for cudaGetSymbolAddress: it is not a device address and must
// never be handed to a kernel as is.  static_scratch_for() below resolves it.
static __device__ __align__(256) double g_static_partial[ABM_STATIC_MAX_SLICES * STATIC_RECORD];

std::mutex g_static_mutex;
double* g_static_ptr[MAX_DEVICES] = {};  // device address of g_static_partial, per GPU (null: not looked up yet)

// Device address of the scratch on `device`, which must be the CURRENT device (the runtime resolves a
// symbol for whichever GPU is current).  Looked up once per GPU, then served from the cache.
cudaError_t static_scratch_for(int device, double** out) {
  if (device < 0 || device >= MAX_DEVICES) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_ptr[device]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, g_static_partial);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_static_ptr[device] = static_cast<double*>(p);
  }
  *out = g_static_ptr[device];
  return cudaSuccess;
}

template <typename Real> struct FrameVec;
template <> struct FrameVec<float> { using V2 = float2; using V4 = float4; };
template <> struct FrameVec<double> { using V2 = double2; using V4 = double4; };

// Pass 1, the frame-reading twin of moments_partial_kernel: same grid (one CTA per slice of a set), same
// per-thread stride, same shuffle tree and same order over the warps, hence the same roundings.
template <typename Real, bool WITH_E>
__global__ void __launch_bounds__(MOM_BLOCK)
frame_moments_partial_kernel(const void* __restrict__ frame, const void* __restrict__ frame0,
                             uint64_t n_particles, uint32_t blocks_per_set, uint32_t slice,
                             double* __restrict__ partial) {
  using V2 = typename FrameVec<Real>::V2;
  using V4 = typename FrameVec<Real>::V4;
  const uint32_t set = blockIdx.x / blocks_per_set;
  const uint32_t blk = blockIdx.x - set * blocks_per_set;
  const uint64_t r0 = static_cast<uint64_t>(blk) * slice;
  uint64_t r1 = r0 + slice;
  if (r1 > n_particles) r1 = n_particles;
  double acc[STATIC_RECORD] = {0, 0, 0, 0, 0, 0, 0};
  for (uint64_t r = r0 + threadIdx.x; r < r1; r += blockDim.x) {
    const uint64_t k = static_cast<uint64_t>(set) * n_particles + r;
    double xi, vi, ei = 0.0, dx = 0.0;
    if (WITH_E) {
      const V4 s = static_cast<const V4*>(frame)[k];
      xi = static_cast<double>(s.x), vi = static_cast<double>(s.y), ei = static_cast<double>(s.z);
      if (frame0) dx = xi - static_cast<double>(static_cast<const V4*>(frame0)[k].x);
    } else {
      const V2 s = static_cast<const V2*>(frame)[k];
      xi = static_cast<double>(s.x), vi = static_cast<double>(s.y);
      if (frame0) dx = xi - static_cast<double>(static_cast<const V2*>(frame0)[k].x);
    }
    acc[0] += xi;
    acc[1] += xi * xi;
    acc[2] += vi;
    acc[3] += vi * vi;
    acc[4] += ei;
    acc[5] += dx;
    acc[6] += dx * dx;
  }
  __shared__ double sm[MOM_BLOCK / 32][STATIC_RECORD];
  const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
#pragma unroll
  for (uint32_t q = 0; q < STATIC_RECORD; ++q) {
    double t = acc[q];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) t += __shfl_xor_sync(0xffffffffu, t, off);
    if (lane == 0) sm[warp][q] = t;
  }
  __syncthreads();
  if (threadIdx.x < STATIC_RECORD) {
    double t = 0;
    const uint32_t n_warps = (blockDim.x + 31u) >> 5;
    for (uint32_t wq = 0; wq < n_warps; ++wq) t += sm[wq][threadIdx.x];
    partial[static_cast<uint64_t>(blockIdx.x) * STATIC_RECORD + threadIdx.x] = t;
  }
}

// Pass 2, moments_final_kernel without the finalised record: one warp per set adds that set's partial
// records in the same fixed order and writes the eight sums straight into the caller's buffer.
__global__ void __launch_bounds__(128)
frame_moments_final_kernel(const double* __restrict__ partial, uint32_t n_sets, uint32_t blocks_per_set,
                           uint64_t n_particles, double* __restrict__ sums) {
  const uint32_t set = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const uint32_t lane = threadIdx.x & 31u;
  if (set >= n_sets) return;  // whole warps leave together
  double s[N_SUMS];
  s[0] = static_cast<double>(n_particles);
  const double* p = partial + static_cast<uint64_t>(set) * blocks_per_set * STATIC_RECORD;
#pragma unroll
  for (uint32_t q = 0; q < STATIC_RECORD; ++q) {
    double t = 0;
    for (uint32_t b = lane; b < blocks_per_set; b += 32) t += p[static_cast<uint64_t>(b) * STATIC_RECORD + q];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) t += __shfl_xor_sync(0xffffffffu, t, off);
    s[q + 1] = t;
  }
  if (lane == 0)
    for (int q = 0; q < N_SUMS; ++q) sums[static_cast<uint64_t>(set) * N_SUMS + q] = s[q];
}

}  // namespace

extern "C" int abm_frame_moment_sums_static(const void* dev_frame, const void* dev_frame0, size_t stride_bytes,
                                            uint32_t precision, uint64_t n_particles, uint32_t n_param_sets,
                                            double* dev_out, void* stream) {
  if (!dev_frame || !dev_out || n_particles == 0 || n_param_sets == 0 || precision > ABM_FP64)
    return ABM_EINVAL;
  const size_t real_size = precision == ABM_FP32 ? 4 : 8;
  if (stride_bytes != 2 * real_size && stride_bytes != 4 * real_size) return ABM_EINVAL;
  if (reinterpret_cast<uintptr_t>(dev_frame) % stride_bytes != 0 ||
      reinterpret_cast<uintptr_t>(dev_frame0) % stride_bytes != 0 ||
      reinterpret_cast<uintptr_t>(dev_out) % sizeof(double) != 0)
    return ABM_EINVAL;
  // the reduction geometry of abm_create, so that the sums come out bit-identical to a context's
  uint32_t mb = MOM_BLOCK;
  if (n_particles < MOM_BLOCK) mb = static_cast<uint32_t>((n_particles + 31) / 32 * 32);
  const uint32_t slice = mb * MOM_PER_THREAD;
  const uint64_t bps = (n_particles + slice - 1) / slice;
  if (bps > ABM_STATIC_MAX_SLICES || bps * n_param_sets > ABM_STATIC_MAX_SLICES) return ABM_ELIMIT;
  int device = -1;
  if (cudaGetDevice(&device) != cudaSuccess) {  // no device: fail loudly, there is no CPU path
    cudaGetLastError();
    return ABM_ECUDA;
  }
  double* scratch = nullptr;  // the DEVICE address of g_static_partial on the current GPU
  if (static_scratch_for(device, &scratch) != cudaSuccess) {
    cudaGetLastError();
    return ABM_ECUDA;
  }
  const cudaStream_t st = static_cast<cudaStream_t>(stream);
  const uint32_t grid = static_cast<uint32_t>(bps) * n_param_sets;
  const uint32_t bpsu = static_cast<uint32_t>(bps);
  const bool with_e = stride_bytes == 4 * real_size;
  if (precision == ABM_FP32) {
    if (with_e)
      frame_moments_partial_kernel<float, true><<<grid, mb, 0, st>>>(dev_frame, dev_frame0, n_particles, bpsu, slice, scratch);
    else
      frame_moments_partial_kernel<float, false><<<grid, mb, 0, st>>>(dev_frame, dev_frame0, n_particles, bpsu, slice, scratch);
  } else {
    if (with_e)
      frame_moments_partial_kernel<double, true><<<grid, mb, 0, st>>>(dev_frame, dev_frame0, n_particles, bpsu, slice, scratch);
    else
      frame_moments_partial_kernel<double, false><<<grid, mb, 0, st>>>(dev_frame, dev_frame0, n_particles, bpsu, slice, scratch);
  }
  if (cudaGetLastError() != cudaSuccess) return ABM_ECUDA;
  frame_moments_final_kernel<<<(n_param_sets + 3) / 4, 128, 0, st>>>(scratch, n_param_sets, bpsu, n_particles, dev_out);
  return cudaGetLastError() == cudaSuccess ? ABM_OK : ABM_ECUDA;
}
