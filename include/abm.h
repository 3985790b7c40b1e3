/*
 * abm.h -- C ABI of the B200-native hot path of arXiv 1104.2499 (M. Zabicki, "OpenCL/OpenGL
 * approach for studying active Brownian motion"): integration of a large ensemble of
 * independent energy-depot active-Brownian trajectories on a ratchet potential, device-side
 * snapshots in place of the paper's shared OpenGL vertex buffer, and ensemble moments.
 *
 * Citations are PAPER.md line numbers (+ section / equation / figure) or BASELINE.json.
 *
 * The model (one trajectory = the paper's "work item"):
 *     dx/dt = v                                                        (implied by Eqs. 2-3)
 *     dv/dt = F0 + d e v - gamma0 v - U'(x) + A cos(omega t) + sqrt(2D) xi(t)
 *                                                (Eq. 2; tilt: BASELINE.json)
 *     de/dt = q - c e - d e v^2                                        (Eq. 1)
 *     U(x)  = A1 sin(th) + A2 sin(2 th) + const,  th = 2 pi (x + phi) / L  (Eq. 3)
 * The paper's own potential of height h is L = 1, phi = 0.1903, A1 = -0.453 h, A2 = -0.11325 h.
 *
 * The loop each trajectory runs is the paper's pseudo kernel (Fig. 1): read the
 * parameters, for every step draw a uniform pair, Box-Muller it, compute the new velocity and
 * energy, and write the state back at the end so the next launch continues.  The generator is
 * counter-based Philox4x32-10 keyed by (seed, trajectory, step) instead of the paper's
 * xorshift (BASELINE.json north_star (b)); the exact stream is documented in
 * DESIGN.md ("Random stream") and is the same one the CPU oracle consumes.
 *
 * Conventions
 *   - All functions are extern "C", take plain pointers and sizes, and never throw.
 *   - Return value: ABM_OK (0) or a negative abm_status; *out arguments are untouched on error.
 *   - Pointers are HOST pointers unless the parameter is named dev_* (DEVICE pointer, valid on
 *     the device that was current at abm_create).
 *   - Trajectory index:  i = traj_base + set * traj_set_stride + r,   r < n_particles,
 *     set < n_param_sets; with the defaults (traj_base = 0, traj_set_stride = 0 meaning
 *     n_particles) this is i = set * n_particles + r.  The random stream, and therefore the
 *     whole trajectory, depends only on (seed, i, parameters): shards of one ensemble on
 *     several GPUs use traj_base / traj_set_stride to address disjoint index ranges.
 *   - In device buffers trajectories are stored in local order  k = set * n_particles + r.
 *   - The library owns the state and its scratch (device memory from a library-owned stream-ordered
 *     pool that keeps at most 1 GiB of freed memory cached; abm_trim releases it); `params` may be
 *     freed after abm_create; the snapshot buffer and all `out` arrays are caller-owned.
 *   - One context is not thread-safe; distinct contexts are independent.  All work of a context
 *     is enqueued on params[0].stream in call order; only abm_moments, abm_moment_sums,
 *     abm_time_averaged_velocity,
 *     abm_snapshot_host and abm_destroy wait for it.
 *   - A context belongs to the device that was current at abm_create.  Later calls may be made
 *     with any device current: the library switches to the context's device and restores the
 *     caller's before it returns.
 *   - Small fp32 ensembles (up to three 32-trajectory CTAs per SM: 14,208 trajectories on a B200) are
 *     integrated by a kernel that splits the work of a trajectory between warps (noise /
 *     integration) instead of one trajectory per thread; the
 *     results are bit-identical.  abm_params.step_kernel overrides the choice: a tuning and test knob,
 *     not part of the semantics.  The library reads no environment variable.
 *   - A handle is valid from a successful abm_create until abm_destroy.  Calls on a NULL, never
 *     created or already destroyed handle return ABM_ESTATE (handles are looked up in a table of live
 *     contexts before they are dereferenced; as with any address, a NEW context may later reuse it).
 *   - There is no CPU fallback: without a CUDA device abm_create returns ABM_ECUDA.
 */
#ifndef ABM_H
#define ABM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum abm_status {
  ABM_OK = 0,
  ABM_EINVAL = -1, /* null pointer, struct_size mismatch, zero counts, run-control fields that
                      differ between parameter sets, unsupported stride, misaligned pointer,
                      non-finite or non-positive dt / L / gamma0 (when init_v = 1)             */
  ABM_ENOMEM = -2, /* device or host allocation failed                                        */
  ABM_ECUDA = -3,  /* CUDA error (sticky: reported by this and every later call)              */
  ABM_ESTATE = -4, /* null or destroyed context                                               */
  ABM_ELIMIT = -5  /* the job needs more of the library's fixed, built-in scratch than exists
                      (abm_frame_moment_sums_static only; nothing was launched)                */
} abm_status;

enum { ABM_FP32 = 0, ABM_FP64 = 1 };               /* abm_params.precision  */
enum { ABM_EULER_MARUYAMA = 0, ABM_HEUN = 1 };     /* abm_params.integrator */
enum { ABM_INIT_V_CONST = 0, ABM_INIT_V_THERMAL = 1 }; /* abm_params.init_v */
/* abm_params.accuracy -- "precise vs fast intrinsics chosen against the stated tolerance"
 * (BASELINE.json north_star (b): fp32 state within 1e-5 of the fp64 oracle after 100 steps).
 *   FAST     angle 2 pi (x + phi) / L handed to MUFU.COS as is; x' = x + dt v in one FMA.
 *   PRECISE  the state carries the position as a 64-bit fixed-point number of periods (changed by
 *            exact integer additions only) plus a float offset that collects the increments of at
 *            most four steps, so nothing is rounded at the magnitude of the unwrapped position;
 *            the force takes its angle from the fraction word.  About +1.5 instructions per step
 *            over FAST, two more words of state per trajectory.  Frames, moments and the raster see
 *            the position rounded once to fp32.  The offset is folded with a 64-bit conversion, so
 *            any speed is legal (|x| < 2^31 L).
 *   AUTO     PRECISE if dt (2 pi / L)^2 (|A1| + 4 |A2|) > 0.15 for any set, else FAST
 *            (configs[0-2]: 0.079 -> FAST; config[3]: 0.39 -> PRECISE).
 * What the modes promise.  S = dt max|U''| <= dt (2 pi / L)^2 (|A1| + 4 |A2|) is the factor by which one
 * step turns a position error into a velocity error; the 100-step deviation from the fp64 oracle grows
 * in proportion to it.  FAST holds 1e-5 (scale-relative, reading G14) for S <= 0.15; forced on
 * a stiffer set it may miss it by about S / 0.15.  PRECISE holds 1e-5 for S <= 0.3 (config[3]: 0.39 is
 * measured at 4.4e-6, but random stiff potentials at 0.39 and 0.53 have missed it by factors up to 2.4:
 * a trajectory near a barrier top amplifies ANY fp32 rounding by exp(sqrt(max U'') t)).  Beyond that no
 * fp32 arithmetic meets 1e-5 after 100 steps: use ABM_FP64 or a smaller dt.  abm_get_accuracy reports
 * the mode in effect and whether the ensemble is beyond these limits.
 * Ignored in fp64.  Both modes consume the same random stream.
 * fp64 runs read two small Box-Muller tables that the library computes on the HOST in long double at first use: on
 * one host results are bit-identical from run to run; between hosts of different architecture or libm an entry may
 * differ in its last bit, so fp64 trajectories then agree to ~1e-16, not bit for bit. */
enum { ABM_ACCURACY_AUTO = 0, ABM_ACCURACY_FAST = 1, ABM_ACCURACY_PRECISE = 2 };
/* flag OR-ed into the value abm_get_accuracy returns: some set is stiffer than the mode in effect is
 * good for (FAST: S > 0.15, PRECISE: S > 0.3), so the fp32 state may deviate from an fp64 integration
 * by more than 1e-5 after 100 steps */
#define ABM_ACCURACY_BEYOND_TOLERANCE 0x100u

/* abm_params.rng -- where the uniform words come from.
 *   PHILOX        counter-based Philox4x32-10 keyed by (seed, trajectory, step): BASELINE.json
 *                 north_star (b); the stream of DESIGN.md "Random stream".  Default.
 *   XORSHIFT128   the paper's generator family ("Marsaglia xor-shift"; the variant is not
 *                 printed -- reading: xor128 of Marsaglia 2003): one state (x, y, z, w) per
 *                 trajectory, kept in device memory between launches, seeded from Philox block
 *                 2^64 - 2 of the trajectory; steps (2p, 2p + 1) use outputs 2p and 2p + 1.  For the
 *                 A/B of generator cost.  Everything else -- initial state,
 *                 uniform maps, Box-Muller, split-launch bit-identity -- is unchanged. */
enum { ABM_RNG_PHILOX = 0, ABM_RNG_XORSHIFT128 = 1 };

/* abm_params.step_kernel -- which kernel integrates (results are bit-identical whichever runs).
 *   AUTO         the library chooses by ensemble size.
 *   PER_THREAD   always one trajectory per thread (step_kernel).
 *   SPLIT_WARPS  the warp-specialised kernel (noise warps + integrating warps) wherever it applies
 *                (fp32, Philox, launches of whole Philox blocks, up to (2^31 - 1) * 32 trajectories: its grid). */
enum { ABM_STEP_KERNEL_AUTO = 0, ABM_STEP_KERNEL_PER_THREAD = 1, ABM_STEP_KERNEL_SPLIT_WARPS = 2 };

typedef struct abm_ctx abm_ctx; /* opaque, owned by the library */

/* One record per parameter set (the paper's per-work-item parameter record).
 * POD; copied at abm_create.  "Run-control" fields (marked RC) must be equal in all sets. */
typedef struct abm_params {
  uint32_t struct_size;    /* RC  = sizeof(abm_params); ABI guard                              */
  uint32_t precision;      /* RC  ABM_FP32 | ABM_FP64 (SP main path, DP optional)  */
  uint32_t integrator;     /* RC  ABM_EULER_MARUYAMA | ABM_HEUN                                */
  uint32_t init_v;         /* RC  v(0) = v0, or v(0) ~ N(0, D/gamma0) from the init block      */
  uint32_t snapshot_every; /* RC  K: abm_step rewrites the bound snapshot buffer after every
                                  global step count that is a multiple of K; 0 = never         */
  uint32_t accuracy;       /* RC  fp32 only: ABM_ACCURACY_AUTO | _FAST | _PRECISE (see above)      */
  uint32_t rng;            /* RC  ABM_RNG_PHILOX | ABM_RNG_XORSHIFT128                          */
  uint32_t step_kernel;    /* RC  ABM_STEP_KERNEL_AUTO | _PER_THREAD | _SPLIT_WARPS (tuning knob)  */
  double dt;               /* RC  time step                                                    */
  double gamma0, q, c, d, D; /*   Eqs. 1-2                                                     */
  double F0;               /*     constant load force, +F0 as printed in Eq. 2   */
  double A, omega;         /*     tilt A cos(omega n dt), n = global 0-based step index;
                                  omega is RC (one tilt table per launch), A is per set        */
  double L, A1, A2, phi;   /*     potential (see top of file)                                  */
  double v0, e0;           /*     constant initial values (x(0) ~ U[0, L) always)              */
  uint64_t traj_base;      /* RC  first global trajectory index of this context                */
  uint64_t traj_set_stride;/* RC  index distance between consecutive sets; 0 = n_particles     */
  void* stream;            /* RC  cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream);
                                  NULL = the legacy default stream                             */
} abm_params;

/* Ensemble moments of one parameter set over its n_particles realisations ("results are
 * averaged"), population normalisation 1/N, at global step `step`.
 * dx = x - x(0), with x(0) recomputed from the trajectory's init block. */
typedef struct abm_moment {
  uint64_t n, step;
  double mean_x, var_x, mean_v, var_v, mean_e, mean_dx, mean_dx2, mean_x2;
} abm_moment; /* 80 bytes */

/* Raw fp64 sums behind abm_moment, for combining shards (one record per set):
 * s = { N, sum x, sum x^2, sum v, sum v^2, sum e, sum dx, sum dx^2 }
 * -- plain sums (no shift of origin), accumulated in fp64 in a fixed order (run-to-run
 * reproducible). */
#define ABM_N_SUMS 8

/* Create a context for n_param_sets parameter sets x n_particles trajectories each and
 * initialise every trajectory from its Philox init block (S0): x(0) = L u, v(0), e(0) = e0.
 * Reads params[0 .. n_param_sets) (HOST).  Enqueues on params[0].stream; does not wait. */
int abm_create(const abm_params* params, uint64_t n_particles, uint32_t n_param_sets,
               uint64_t seed, abm_ctx** out);

/* Advance every trajectory by n_steps steps (S1-S5, S7; Fig. 1's loop), in one or a
 * few kernel launches with the state in registers in between.  Asynchronous.
 * abm_step(a); abm_step(b) is bit-identical to abm_step(a + b). n_steps = 0 is a no-op. */
int abm_step(abm_ctx* ctx, uint64_t n_steps);

/* Snapshot sink -- the headless replacement of the shared OpenGL vertex buffer.
 * dev_ptr != NULL: write the current state of all trajectories to dev_ptr now, and bind it as
 * the buffer that abm_step overwrites after every K-th step (K = snapshot_every; one frame,
 * overwritten).  dev_ptr == NULL: unbind.  stride_bytes = distance between trajectories:
 *   fp32:  8 -> float2 (x, v)        16 -> float4 (x, v, e, 1.0f)  (homogeneous vertex, :162)
 *   fp64: 16 -> double2 (x, v)       32 -> double4 (x, v, e, 1.0)
 * dev_ptr must be aligned to stride_bytes and hold n_particles * n_param_sets * stride_bytes. */
int abm_snapshot(abm_ctx* ctx, void* dev_ptr, size_t stride_bytes);

/* Same frame, copied to HOST memory (the paper's non-shared path); waits. */
int abm_snapshot_host(abm_ctx* ctx, void* host_ptr, size_t stride_bytes);

/* Ensemble moments of every set at the current step (S6): warp-shuffle + block + fixed-order
 * grid reduction in fp64 on the device, then a copy to out[0 .. n_param_sets) (HOST); waits. */
int abm_moments(abm_ctx* ctx, abm_moment* out);

/* The same reduction and copy, enqueued on the context's stream WITHOUT waiting: for moments every so
 * many steps (BASELINE.json configs[3]) the integration then never stalls on a host round trip.
 * out[0 .. n_param_sets) (HOST) must stay valid, and is defined, only after the stream has been
 * synchronised by the caller (or by a later waiting call of this context); page-locked memory makes
 * the copy a true asynchronous DMA, pageable memory is staged by the driver. */
int abm_moments_async(abm_ctx* ctx, abm_moment* out);

/* The raw sums (HOST, out[n_param_sets][ABM_N_SUMS]; waits) and the pure host-side finalisation used
 * after summing shards: out_moments[s] from sums[s]. */
int abm_moment_sums(abm_ctx* ctx, double* out);

/* The same raw sums written to a caller-owned DEVICE buffer dev_out[n_param_sets][ABM_N_SUMS] (8-byte
 * aligned; e.g. rows of a torch tensor that an NCCL all-reduce then sums across shards):
 * the reduction and a device-to-device copy are enqueued on the context's stream, nothing waits. */
int abm_moment_sums_dev(abm_ctx* ctx, double* dev_out);
int abm_moments_from_sums(const double* sums, uint32_t n_param_sets, uint64_t step,
                          abm_moment* out_moments);

/* The moment sums of a FRAME, for callers that must not allocate device memory.
 *
 * Who this is for.  Every other reduction above works on a context, and abm_create takes the context's
 * state and its reduction scratch from the CUDA allocator.  Some programs cannot do that at the point
 * where they want the moments: a host application that hands this library a fixed memory budget and owns
 * every device allocation itself (the frame then lives in ITS buffer, e.g. a tensor of its framework's
 * caching allocator, which cannot see memory a library takes behind its back); a service that has pinned
 * all of the GPU's memory up front; a latency-critical loop in which cudaMalloc / cudaFree -- which may
 * take driver locks and synchronise the whole device -- are forbidden after start-up.  Such a caller
 * passes the frame it already holds and a place for the result; this function calls no cudaMalloc,
 * cudaFree, pool or any other allocating routine, neither on the host nor on the device.
 *
 * What it computes.  The same eight sums per parameter set as abm_moment_sums_dev, in the same order of
 * additions (so the results are bit-identical to that call on the same state):
 *   dev_out[s][0..7] = { N, sum x, sum x^2, sum v, sum v^2, sum e, sum dx, sum dx^2 },  dx = x - x(0)
 * over the n_particles trajectories of set s, which occupy rows [s n_particles, (s + 1) n_particles).
 *   dev_frame   DEVICE, read only: a frame as abm_snapshot writes it -- fp32: stride 8 (x, v) or 16
 *               (x, v, e, 1); fp64: stride 16 or 32 -- aligned to stride_bytes.  With the short stride
 *               there is no e: sum e is 0.
 *   dev_frame0  DEVICE, read only, or NULL: a frame of the same layout taken at step 0; its x column is
 *               x(0).  NULL: sum dx = sum dx^2 = 0.
 *   dev_out     DEVICE, 8-byte aligned, [n_param_sets][ABM_N_SUMS] doubles, overwritten.  Feed a host copy
 *               to abm_moments_from_sums for means and variances.
 *   precision   ABM_FP32 | ABM_FP64 (the element type of the frames);  stream: cudaStream_t or NULL.
 * Asynchronous on `stream`; the caller keeps ownership of all three buffers.
 *
 * The scratch.  The per-CTA partial sums go into an array that is part of the library image itself (a
 * file-scope __device__ array, ABM_STATIC_SCRATCH_BYTES = 3.5 MiB).  Every GPU on which the library's code is
 * loaded holds that array from load until the process exits, whether or not this function is ever called.
 * It has room for ABM_STATIC_MAX_SLICES partial records; a set needs ceil(n_particles / 4096) of them (one
 * when n_particles <= 4096), so the limit is  n_param_sets * ceil(n_particles / 4096) <= 65,536  -- e.g. one
 * set of 268 million trajectories, or BASELINE.json's sweep of 65,536 sets x 64.  Beyond it the call
 * returns ABM_ELIMIT and launches nothing.
 *
 * Rules that follow from one shared array:
 *   - Calls whose kernels may run at the same time on one GPU (different streams, several host threads)
 *     write the same partial records and corrupt each other's sums.  Put them on one stream, or order
 *     them with events.  (Calls on different GPUs do not interfere: each GPU has its own copy.)
 *   - The array keeps what the previous call left in it.  Nothing here depends on that: every record a
 *     call reads back has been written by that same call first, so no clearing is needed or done.
 *   - The first call on each GPU looks up the array's device address (cudaGetSymbolAddress, with that GPU
 *     current; the result is cached per device).  Make that first call during start-up, outside any
 *     stream capture.
 * Errors: ABM_EINVAL (null / misaligned pointer, zero counts, bad stride or precision), ABM_ELIMIT,
 * ABM_ECUDA (no device, address lookup or launch failed). */
#define ABM_STATIC_MAX_SLICES 65536u
#define ABM_STATIC_SCRATCH_BYTES (ABM_STATIC_MAX_SLICES * 7u * 8u)
int abm_frame_moment_sums_static(const void* dev_frame, const void* dev_frame0, size_t stride_bytes,
                                 uint32_t precision, uint64_t n_particles, uint32_t n_param_sets,
                                 double* dev_out, void* stream);

/* The quantity the paper plots (Fig. 2: mean velocity against the load force, "over
 * time, results ... are averaged", :74): the velocity of each set averaged over its realisations AND
 * over the time since step 0 (hence over all launches so far),
 *     out[s] = < x(t) - x(0) >_s / (step * dt)
 * -- for Euler-Maruyama x(t) - x(0) = dt * (sum of v over the steps) exactly, for Heun it is the trapezoid
 * sum -- from the same device reduction as abm_moments.  out[0 .. n_param_sets) (HOST); waits.
 * ABM_EINVAL before the first step (no time has passed). */
int abm_time_averaged_velocity(abm_ctx* ctx, double* out);

/* Headless presentation of the current frame.  The paper draws every work
 * item as one vertex of the shared OpenGL buffer; here the same frame is
 * rasterised on the device: a 2-D histogram of the points (x mod L, v) -- a point splat with
 * additive blending -- and, optionally, an RGBA8 image of it.
 *   dev_counts  DEVICE uint32[height][width], row-major, 4-byte aligned; overwritten.  Column
 *               ix = position bin over [0, L), row iy = velocity bin over [v_min, v_max), row 0 at v_min.
 *   dev_rgba    DEVICE uint8[height][width][4] or NULL; grey ramp R = G = B =
 *               min(255, floor(255 * count / saturation)), A = 255; saturation >= 1.
 * Bin rule, in IEEE fp64 with every operation rounded on its own (no contraction), on the state
 * values converted exactly to double:
 *   xi = x / L;  f = xi - floor(xi);  ix = min(width - 1, floor(f * width))
 *   eta = (v - v_min) / (v_max - v_min);  the point is dropped unless 0 <= eta < 1;
 *   iy = min(height - 1, floor(eta * height)).
 * Non-finite states are dropped.  width * height <= 2^30.  Asynchronous on the context's stream. */
int abm_raster(abm_ctx* ctx, uint32_t* dev_counts, uint32_t width, uint32_t height, double v_min,
               double v_max, uint8_t* dev_rgba, uint32_t saturation);

/* Global step count reached so far. */
int abm_get_step(const abm_ctx* ctx, uint64_t* out_step);

/* The fp32 accuracy mode in effect (ABM_ACCURACY_FAST or _PRECISE; AUTO is resolved at create), OR-ed
 * with ABM_ACCURACY_BEYOND_TOLERANCE if some set is stiffer than that mode is good for (see above). */
int abm_get_accuracy(const abm_ctx* ctx, uint32_t* out_mode);

/* Wait for the context's stream and free everything the library owns.  ABM_ESTATE for a NULL, never
 * created or already destroyed handle (nothing is dereferenced). */
int abm_destroy(abm_ctx* ctx);

/* Give the freed device memory the library's pool of the CURRENT device still caches back to the driver
 * (waits for the device).  Live contexts keep theirs. */
int abm_trim(void);

/* Diagnostics of the random stream (tests: "bit-exact for the RNG integer stream", BASELINE.json).
 * dev_out[(k * n_blocks + j) * 4 + w] = word w of Philox block block_first + j of trajectory
 * traj_first + k.  stream: cudaStream_t or NULL.  Asynchronous.
 *
 * abm_philox_blocks computes every block with the plain ten-round function (philox_block), the code the
 * single-step path, the init / moment kernels and the small-ensemble kernel's noise warps call.
 *
 * abm_philox_blocks_loop produces the same words THE WAY THE BLOCK LOOP OF THE STEP KERNELS DOES: it
 * launches, with abm_step's launch geometry (128 threads, one trajectory per thread), a kernel that
 * instantiates the very loop function the step kernels run (run_steps) with a body that stores each
 * block's words instead of integrating with them -- the per-trajectory half of rounds 0-1 done once,
 * the per-block half fetched from the double-buffered shared-memory table that is refilled every 128
 * blocks, rounds 2-9 with the round keys the host computes, the look-ahead pipeline, and
 *   loop_shape 0: the loop as the fp32 kernels instantiate it, 1: as the fp64 kernels do (both run two blocks per
 *   loop trip since round 2; the value only selects the instantiation);
 *   frame_every_blocks != 0: the loop is cut into segments of that many blocks as by a frame period of
 *   4 * frame_every_blocks steps (odd segments exercise the loop's one-block prologue).
 * A trajectory range that straddles a multiple of 2^32 runs the loop's table-free branch, as in abm_step.
 * n_blocks <= 2^28; block_first + n_blocks <= 2^62. */
int abm_philox_blocks(uint64_t seed, uint64_t traj_first, uint64_t n_traj, uint64_t block_first,
                      uint64_t n_blocks, uint32_t* dev_out, void* stream);
int abm_philox_blocks_loop(uint64_t seed, uint64_t traj_first, uint64_t n_traj, uint64_t block_first,
                           uint64_t n_blocks, uint32_t loop_shape, uint32_t frame_every_blocks,
                           uint32_t* dev_out, void* stream);

/* Static, non-owning description of a status code. */
const char* abm_strerror(int status);

/* Version of this ABI (bumped when abm_params or a signature changes). */
uint32_t abm_abi_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ABM_H */
