/* abm_demo.c -- the C ABI of include/abm.h called from plain C99 (no CUDA headers, no Python):
 * BASELINE.json configs[0] with fewer trajectories -- create, step, read the frame back to the
 * host (the paper's non-shared path), ensemble moments, destroy.
 *
 *   gcc -std=c99 -I include -o abm_demo paper_1104_2499_b200/examples/abm_demo.c \
 *       -L paper_1104_2499_b200 -labm_b200 -Wl,-rpath,$PWD/paper_1104_2499_b200
 *   ./abm_demo [n_particles] [n_steps]      prints "moment ..." and one "traj i x v e" line per trajectory
 *
 * Exit code 0 on success, 3 when there is no CUDA device (abm_create returns ABM_ECUDA: no fallback). */
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "abm.h"

int main(int argc, char** argv) {
  const uint64_t n_particles = argc > 1 ? strtoull(argv[1], NULL, 10) : 256;
  const uint64_t n_steps = argc > 2 ? strtoull(argv[2], NULL, 10) : 100;
  abm_params p;
  memset(&p, 0, sizeof(p));
  p.struct_size = (uint32_t)sizeof(p);
  p.precision = ABM_FP32;
  p.integrator = ABM_EULER_MARUYAMA;
  p.init_v = ABM_INIT_V_CONST;
  p.dt = 1e-3;
  p.gamma0 = 1.0; p.q = 1.0; p.c = 0.1; p.d = 1.0; p.D = 0.1;   /* Eqs. 1-2, BASELINE.json configs[0] */
  p.L = 1.0; p.A1 = 1.0; p.A2 = 0.25; p.phi = 0.0;              /* U = sin(2 pi x) + sin(4 pi x) / 4     */
  abm_ctx* ctx = NULL;
  int rc = abm_create(&p, n_particles, 1, 42, &ctx);
  if (rc != ABM_OK) {
    fprintf(stderr, "abm_create: %d (%s)\n", rc, abm_strerror(rc));
    return rc == ABM_ECUDA ? 3 : 1;
  }
  float* frame = (float*)malloc(sizeof(float) * 4 * n_particles);   /* (x, v, e, 1) per trajectory */
  abm_moment m;
  if (!frame) return 1;
  if ((rc = abm_step(ctx, n_steps)) != ABM_OK || (rc = abm_snapshot_host(ctx, frame, 16)) != ABM_OK ||
      (rc = abm_moments(ctx, &m)) != ABM_OK) {
    fprintf(stderr, "abm: %d (%s)\n", rc, abm_strerror(rc));
    return 1;
  }
  printf("moment n %llu step %llu mean_v %.17g var_v %.17g mean_x %.17g var_x %.17g mean_e %.17g\n",
         (unsigned long long)m.n, (unsigned long long)m.step, m.mean_v, m.var_v, m.mean_x, m.var_x, m.mean_e);
  for (uint64_t i = 0; i < n_particles; ++i)
    printf("traj %llu %.9g %.9g %.9g\n", (unsigned long long)i, frame[4 * i], frame[4 * i + 1], frame[4 * i + 2]);
  free(frame);
  return abm_destroy(ctx) == ABM_OK ? 0 : 1;
}
