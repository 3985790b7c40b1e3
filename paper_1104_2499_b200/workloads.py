"""Seeded synthetic workloads: the five BASELINE.json configs as plain parameter records.

This module serves BOTH the CUDA path (tests, bench.py) and the CPU oracle's tests.  It holds
none of the method's arithmetic: only parameter values, sizes, seeds and the sweep grid of
config[2].  The paper uses no dataset; its workload is a set of
independent work items that differ in one parameter run for 10^3..10^4 iterations
per launch, which configs [1] and [2] scale up.
"""
from dataclasses import dataclass, field
import math

import numpy as np

# Parameters shared by every config unless overridden (BASELINE.json configs[0]).
DEFAULTS = dict(
    precision=0, integrator=0, init_v=0,
    dt=1e-3, gamma0=1.0, q=1.0, c=0.1, d=1.0, D=0.1, F0=0.0, A=0.0, omega=0.0,
    L=1.0, A1=1.0, A2=0.25, phi=0.0, v0=0.0, e0=0.0,
)

# The paper's own Eq. 3 potential (reading G2): U = h[0.499 - 0.453(sin th + 1/4 sin 2th)],
# th = 2 pi (x + 0.1903).  In the (A1, A2, phi) parametrisation, for height h:
def paper_potential(h: float = 1.0) -> dict:
    return dict(L=1.0, phi=0.1903, A1=-0.453 * h, A2=-0.453 * 0.25 * h)


@dataclass
class Workload:
    name: str
    n_particles: int            # per parameter set
    n_param_sets: int
    seed: int
    n_steps: int
    snapshot_every: int = 0     # K: float2 frame every K steps (0 = none)
    moments_every: int = 0      # moments every M steps (0 = only at the end)
    base: dict = field(default_factory=dict)
    sweep: dict = field(default_factory=dict)   # name -> float64 array [n_param_sets]

    @property
    def n_trajectories(self) -> int:
        return self.n_particles * self.n_param_sets

    @property
    def particle_steps(self) -> int:
        return self.n_trajectories * self.n_steps

    def set_params(self, s: int) -> dict:
        """Parameter record of set s (scalars only)."""
        p = dict(self.base)
        for k, arr in self.sweep.items():
            p[k] = float(arr[s])
        return p


def _base(**over) -> dict:
    p = dict(DEFAULTS)
    p.update(over)
    return p


def config0() -> Workload:
    return Workload("cfg0_ref_4096x1e4_em_f32", 4096, 1, 42, 10_000, base=_base())


def config1(n_particles: int = 1_048_576, n_steps: int = 100_000) -> Workload:
    return Workload("cfg1_1Mx1e5_em_f32_snap100", n_particles, 1, 7, n_steps,
                    snapshot_every=100, base=_base())


def config2(n_D: int = 256, n_q: int = 256, realisations: int = 64, n_steps: int = 10_000) -> Workload:
    """Sweep: D_i = 10^(-3 + 3 i/(n_D-1)), q_j = 2 j/(n_q-1); set index s = n_q * i + j (reading G18)."""
    i = np.arange(n_D, dtype=np.float64)
    j = np.arange(n_q, dtype=np.float64)
    Dv = 10.0 ** (-3.0 + 3.0 * i / max(n_D - 1, 1))
    qv = 2.0 * j / max(n_q - 1, 1)
    D = np.repeat(Dv, n_q)
    q = np.tile(qv, n_D)
    return Workload("cfg2_sweep_256Dx256qx64_em_f32", realisations, n_D * n_q, 1234, n_steps,
                    base=_base(), sweep=dict(D=D, q=q))


def config3(n_particles: int = 1_048_576, n_steps: int = 20_000) -> Workload:
    return Workload("cfg3_1Mx2e4_heun_tilt_f32", n_particles, 1, 99, n_steps, moments_every=1000,
                    base=_base(integrator=1, dt=5e-3, A=0.5, omega=2.0 * math.pi * 0.1, D=0.05))


def config4(n_particles: int = 4_194_304, n_steps: int = 50_000) -> Workload:
    return Workload("cfg4_4Mx5e4_em_f64", n_particles, 1, 2024, n_steps,
                    base=_base(precision=1, dt=1e-4, A1=2.0, A2=0.5, D=0.2, q=1.5, init_v=1))


def paper_f0_sweep(n_F0: int = 65_536, F0_min: float = -1.0, F0_max: float = 0.0, realisations: int = 1,
                   n_steps: int = 10_000, h: float = 1.0, seed: int = 1104) -> Workload:
    """The paper's own workload: work items that
    differ only in the load force F0 ("opposing" = negative, reading G13), 2^0 .. 2^16 of them, on the Eq. 3
    potential of height h (reading G2), run for 10^3..10^4 iterations per launch; the plotted quantity is the
    mean velocity averaged over time and launches, i.e. <x(t) - x(0)> / t (abm_time_averaged_velocity).
    The paper prints no parameter values: the depot parameters are those of BASELINE.json configs[0].
    F0_k = F0_min + (F0_max - F0_min) k / (n_F0 - 1)."""
    k = np.arange(n_F0, dtype=np.float64)
    F0 = F0_min + (F0_max - F0_min) * k / max(n_F0 - 1, 1)
    return Workload(f"paper_f0_sweep_{n_F0}x{realisations}", realisations, n_F0, seed, n_steps,
                    base=_base(**paper_potential(h)), sweep=dict(F0=F0))


CONFIGS = [config0, config1, config2, config3, config4]
