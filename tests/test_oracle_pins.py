"""Pins of the CPU oracle against what the paper and the mathematics fix.

Every test here compares the oracle with something other than itself: published known answers,
closed forms, exact discrete recursions, physical limits, quadrature, or an independent
brute-force restatement in numpy/Python integers.  No GPU needed.
"""
import math
import os

import numpy as np
import pytest

from paper_1104_2499_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
Z = 3.5  # statistical tests accept |deviation| <= Z standard errors (seeded, so deterministic)


def cfg(**over):
    p = dict(W.DEFAULTS)
    p.update(over)
    return p


def free(**over):
    """No potential, no depot coupling, no forces: the pieces are switched on by the caller."""
    p = cfg(A1=0.0, A2=0.0, d=0.0, q=0.0, c=0.0, F0=0.0, A=0.0)
    p.update(over)
    return p


# ---------------------------------------------------------------------------------------------
# P1  Philox4x32-10 known answers (Salmon et al., SC'11; Random123 kat_vectors)
# ---------------------------------------------------------------------------------------------

def test_p1_philox_known_answers(oracle):
    rows = [l.split() for l in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        h = [int(t, 16) for t in r]
        assert oracle.philox4x32_10(h[0:4], h[4:6]) == h[6:10]


def _philox_py(ctr, key):
    """Independent restatement in Python integers (round function as published)."""
    c, k = list(ctr), list(key)
    for _ in range(10):
        p0 = 0xD2511F53 * c[0]
        p1 = 0xCD9E8D57 * c[2]
        c = [((p1 >> 32) ^ c[1] ^ k[0]) & 0xffffffff, p1 & 0xffffffff,
             ((p0 >> 32) ^ c[3] ^ k[1]) & 0xffffffff, p0 & 0xffffffff]
        k = [(k[0] + 0x9E3779B9) & 0xffffffff, (k[1] + 0xBB67AE85) & 0xffffffff]
    return c


def test_p1b_philox_python_restatement_and_layout(oracle):
    # the restatement itself reproduces the published vectors ...
    assert _philox_py([0, 0, 0, 0], [0, 0]) == [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]
    rng = np.random.default_rng(5)
    for _ in range(200):
        ctr = [int(v) for v in rng.integers(0, 2**32, 4)]
        key = [int(v) for v in rng.integers(0, 2**32, 2)]
        assert oracle.philox4x32_10(ctr, key) == _philox_py(ctr, key)
    # ... and the stream layout: key = (seed lo, hi), ctr = (b lo, b hi, traj lo, traj hi)
    for seed, traj, b in [(42, 0, 0), (7, 1_048_575, 24_999), (2**63 + 12345, 2**40 + 3, 2**35 + 1),
                          (1234, 5, 2**64 - 1)]:
        want = _philox_py([b & 0xffffffff, b >> 32, traj & 0xffffffff, traj >> 32],
                          [seed & 0xffffffff, seed >> 32])
        assert oracle.block(seed, traj, b) == want


# ---------------------------------------------------------------------------------------------
# P3  uniform and normal maps
# ---------------------------------------------------------------------------------------------

def test_p3_uniform_map_range_and_exactness(oracle):
    assert oracle.uniform(0, 0) == 2.0**-24
    assert oracle.uniform(0xffffffff, 0) == 1.0 - 2.0**-24
    assert oracle.uniform(0x1ff, 0) == 2.0**-24            # low 9 bits unused
    assert oracle.uniform(0x200, 0) == 1.5 * 2.0**-23
    assert oracle.uniform(0, 1) == 2.0**-33
    assert oracle.uniform(0xffffffff, 1) == 1.0 - 2.0**-33
    rng = np.random.default_rng(1)
    for w in rng.integers(0, 2**32, 2000):
        u = oracle.uniform(int(w), 0)
        assert 0.0 < u < 1.0 and float(np.float32(u)) == u   # exact in fp32
        assert oracle.uniform(int(w), 1) == (int(w) + 0.5) / 2**32


@pytest.mark.parametrize("precision,zmax", [(0, math.sqrt(48 * math.log(2))),
                                            (1, math.sqrt(66 * math.log(2)))])
def test_p3_normal_moments(oracle, precision, zmax):
    n_traj, n_steps = 2500, 4000                       # 10^7 draws
    z = oracle.normals(2718, 10, n_traj, 0, n_steps, precision)
    N = z.size
    assert np.abs(z).max() <= zmax + 1e-12             # bound implied by u1 >= 2^-24 (2^-33)
    assert abs(z.mean()) < Z / math.sqrt(N)
    assert abs(z.var() - 1.0) < Z * math.sqrt(2.0 / N)
    kurt = np.mean(z**4) / z.var()**2
    assert abs(kurt - 3.0) < Z * math.sqrt(96.0 / N)
    assert abs(np.mean(np.abs(z) < 1.0) - math.erf(1 / math.sqrt(2))) < Z * 0.47 / math.sqrt(N)
    # even/odd steps of a pair share r and use cos/sin of the same angle
    ze, zo = z[:, 0::2], z[:, 1::2]
    assert abs(np.mean(ze * zo)) < Z / math.sqrt(ze.size)
    r2 = ze**2 + zo**2                                  # = -2 ln u1 ~ chi^2 with 2 dof
    assert abs(r2.mean() - 2.0) < Z * 2.0 / math.sqrt(r2.size)
    # consecutive steps, consecutive trajectories: uncorrelated
    assert abs(np.mean(z[:, 1:-1:2] * z[:, 2::2])) < Z / math.sqrt(z[:, 2::2].size)
    assert abs(np.mean(z[:-1] * z[1:])) < Z / math.sqrt(z[1:].size)


def test_p3_normal_definition_single_values(oracle):
    """z_n from words by the textbook Box-Muller formula, written with numpy's own functions."""
    seed, traj = 99, 17
    for n in range(8):
        w = oracle.block(seed, traj, n >> 2)
        p = (n >> 1) & 1
        for prec, u in [(0, lambda t: ((t >> 9) + 0.5) / 2**23), (1, lambda t: (t + 0.5) / 2**32)]:
            u1, u2 = u(w[2 * p]), u(w[2 * p + 1])
            r = np.sqrt(-2.0 * np.log(u1))
            want = r * (np.cos(2 * np.pi * u2) if n % 2 == 0 else np.sin(2 * np.pi * u2))
            assert oracle.normal(seed, traj, n, prec) == pytest.approx(want, rel=1e-14, abs=1e-15)


# ---------------------------------------------------------------------------------------------
# Eq. 3 and the force
# ---------------------------------------------------------------------------------------------

def test_eq3_normalisation_height_h(oracle):
    """'ratchet potential of the height h' with printed constants 0.499, 0.453,
    0.1903 -- under reading G2 U + 0.499 h spans [0, h] with its minimum at x = 0."""
    p = cfg(**W.paper_potential(1.0))
    xs = np.linspace(0.0, 1.0, 20001)
    U = np.array([oracle.potential(p, x) for x in xs]) + 0.499
    assert abs(U.min()) < 2e-3 and abs(U.max() - 1.0) < 3e-3
    xmin = xs[U.argmin()]
    assert min(xmin, 1 - xmin) < 2e-3                  # minimum at x = 0 (mod 1)
    assert abs(xs[U.argmax()] - 0.6193) < 2e-3         # asymmetric: a ratchet
    assert oracle.potential(p, 0.3) == pytest.approx(oracle.potential(p, 1.3), abs=1e-12)


@pytest.mark.parametrize("pot", [dict(A1=1.0, A2=0.25, L=1.0, phi=0.0),
                                 dict(A1=-0.453, A2=-0.11325, L=1.0, phi=0.1903),
                                 dict(A1=0.7, A2=-0.3, L=2.5, phi=0.4)])
def test_force_is_minus_gradient(oracle, pot):
    p = free(**pot)
    p["gamma0"] = 0.0
    h = 1e-6
    for x in np.linspace(-1.3, 2.9, 37):
        ax, av, ae = oracle.rhs(p, x, 0.0, 0.0, 0.0)
        fd = -(oracle.potential(p, x + h) - oracle.potential(p, x - h)) / (2 * h)
        assert av == pytest.approx(fd, abs=2e-8)
        assert ax == 0.0 and ae == 0.0


def test_rhs_terms_signs(oracle):
    """Each term of Eqs. 1-2 in isolation."""
    p = free(gamma0=0.0)
    assert oracle.rhs(dict(p, gamma0=2.0), 0, 3.0, 0, 0)[1] == -6.0            # -gamma v
    assert oracle.rhs(dict(p, d=0.5), 0, 3.0, 4.0, 0)[1] == 6.0                # +d e v
    assert oracle.rhs(dict(p, F0=-0.25), 0, 0, 0, 0)[1] == -0.25               # +F0
    assert oracle.rhs(dict(p, A=2.0, omega=math.pi), 0, 0, 0, 1.0)[1] == pytest.approx(-2.0)
    assert oracle.rhs(dict(p, q=1.5), 0, 0, 0, 0)[2] == 1.5                    # +q
    assert oracle.rhs(dict(p, c=0.1), 0, 0, 2.0, 0)[2] == pytest.approx(-0.2)  # -c e
    assert oracle.rhs(dict(p, d=0.5), 0, 3.0, 2.0, 0)[2] == -9.0               # -d e v^2
    assert oracle.rhs(p, 0, 1.25, 0, 0)[0] == 1.25                             # dx/dt = v


def test_energy_conservation_heun(oracle):
    """gamma0 = d = D = 0: v^2/2 + U(x) is conserved; Heun's drift is O(dt^2)."""
    p = free(gamma0=0.0, D=0.0, A1=1.0, A2=0.25, integrator=1, dt=1e-3, v0=2.5)
    x, v, e = oracle.init_many(p, 3, 4)
    E0 = 0.5 * v**2 + np.array([oracle.potential(p, t) for t in x])
    oracle.run(p, 3, x, v, e, 0, 5000)
    E1 = 0.5 * v**2 + np.array([oracle.potential(p, t) for t in x])
    assert np.abs(E1 - E0).max() < 5e-5


# ---------------------------------------------------------------------------------------------
# P4  Ornstein-Uhlenbeck limit
# ---------------------------------------------------------------------------------------------

def test_p4_ou_velocity_variance_exact_recursion(oracle):
    """EM on dv = -gamma v dt + sqrt(2D) dW is v' = a v + sigma z: var v_n is exact."""
    D, g, dt, n, N = 0.5, 1.0, 1e-3, 3000, 16384
    p = free(D=D, gamma0=g, dt=dt)
    x, v, e = oracle.init_many(p, 11, N)
    x0 = x.copy()
    oracle.run(p, 11, x, v, e, 0, n)
    a = 1.0 - g * dt
    var_exact = 2 * D * dt * (1 - a**(2 * n)) / (1 - a * a)
    assert abs(v.mean()) < Z * math.sqrt(var_exact / N)
    assert abs(v.var() - var_exact) < Z * var_exact * math.sqrt(2.0 / N)
    # continuous MSD from v0 = 0 (Ornstein-Furth); EM bias is O(dt) = 0.1 %
    t = n * dt
    msd = (D / g**3) * (2 * g * t - 3 + 4 * math.exp(-g * t) - math.exp(-2 * g * t))
    dx = x - x0
    assert abs(np.mean(dx**2) - msd) < Z * msd * math.sqrt(2.0 / N) + 5e-3 * msd
    assert abs(dx.mean()) < Z * math.sqrt(msd / N)


def test_p4_ou_stationary_variance_and_thermal_start(oracle):
    """Stationary EM variance D / (gamma (1 - gamma dt / 2)); thermal v0 ~ N(0, D/gamma) and its
    MSD (2D/gamma^3)(gamma t - 1 + exp(-gamma t))."""
    D, g, dt, N = 0.2, 2.0, 2e-3, 16384
    p = free(D=D, gamma0=g, dt=dt, init_v=1, precision=1)
    x, v, e = oracle.init_many(p, 5, N)
    assert abs(v.var() - D / g) < Z * (D / g) * math.sqrt(2.0 / N)      # init block normal
    assert abs(v.mean()) < Z * math.sqrt(D / g / N)
    assert np.all((x >= 0) & (x < 1.0)) and abs(x.mean() - 0.5) < Z / math.sqrt(12 * N)
    x0 = x.copy()
    n = 2500
    oracle.run(p, 5, x, v, e, 0, n)
    var_st = D / (g * (1 - g * dt / 2))
    assert abs(v.var() - var_st) < Z * var_st * math.sqrt(2.0 / N)
    t = n * dt
    msd = (2 * D / g**3) * (g * t - 1 + math.exp(-g * t))
    assert abs(np.mean((x - x0)**2) - msd) < Z * msd * math.sqrt(2.0 / N) + 1e-2 * msd


def test_p4_heun_ou_variance_exact_recursion(oracle):
    """Heun on the linear SDE: v' = (1 - g dt + (g dt)^2/2) v + sigma (1 - g dt/2) z exactly --
    pins that the SAME noise increment enters predictor and corrector (reading G16)."""
    D, g, dt, n, N = 0.5, 1.0, 0.2, 100, 16384
    p = free(D=D, gamma0=g, dt=dt, integrator=1)
    x, v, e = oracle.init_many(p, 21, N)
    oracle.run(p, 21, x, v, e, 0, n)
    a = 1 - g * dt + (g * dt)**2 / 2
    b2 = 2 * D * dt * (1 - g * dt / 2)**2
    var_exact = b2 * (1 - a**(2 * n)) / (1 - a * a)
    assert abs(v.var() - var_exact) < Z * var_exact * math.sqrt(2.0 / N)
    # and it differs measurably from what EM would give, so the test can tell them apart
    a_em = 1 - g * dt
    var_em = 2 * D * dt * (1 - a_em**(2 * n)) / (1 - a_em**2)
    assert abs(var_em - var_exact) > Z * var_exact * math.sqrt(2.0 / N)


# ---------------------------------------------------------------------------------------------
# P5, P6  energy depot
# ---------------------------------------------------------------------------------------------

def test_p5_depot_stationary_speed(oracle):
    """D = 0, no potential: v^2 -> q/gamma0 - c/d, e -> gamma0/d (fixed point of Eqs. 1-2;
    v = 0 is unstable so v(0) != 0)."""
    for q, g, c, d in [(1.0, 1.0, 0.1, 1.0), (1.5, 0.5, 0.2, 2.0)]:
        p = cfg(A1=0.0, A2=0.0, D=0.0, q=q, gamma0=g, c=c, d=d, v0=0.05, dt=1e-3)
        x, v, e = oracle.init_many(p, 1, 2)
        oracle.run(p, 1, x, v, e, 0, 200_000)
        assert v[0]**2 == pytest.approx(q / g - c / d, rel=1e-10)
        assert e[0] == pytest.approx(g / d, rel=1e-10)
    # below threshold q d < c gamma0 the particle comes to rest
    p = cfg(A1=0.0, A2=0.0, D=0.0, q=0.05, v0=0.5)
    x, v, e = oracle.init_many(p, 1, 1)
    oracle.run(p, 1, x, v, e, 0, 200_000)
    assert abs(v[0]) < 1e-6 and e[0] == pytest.approx(0.05 / 0.1, rel=1e-6)


def test_p6_depot_filling_closed_form(oracle):
    """d = 0: EM gives e_n = (q/c)(1 - (1 - c dt)^n) exactly."""
    q, c, dt, n = 1.3, 0.25, 1e-3, 12_345
    p = cfg(d=0.0, q=q, c=c, dt=dt)
    x, v, e = oracle.init_many(p, 8, 3)
    oracle.run(p, 8, x, v, e, 0, n)
    assert e == pytest.approx((q / c) * (1 - (1 - c * dt)**n), rel=1e-12)


# ---------------------------------------------------------------------------------------------
# P7, P8  zero-current limits;  Boltzmann average
# ---------------------------------------------------------------------------------------------

def _se_mean(a):
    return a.std() / math.sqrt(a.size)


def _late_displacement(oracle, p, seed, N, n_relax, n_meas):
    """Displacement over [n_relax, n_relax + n_meas): the relaxation of the uniform initial
    positions into the wells (a transient shift of the mean, not a current) is excluded."""
    thr = oracle.host_threads()
    x, v, e = oracle.init_many(p, seed, N)
    oracle.run(p, seed, x, v, e, 0, n_relax, threads=thr)
    x1 = x.copy()
    oracle.run(p, seed, x, v, e, n_relax, n_meas, threads=thr)
    return x - x1, v


def test_p7_symmetric_potential_no_current(oracle):
    p = cfg(A2=0.0)                                   # single harmonic: no ratchet effect
    dx, v = _late_displacement(oracle, p, 77, 8192, 2000, 5000)
    assert abs(v.mean()) < Z * _se_mean(v)
    assert abs(dx.mean()) < Z * _se_mean(dx)


def test_p8_passive_particle_on_ratchet_no_current(oracle):
    p = cfg(d=0.0, D=0.5)                             # equilibrium: no current for any A2
    dx, v = _late_displacement(oracle, p, 78, 8192, 3000, 5000)
    assert abs(v.mean()) < Z * _se_mean(v)
    assert abs(dx.mean()) < Z * _se_mean(dx)


@pytest.mark.parametrize("integrator,dt,bias", [(1, 2e-3, 2e-3), (0, 2e-4, 5e-3)])
def test_boltzmann_position_average(oracle, integrator, dt, bias):
    """Passive particle (d = 0): stationary density is exp(-U/T)/Z with T = D/gamma0
    (fluctuation-dissipation).  Pins noise amplitude vs force vs friction, and the force sign.
    EM heats the particle by O(U'' dt / gamma0) (about 4 % at dt = 1e-3 here), so it
    is pinned at a smaller dt than Heun, whose bias is O(dt^2)."""
    D, g = 0.5, 1.0
    p = cfg(d=0.0, D=D, gamma0=g, dt=dt, integrator=integrator)
    T = D / g
    xs = (np.arange(20000) + 0.5) / 20000
    w = np.exp(-np.array([oracle.potential(p, t) for t in xs]) / T)
    sin_b = float((np.sin(2 * np.pi * xs) * w).sum() / w.sum())
    cos2_b = float((np.cos(4 * np.pi * xs) * w).sum() / w.sum())
    assert sin_b < -0.5                               # strongly non-trivial value
    N = 4096
    x, v, e = oracle.init_many(p, 31, N)
    thr = oracle.host_threads()
    n = int(round(6.0 / dt))
    oracle.run(p, 31, x, v, e, 0, n, threads=thr)
    s, c2, v2 = [], [], []
    gap = int(round(1.5 / dt))                        # snapshots 1.5 relaxation times apart
    for _ in range(8):
        oracle.run(p, 31, x, v, e, n, gap, threads=thr)
        n += gap
        s.append(np.sin(2 * np.pi * x)); c2.append(np.cos(4 * np.pi * x)); v2.append(v * v)
    s, c2, v2 = np.concatenate(s), np.concatenate(c2), np.concatenate(v2)
    # snapshots are positively correlated: count them as 2 independent ones (conservative)
    n_eff = 2 * N
    assert abs(s.mean() - sin_b) < Z * s.std() / math.sqrt(n_eff) + bias
    assert abs(c2.mean() - cos2_b) < Z * c2.std() / math.sqrt(n_eff) + bias
    assert abs(v2.mean() - T) < Z * T * math.sqrt(2.0 / n_eff) + 4 * bias


# ---------------------------------------------------------------------------------------------
# P9, P10, P11  integrators
# ---------------------------------------------------------------------------------------------

def test_p9_update_order_closed_forms(oracle):
    """gamma0 = d = D = 0, no potential, constant F0, v0 = 0.
    EM (simultaneous update from the old state, reading G4): x_n = x0 + F0 dt^2 n(n-1)/2.
    Heun: x_n = x0 + F0 (n dt)^2 / 2."""
    F0, dt, n = 0.7, 1e-3, 1000
    for integ, want in [(0, F0 * dt * dt * n * (n - 1) / 2), (1, F0 * (n * dt)**2 / 2)]:
        p = free(gamma0=0.0, D=0.0, F0=F0, dt=dt, integrator=integ)
        x, v, e = oracle.init_many(p, 4, 5)
        x0 = x.copy()
        oracle.run(p, 4, x, v, e, 0, n)
        assert (x - x0) == pytest.approx(want, rel=1e-11)
        assert v == pytest.approx(F0 * n * dt, rel=1e-12)


def _final_state(oracle, p, n):
    x, v, e = oracle.init_many(p, 9, 1)
    oracle.run(p, 9, x, v, e, 0, n)
    return np.array([x[0], v[0], e[0]])


def test_p10_convergence_order(oracle):
    """D = 0, full model: halving dt cuts the error x2 (EM) and x4 (Heun)."""
    base = cfg(D=0.0, v0=0.8, e0=0.3, A=0.5, omega=2 * math.pi * 0.1)
    Tend = 2.0
    ref = _final_state(oracle, dict(base, integrator=1, dt=Tend / 256000), 256000)
    for integ, order in [(0, 1), (1, 2)]:
        errs = []
        for n in ((4000, 8000, 16000) if integ == 0 else (500, 1000, 2000)):
            s = _final_state(oracle, dict(base, integrator=integ, dt=Tend / n), n)
            errs.append(np.abs(s - ref).max())
        for a, b in zip(errs[:-1], errs[1:]):
            assert a / b == pytest.approx(2.0**order, rel=0.12)


def test_p11_tilt_analytic_solution(oracle):
    """No potential, d = D = 0: dv/dt = -g v + A cos(w t), v(0) = 0 ->
    v = A (g cos wt + w sin wt - g exp(-g t)) / (g^2 + w^2).  Pins phase and time origin of the
    tilt (reading G15) and Heun's use of t_{n+1} in the corrector."""
    A, w, g, dt, n = 0.5, 2 * math.pi * 0.1, 1.0, 1e-3, 10_000
    p = free(gamma0=g, D=0.0, A=A, omega=w, dt=dt, integrator=1)
    x, v, e = oracle.init_many(p, 2, 1)
    for k in range(1, 5):
        oracle.run(p, 2, x, v, e, (k - 1) * n // 4, n // 4)
        t = k * (n // 4) * dt
        want = A * (g * math.cos(w * t) + w * math.sin(w * t) - g * math.exp(-g * t)) / (g * g + w * w)
        assert v[0] == pytest.approx(want, abs=2e-7)
    # EM sees the same tilt, to first order
    p = free(gamma0=g, D=0.0, A=A, omega=w, dt=dt, integrator=0)
    x, v, e = oracle.init_many(p, 2, 1)
    oracle.run(p, 2, x, v, e, 0, n)
    assert v[0] == pytest.approx(want, abs=1e-3)


# ---------------------------------------------------------------------------------------------
# P12  brute force: independent restatement (Python-integer Philox + numpy fp64)
# ---------------------------------------------------------------------------------------------

def _brute(p, seed, trajs, n0, n1, state=None):
    two_pi = 2 * np.pi

    def u(w):
        return ((w >> 9) + 0.5) / 2**23 if p["precision"] == 0 else (w + 0.5) / 2**32

    def blk(i, b):
        return _philox_py([b & 0xffffffff, b >> 32, i & 0xffffffff, i >> 32],
                          [seed & 0xffffffff, seed >> 32])

    def drift(x, v, e, t):
        th = two_pi * (x + p["phi"]) / p["L"]
        dU = two_pi / p["L"] * (p["A1"] * np.cos(th) + 2 * p["A2"] * np.cos(2 * th))
        return (v, -p["gamma0"] * v + p["d"] * e * v - dU + p["F0"] + p["A"] * np.cos(p["omega"] * t),
                p["q"] - p["c"] * e - p["d"] * e * v * v)

    out = []
    for k, i in enumerate(trajs):
        if state is None:
            w = blk(i, 2**64 - 1)
            x = p["L"] * ((w[0] >> 8) / 2**24 if p["precision"] == 0 else w[0] / 2**32)
            v = p["v0"] if p["init_v"] == 0 else (np.sqrt(p["D"] / p["gamma0"])
                                                  * np.sqrt(-2 * np.log(u(w[2]))) * np.cos(two_pi * u(w[3])))
            e = p["e0"]
        else:
            x, v, e = state[k]
        sig = np.sqrt(2 * p["D"] * p["dt"])
        for n in range(n0, n1):
            w = blk(i, n >> 2)
            pr = (n >> 1) & 1
            r = np.sqrt(-2 * np.log(u(w[2 * pr])))
            ang = two_pi * u(w[2 * pr + 1])
            z = r * np.cos(ang) if n % 2 == 0 else r * np.sin(ang)
            ax, av, ae = drift(x, v, e, n * p["dt"])
            if p["integrator"] == 0:
                x, v, e = x + ax * p["dt"], v + av * p["dt"] + sig * z, e + ae * p["dt"]
            else:
                xp, vp, ep = x + ax * p["dt"], v + av * p["dt"] + sig * z, e + ae * p["dt"]
                bx, bv, be = drift(xp, vp, ep, (n + 1) * p["dt"])
                x, v, e = (x + 0.5 * (ax + bx) * p["dt"], v + 0.5 * (av + bv) * p["dt"] + sig * z,
                           e + 0.5 * (ae + be) * p["dt"])
        out.append((x, v, e))
    return np.array(out)


@pytest.mark.parametrize("over", [
    dict(),                                                           # config[0] model
    dict(integrator=1, dt=5e-3, A=0.5, omega=2 * math.pi * 0.1, D=0.05),  # config[3] model
    dict(precision=1, dt=1e-4, A1=2.0, A2=0.5, D=0.2, q=1.5, init_v=1),   # config[4] model
    dict(F0=-0.3, phi=0.1903, A1=-0.453, A2=-0.11325, L=1.0, e0=0.4, v0=-0.2),  # paper's Eq. 3
    dict(L=2.5, phi=0.3, integrator=1, init_v=1, gamma0=0.7),
])
def test_p12_brute_force_restatement(oracle, over):
    p = cfg(**over)
    seed, trajs = 4242, [0, 1, 2, 5, 2**32 + 7, 1_048_575, 4_194_303, 77]
    want = _brute(p, seed, trajs, 0, 16)
    for k, i in enumerate(trajs):
        x, v, e = oracle.init_many(p, seed, 1, traj_first=i)
        oracle.run(p, seed, x, v, e, 0, 16, traj_first=i)
        assert [x[0], v[0], e[0]] == pytest.approx(list(want[k]), rel=1e-13, abs=1e-15)


# ---------------------------------------------------------------------------------------------
# P13  invariants of the driver loop
# ---------------------------------------------------------------------------------------------

def test_p13_split_runs_and_index_independence(oracle):
    p = cfg()
    N = 64
    xa, va, ea = oracle.init_many(p, 42, N)
    xb, vb, eb = xa.copy(), va.copy(), ea.copy()
    oracle.run(p, 42, xa, va, ea, 0, 37)
    oracle.run(p, 42, xb, vb, eb, 0, 7)
    oracle.run(p, 42, xb, vb, eb, 7, 9)
    oracle.run(p, 42, xb, vb, eb, 16, 21, threads=4)
    assert np.array_equal(xa, xb) and np.array_equal(va, vb) and np.array_equal(ea, eb)
    # trajectory i depends only on (seed, i): strided subset == slice of the full run
    xs, vs, es = oracle.init_many(p, 42, N // 8, traj_first=3, traj_stride=8)
    oracle.run(p, 42, xs, vs, es, 0, 37, traj_first=3, traj_stride=8)
    assert np.array_equal(xs, xa[3::8]) and np.array_equal(vs, va[3::8]) and np.array_equal(es, ea[3::8])
    # and a different seed gives a different stream
    xc, vc, ec = oracle.init_many(p, 43, N)
    assert not np.array_equal(xc, oracle.init_many(p, 42, N)[0])


def test_moments_against_numpy(oracle):
    rng = np.random.default_rng(0)
    n = 1000
    x, v, e, x0 = (rng.normal(3, 2, n), rng.normal(-1, 0.5, n), rng.uniform(0, 2, n), rng.uniform(0, 1, n))
    m = oracle.moments(x, v, e, x0)
    want = dict(mean_x=x.mean(), var_x=x.var(), mean_v=v.mean(), var_v=v.var(), mean_e=e.mean(),
                mean_dx=(x - x0).mean(), mean_dx2=((x - x0)**2).mean(), mean_x2=(x * x).mean())
    for k in want:
        assert m[k] == pytest.approx(want[k], rel=1e-12)


def test_config0_orientation_magnitudes(oracle):
    """Sanity magnitudes only ('parity unpinned' for the ratchet current): the
    config[0] ensemble stays bounded and near the probe values var v ~ 1, <e> ~ 0.94."""
    wl = W.config0()
    p = wl.set_params(0)
    x, v, e = oracle.init_many(p, wl.seed, 1024)
    oracle.run(p, wl.seed, x, v, e, 0, wl.n_steps, threads=oracle.host_threads())
    assert 0.7 < v.var() < 1.4 and 0.8 < e.mean() < 1.1 and np.abs(x).max() < 30


# ---- headless presentation ------------------------------------------------

def _load_raster_fixture():
    pts, rows = [], []
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "raster_small.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        tok = line.split()
        if tok[0] == "counts":
            rows.append([int(t) for t in tok[1:]])
        else:
            pts.append((float(tok[0]), float(tok[1])))
    return np.array(pts), np.array(rows, np.uint32)


def test_raster_hand_counted_fixture(oracle):
    pts, want = _load_raster_fixture()
    got = oracle.raster(pts[:, 0], pts[:, 1], 1.0, 4, 2, -1.0, 1.0)
    assert np.array_equal(got, want)
    assert got.sum() == 6                      # two points fall outside the half-open velocity window


@pytest.mark.parametrize("L,W,H", [(1.0, 64, 48), (2.5, 1000, 7), (1.0, 1, 1)])
def test_raster_matches_numpy_histogram2d(oracle, L, W, H):
    rng = np.random.default_rng(5)
    n = 200_000
    x = rng.normal(0.0, 3.0 * L, n)            # many periods, both signs
    v = rng.normal(0.0, 1.0, n)
    v_min, v_max = -2.0, 2.5
    # keep points clear of bin edges: numpy bins by comparing with linspace edges, the rule divides
    fx = (x / L - np.floor(x / L)) * W
    fy = (v - v_min) / (v_max - v_min) * H
    ok = (np.abs(fx - np.round(fx)) > 1e-6) & (np.abs(fy - np.round(fy)) > 1e-6)
    x, v = x[ok], v[ok]
    got = oracle.raster(x, v, L, W, H, v_min, v_max)
    want, _, _ = np.histogram2d(v, np.mod(x, L), bins=[H, W], range=[[v_min, v_max], [0.0, L]])
    assert np.array_equal(got, want.astype(np.uint32))
    inside = (v >= v_min) & (v < v_max)
    assert got.sum() == inside.sum()


def test_raster_edges_and_nonfinite(oracle):
    x = np.array([0.0, -1e-20, 1.0 - 1e-17, np.nan, 0.5, 0.5, np.inf])
    v = np.array([0.0, 0.0, 0.0, 0.0, np.nan, 0.9999, 0.0])
    got = oracle.raster(x, v, 1.0, 8, 4, -1.0, 1.0)
    # x = -1e-20: xi - floor(xi) rounds to 1 -> last column; 1 - 1e-17 rounds to 1.0 -> f = 0 -> column 0
    assert got[2, 0] == 2 and got[2, 7] == 1 and got[3, 4] == 1 and got.sum() == 4


def test_colormap_ramp(oracle):
    counts = np.array([[0, 1, 2, 3], [4, 5, 1000, 2**32 - 1]], np.uint32)
    rgba = oracle.colormap(counts, 4)
    assert rgba.shape == (2, 4, 4) and np.all(rgba[..., 3] == 255)
    assert np.array_equal(rgba[..., 0], np.minimum(255, (255 * counts.astype(np.uint64)) // 4).astype(np.uint8))
    assert np.array_equal(rgba[..., 0], rgba[..., 1]) and np.array_equal(rgba[..., 0], rgba[..., 2])
    assert np.array_equal(oracle.colormap(counts, 1)[..., 0], np.where(counts > 0, 255, 0))


# ---- the paper's own workload: <v>(F0) -------------------------------------

def test_time_averaged_velocity_of_a_loaded_free_particle(oracle):
    """D = 0, no potential: the time average <x(t) - x(0)> / t converges to the stationary speed, the root of
    F0 + d e v - gamma0 v = 0 with e = q / (c + d v^2) (Eqs. 1-2 at rest); the sign of F0 selects the branch
    (reading G13: +F0 as printed)."""
    from scipy.optimize import brentq
    base = dict(W.DEFAULTS, A1=0.0, A2=0.0, D=0.0, v0=0.0, e0=0.0, dt=1e-3)
    for F0 in (-0.5, 0.3):
        p = dict(base, F0=F0)
        g = lambda vv: F0 + p["d"] * p["q"] / (p["c"] + p["d"] * vv * vv) * vv - p["gamma0"] * vv
        root = brentq(g, 0.5 * np.sign(F0), 3.0 * np.sign(F0))
        x, v, e = oracle.init_many(p, 3, 4)
        x0 = x.copy()
        n = 200_000
        oracle.run(p, 3, x, v, e, 0, n)
        assert np.allclose(v, root, rtol=1e-6)
        vbar = (x - x0) / (n * p["dt"])
        assert np.allclose(vbar, root, rtol=2e-2)           # transient of a few time units out of 200
        assert np.sign(vbar[0]) == np.sign(F0)


def test_paper_f0_sweep_workload_shape():
    wl = W.paper_f0_sweep(n_F0=17, F0_min=-1.0, F0_max=0.0, realisations=3, n_steps=100)
    assert wl.n_param_sets == 17 and wl.n_particles == 3 and wl.n_trajectories == 51
    f = [wl.set_params(s)["F0"] for s in range(17)]
    assert f[0] == -1.0 and f[-1] == 0.0 and np.allclose(np.diff(f), 1 / 16)
    p = wl.set_params(5)
    assert p["phi"] == 0.1903 and p["A1"] == -0.453 and p["A2"] == -0.11325 and p["L"] == 1.0


# ---- NEXT-4: the paper's generator family --------------------------------------------

def test_xorshift128_known_answers(oracle):
    state, outs = None, []
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "xorshift128_kat.txt")):
        tok = line.split("#")[0].split()
        if tok and tok[0] == "state":
            state = [int(t) for t in tok[1:]]
        elif tok and tok[0] == "out":
            outs.append(int(tok[1]))
    assert len(outs) == 5
    for want in outs:
        got, state = oracle.xorshift128(state)
        assert got == want and state[3] == want


def test_xorshift128_python_restatement_and_bijectivity(oracle):
    rng = np.random.default_rng(11)
    seen = set()
    for _ in range(200):
        s = [int(t) for t in rng.integers(0, 2**32, 4)]
        x, y, z, w = s
        t = (x ^ (x << 11)) & 0xffffffff
        want = [y, z, w, (w ^ (w >> 19) ^ t ^ (t >> 8)) & 0xffffffff]
        out, new = oracle.xorshift128(s)
        assert new == want and out == want[3]
        seen.add(tuple(new))
    assert len(seen) == 200
    # the transition is linear over GF(2): T(a ^ b) = T(a) ^ T(b), and T(0) = 0 (the forbidden state)
    a = [int(t) for t in rng.integers(0, 2**32, 4)]
    b = [int(t) for t in rng.integers(0, 2**32, 4)]
    ta, tb = oracle.xorshift128(a)[1], oracle.xorshift128(b)[1]
    tab = oracle.xorshift128([p ^ q for p, q in zip(a, b)])[1]
    assert tab == [p ^ q for p, q in zip(ta, tb)]
    assert oracle.xorshift128([0, 0, 0, 0]) == (0, [0, 0, 0, 0])


def test_xorshift_seed_and_stream_layout(oracle):
    seed, traj = 0x1234_5678_9abc_def0, 77
    s = oracle.xorshift_seed(seed, traj)
    assert s == [int(t) for t in oracle.block(seed, traj, 2**64 - 2)] and any(s)
    # pair p of steps (2p, 2p + 1) uses outputs 2p and 2p + 1
    outs = []
    for _ in range(6):
        o, s = oracle.xorshift128(s)
        outs.append(o)
    for n in range(6):
        a, b = outs[2 * (n // 2)], outs[2 * (n // 2) + 1]
        for prec in (0, 1):
            u1, u2 = oracle.uniform(a, prec), oracle.uniform(b, prec)
            r = math.sqrt(-2.0 * math.log(u1))
            want = r * (math.cos(2 * math.pi * u2) if n % 2 == 0 else math.sin(2 * math.pi * u2))
            assert oracle.normal_xorshift(seed, traj, n, prec) == pytest.approx(want, rel=1e-14, abs=1e-15)


def test_xorshift_normals_moments(oracle):
    """Normals of the xorshift stream over many trajectories and steps: mean 0, variance 1, kurtosis 3."""
    p = dict(W.DEFAULTS, rng=1, A1=0.0, A2=0.0, d=0.0, q=0.0, c=0.0, gamma0=1.0 / 2.0**-10, dt=2.0**-10,
             D=0.5 / 2.0**-10)                      # EM: v_{n+1} = z_n exactly (sigma = 1)
    n_traj, zs = 20_000, []
    x, v, e = oracle.init_many(p, 5, n_traj)
    for n in range(24):
        oracle.run(p, 5, x, v, e, n, 1, threads=8)
        zs.append(v.copy())
    z = np.concatenate(zs)
    N = z.size
    assert abs(z.mean()) < 3 / math.sqrt(N)
    assert abs(z.var() - 1) < 3 * math.sqrt(2 / N)
    assert abs(np.mean(z**4) - 3) < 3 * math.sqrt(96 / N)
    # consecutive steps (cos / sin of one pair, then the next pair) are uncorrelated
    zz = np.stack(zs)
    for lag in (1, 2):
        c = np.mean(zz[:-lag] * zz[lag:])
        assert abs(c) < 4 / math.sqrt(zz[:-lag].size)
    # and the first steps equal the definition evaluated from the seed
    assert zs[3][17] == oracle.normal_xorshift(5, 17, 3, 0)


def test_xorshift_run_matches_stepwise_definition_and_splits(oracle):
    p = dict(W.config3().set_params(0), rng=1)
    seed, n = 99, 6
    x, v, e = oracle.init_many(p, seed, n, 40)
    x1, v1, e1 = x.copy(), v.copy(), e.copy()
    x2, v2, e2 = x.copy(), v.copy(), e.copy()
    oracle.run(p, seed, x, v, e, 0, 23, 40)
    for a, b in ((0, 5), (5, 1), (6, 7), (13, 10)):         # odd and even split points
        oracle.run(p, seed, x1, v1, e1, a, b, 40)
    assert np.array_equal(x, x1) and np.array_equal(v, v1) and np.array_equal(e, e1)
    L = oracle.lib()
    pp = oracle.make_params(p)
    import ctypes as C
    for k in range(n):
        xs, vs, es = (C.c_double(t[k]) for t in (x2, v2, e2))
        for step in range(23):
            L.abo_step(C.byref(pp), seed, 40 + k, step, C.byref(xs), C.byref(vs), C.byref(es))
        assert (xs.value, vs.value, es.value) == (x[k], v[k], e[k])
    # a different stream from the Philox one, same physics
    xp, vp, ep = oracle.init_many(dict(p, rng=0), seed, n, 40)
    oracle.run(dict(p, rng=0), seed, xp, vp, ep, 0, 23, 40)
    assert not np.array_equal(v, vp)


# ---------------------------------------------------------------------------------------------
# Reading G14: "relative error 1e-5 after 100 steps" is scale-relative per variable.
# The element-wise reading cannot be met by ANY fp32 integration of config[0], however exact its
# functions: this restatement does every state update in IEEE float32 (one rounding per operation,
# no FMA) with the normals and the cosine evaluated in fp64 and rounded once.
# ---------------------------------------------------------------------------------------------

def test_g14_elementwise_relative_error_is_unattainable_in_fp32(oracle):
    wl = W.config0()
    p = wl.set_params(0)
    n, steps = wl.n_particles, 100
    x, v, e = oracle.init_many(p, wl.seed, n)
    z = oracle.normals(wl.seed, 0, n, 0, steps, 0)
    f32 = np.float32
    xs, vs, es = x.astype(f32), v.astype(f32), e.astype(f32)
    dt, g0, d, q, c = (f32(p[k]) for k in ("dt", "gamma0", "d", "q", "c"))
    sig = f32(math.sqrt(2 * p["D"] * p["dt"]))
    kk = 2 * math.pi / p["L"]
    for n_ in range(steps):
        th = kk * (xs.astype(np.float64) + p["phi"])
        f = (-(kk * (p["A1"] * np.cos(th) + 2 * p["A2"] * np.cos(2 * th))) + p["F0"]).astype(f32)
        av = (d * es - g0) * vs + f
        ae = q - es * (c + d * (vs * vs))
        xs, vs, es = xs + dt * vs, (vs + dt * av) + sig * z[:, n_].astype(f32), es + dt * ae
        assert xs.dtype == f32 and vs.dtype == f32 and es.dtype == f32
    oracle.run(p, wl.seed, x, v, e, 0, steps)
    want = np.stack([x, v, e], 1)
    got = np.stack([xs, vs, es], 1).astype(np.float64)
    rms = np.sqrt(np.mean(want * want, axis=0))
    scale_rel = (np.abs(got - want) / np.maximum(np.abs(want), rms)).max(axis=0)
    elem_rel_v = np.abs(got[:, 1] - want[:, 1]) / np.abs(want[:, 1])
    assert np.all(scale_rel < 1e-5), scale_rel                # the reading taken: met, with room
    assert np.mean(elem_rel_v > 1e-5) > 0.005, np.mean(elem_rel_v > 1e-5)   # the other reading: not attainable
    assert elem_rel_v.max() > 1e-4
