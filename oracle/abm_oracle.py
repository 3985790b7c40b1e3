"""ctypes front end of the CPU oracle (oracle/abm_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from paper_1104_2499_b200 and holds no arithmetic of
its own: every number comes from the C functions, which cite the paper passage they follow.
"""
import ctypes as C
import os
import threading

import numpy as np

from . import build as _build

_LIB = None


class Params(C.Structure):
    """Mirror of `abo_params` (oracle/abm_oracle.h)."""
    _fields_ = [("precision", C.c_int32), ("integrator", C.c_int32), ("init_v", C.c_int32),
                ("rng", C.c_int32),
                ("dt", C.c_double), ("gamma0", C.c_double), ("q", C.c_double), ("c", C.c_double),
                ("d", C.c_double), ("D", C.c_double), ("F0", C.c_double), ("A", C.c_double),
                ("omega", C.c_double), ("L", C.c_double), ("A1", C.c_double), ("A2", C.c_double),
                ("phi", C.c_double), ("v0", C.c_double), ("e0", C.c_double)]


_FIELDS = [f[0] for f in Params._fields_]


def make_params(cfg: dict) -> Params:
    """cfg: plain dict of workload parameters (see paper_1104_2499_b200/workloads.py)."""
    p = Params()
    for k in _FIELDS:
        if k in cfg:
            setattr(p, k, cfg[k])
    return p


def lib():
    global _LIB
    if _LIB is None:
        path = _build.build()
        L = C.CDLL(path)
        u32p, dp = C.POINTER(C.c_uint32), C.POINTER(C.c_double)
        pp = C.POINTER(Params)
        L.abo_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.abo_philox4x32_10.restype = None
        L.abo_block.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, u32p]
        L.abo_block.restype = None
        L.abo_uniform.argtypes = [C.c_uint32, C.c_int32]
        L.abo_uniform.restype = C.c_double
        L.abo_normal.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_int32]
        L.abo_normal.restype = C.c_double
        L.abo_normals.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint64,
                                  C.c_int32, dp]
        L.abo_normals.restype = None
        L.abo_potential.argtypes = [pp, C.c_double]
        L.abo_potential.restype = C.c_double
        L.abo_rhs.argtypes = [pp, C.c_double, C.c_double, C.c_double, C.c_double, dp, dp, dp]
        L.abo_rhs.restype = None
        L.abo_init.argtypes = [pp, C.c_uint64, C.c_uint64, dp, dp, dp]
        L.abo_init.restype = None
        L.abo_step.argtypes = [pp, C.c_uint64, C.c_uint64, C.c_uint64, dp, dp, dp]
        L.abo_step.restype = None
        L.abo_init_many.argtypes = [pp, C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint64, dp, dp, dp]
        L.abo_init_many.restype = None
        L.abo_run.argtypes = [pp, C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint64, C.c_uint64,
                              C.c_uint64, dp, dp, dp]
        L.abo_run.restype = None
        L.abo_moments.argtypes = [dp, dp, dp, dp, C.c_uint64, dp]
        L.abo_moments.restype = None
        L.abo_xorshift128.argtypes = [u32p]
        L.abo_xorshift128.restype = C.c_uint32
        L.abo_xorshift_seed.argtypes = [C.c_uint64, C.c_uint64, u32p]
        L.abo_xorshift_seed.restype = None
        L.abo_normal_xorshift.argtypes = [C.c_uint64, C.c_uint64, C.c_uint64, C.c_int32]
        L.abo_normal_xorshift.restype = C.c_double
        L.abo_raster.argtypes = [dp, dp, C.c_uint64, C.c_double, C.c_uint32, C.c_uint32, C.c_double,
                                 C.c_double, u32p]
        L.abo_raster.restype = None
        L.abo_colormap.argtypes = [u32p, C.c_uint64, C.c_uint32, C.POINTER(C.c_uint8)]
        L.abo_colormap.restype = None
        _LIB = L
    return _LIB


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xffffffff for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xffffffff for v in key])
    o = (C.c_uint32 * 4)()
    lib().abo_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def block(seed, traj, b):
    o = (C.c_uint32 * 4)()
    lib().abo_block(seed, traj, b & 0xffffffffffffffff, o)
    return [int(v) for v in o]


def uniform(w, precision):
    return lib().abo_uniform(int(w), int(precision))


def normal(seed, traj, n, precision):
    return lib().abo_normal(seed, traj, n, int(precision))


def normals(seed, traj_first, n_traj, step_first, n_steps, precision):
    """-> float64 array [n_traj, n_steps] of the normals the run consumes."""
    out = np.empty((n_traj, n_steps), np.float64)
    lib().abo_normals(seed, traj_first, n_traj, step_first, n_steps, int(precision), _dp(out))
    return out


def potential(cfg, x):
    p = make_params(cfg)
    return lib().abo_potential(C.byref(p), float(x))


def rhs(cfg, x, v, e, t):
    p = make_params(cfg)
    ax, av, ae = C.c_double(), C.c_double(), C.c_double()
    lib().abo_rhs(C.byref(p), x, v, e, t, C.byref(ax), C.byref(av), C.byref(ae))
    return ax.value, av.value, ae.value


def init_many(cfg, seed, n_traj, traj_first=0, traj_stride=1):
    """-> (x, v, e) float64 arrays of trajectories traj_first + k * traj_stride."""
    p = make_params(cfg)
    x = np.empty(n_traj, np.float64)
    v = np.empty(n_traj, np.float64)
    e = np.empty(n_traj, np.float64)
    lib().abo_init_many(C.byref(p), seed, traj_first, traj_stride, n_traj, _dp(x), _dp(v), _dp(e))
    return x, v, e


def run(cfg, seed, x, v, e, step_first, n_steps, traj_first=0, traj_stride=1, threads=1):
    """Advance state arrays in place over steps [step_first, step_first + n_steps).

    threads > 1 splits the SAME plain loop by trajectory range over host threads (ctypes drops
    the GIL); each trajectory is still integrated by the single-threaded C code.
    """
    p = make_params(cfg)
    n = x.shape[0]
    assert x.dtype == np.float64 and x.flags.c_contiguous
    if threads <= 1 or n < 2 * threads:
        lib().abo_run(C.byref(p), seed, traj_first, traj_stride, n, step_first, n_steps,
                      _dp(x), _dp(v), _dp(e))
        return
    L = lib()
    bounds = np.linspace(0, n, threads + 1).astype(np.int64)

    def work(a, b):
        L.abo_run(C.byref(p), seed, traj_first + int(a) * traj_stride, traj_stride, int(b - a),
                  step_first, n_steps, _dp(x[a:b]), _dp(v[a:b]), _dp(e[a:b]))

    ts = [threading.Thread(target=work, args=(bounds[i], bounds[i + 1])) for i in range(threads)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()


def moments(x, v, e, x0):
    """-> dict of the eight ensemble moments (population normalisation)."""
    x, v, e, x0 = (np.ascontiguousarray(a, np.float64) for a in (x, v, e, x0))
    out = np.empty(8, np.float64)
    lib().abo_moments(_dp(x), _dp(v), _dp(e), _dp(x0), x.shape[0], _dp(out))
    names = ["mean_x", "var_x", "mean_v", "var_v", "mean_e", "mean_dx", "mean_dx2", "mean_x2"]
    return dict(zip(names, out.tolist()))


def xorshift128(state):
    """state: 4 uint32 (x, y, z, w) -> (output, new state)"""
    s = (C.c_uint32 * 4)(*[int(t) for t in state])
    out = lib().abo_xorshift128(s)
    return int(out), [int(t) for t in s]


def xorshift_seed(seed, traj):
    s = (C.c_uint32 * 4)()
    lib().abo_xorshift_seed(seed, traj, s)
    return [int(t) for t in s]


def normal_xorshift(seed, traj, n, precision):
    return lib().abo_normal_xorshift(seed, traj, n, int(precision))


def raster(x, v, L, width, height, v_min, v_max):
    """-> uint32 [height, width] histogram of (x mod L, v)."""
    x, v = (np.ascontiguousarray(a, np.float64) for a in (x, v))
    counts = np.zeros((height, width), np.uint32)
    lib().abo_raster(_dp(x), _dp(v), x.shape[0], float(L), width, height, float(v_min), float(v_max),
                     counts.ctypes.data_as(C.POINTER(C.c_uint32)))
    return counts


def colormap(counts, saturation):
    counts = np.ascontiguousarray(counts, np.uint32)
    rgba = np.zeros(counts.shape + (4,), np.uint8)
    lib().abo_colormap(counts.ctypes.data_as(C.POINTER(C.c_uint32)), counts.size, int(saturation),
                       rgba.ctypes.data_as(C.POINTER(C.c_uint8)))
    return rgba


def host_threads():
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
