"""Shared helpers of the parity tests: oracle runs on index subsets, the G14 error metric, SE."""
import math

import numpy as np


def oracle_states(oracle, params, seed, traj_idx, n_steps, step_first=0, state=None, threads=None):
    """Oracle state (float64 [len(traj_idx), 3]) of the listed GLOBAL trajectory indices after
    steps [step_first, step_first + n_steps), starting from the init block (or `state`)."""
    traj_idx = np.asarray(traj_idx, dtype=np.uint64)
    threads = threads or oracle.host_threads()
    # contiguous or strided runs go through one call; arbitrary index lists one trajectory at a time
    d = np.diff(traj_idx.astype(np.int64))
    out = np.empty((traj_idx.size, 3), np.float64)
    if traj_idx.size > 1 and np.all(d == d[0]) and d[0] > 0:
        first, stride = int(traj_idx[0]), int(d[0])
        if state is None:
            x, v, e = oracle.init_many(params, seed, traj_idx.size, first, stride)
        else:
            x, v, e = (np.ascontiguousarray(state[:, j]) for j in range(3))
        oracle.run(params, seed, x, v, e, step_first, n_steps, first, stride, threads=threads)
        out[:, 0], out[:, 1], out[:, 2] = x, v, e
        return out
    for k, i in enumerate(traj_idx):
        if state is None:
            x, v, e = oracle.init_many(params, seed, 1, int(i))
        else:
            x, v, e = (np.array([state[k, j]]) for j in range(3))
        oracle.run(params, seed, x, v, e, step_first, n_steps, int(i))
        out[k] = (x[0], v[0], e[0])
    return out


def oracle_states_all(oracle, sets, n_particles, seed, n_steps, threads=None):
    """Oracle state (float64 [n_sets * n_particles, 3], local order k = set * n_particles + r) of EVERY trajectory
    of an ensemble after n_steps steps from the init block.  One set: one call, split over the host threads
    by trajectory range.  Many sets: a pool of host threads, each taking a contiguous range of sets and calling
    the oracle once per set (single-threaded calls; ctypes drops the GIL).  No arithmetic here."""
    import concurrent.futures as cf
    threads = threads or oracle.host_threads()
    n_sets = len(sets)
    out = np.empty((n_sets * n_particles, 3), np.float64)
    if n_sets == 1:
        x, v, e = oracle.init_many(sets[0], seed, n_particles, 0)
        oracle.run(sets[0], seed, x, v, e, 0, n_steps, 0, threads=threads)
        out[:, 0], out[:, 1], out[:, 2] = x, v, e
        return out

    def work(s0, s1):
        for s in range(s0, s1):
            first = s * n_particles
            x, v, e = oracle.init_many(sets[s], seed, n_particles, first)
            oracle.run(sets[s], seed, x, v, e, 0, n_steps, first, threads=1)
            blk = out[first:first + n_particles]
            blk[:, 0], blk[:, 1], blk[:, 2] = x, v, e

    bounds = np.linspace(0, n_sets, threads + 1).astype(int)
    with cf.ThreadPoolExecutor(threads) as pool:
        for f in [pool.submit(work, int(bounds[i]), int(bounds[i + 1])) for i in range(threads)]:
            f.result()
    return out


def scale_rel_err_elements(got, want, n_sets=1):
    """Reading G14 element by element: |got - want| / max(|want|, RMS of that variable over the ensemble the
    trajectory belongs to -- the realisations of ITS parameter set).  Returns the [n, 3] array of errors."""
    got, want = np.asarray(got, np.float64), np.asarray(want, np.float64)
    w = want.reshape(n_sets, -1, 3)
    rms = np.sqrt(np.mean(w * w, axis=1, keepdims=True))                     # [n_sets, 1, 3]
    scale = np.maximum(np.abs(w), np.maximum(rms, 1e-300))
    return (np.abs(got.reshape(n_sets, -1, 3) - w) / scale).reshape(-1, 3)


def scale_rel_err(got, want):
    """Reading G14: per variable, |got - want| / max(|want|, RMS of that variable over
    the compared ensemble).  Returns the max over trajectories, per variable (x, v, e)."""
    got, want = np.asarray(got, np.float64), np.asarray(want, np.float64)
    rms = np.sqrt(np.mean(want * want, axis=0))
    scale = np.maximum(np.abs(want), np.maximum(rms, 1e-300))
    return (np.abs(got - want) / scale).max(axis=0)


def se_mean(a):
    return float(np.std(a) / math.sqrt(a.size))


def se_var(a):
    """Standard error of the population variance: sqrt((m4 - s^4) / N)."""
    c = a - a.mean()
    m2, m4 = np.mean(c**2), np.mean(c**4)
    return float(math.sqrt(max(m4 - m2 * m2, 0.0) / a.size))


def global_indices(wl, local_idx, traj_base=0, set_stride=0):
    """Local trajectory order k = set * n_particles + r -> global stream index."""
    local_idx = np.asarray(local_idx, dtype=np.int64)
    stride = set_stride or wl.n_particles
    s, r = np.divmod(local_idx, wl.n_particles)
    return (traj_base + s * stride + r).astype(np.uint64)
