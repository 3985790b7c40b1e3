"""Thin ctypes binding of the C ABI in include/abm.h -- same names, argument marshalling only.

Every step of the path runs in the CUDA kernels behind `libabm_b200.so`; this module never
computes anything itself and has no fallback: if the library is missing or a call fails it raises.
PyTorch is used by callers for device memory (snapshot buffers) and streams; this module only
passes raw pointers / stream handles through.
"""
import ctypes as C
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libabm_b200.so")

ABM_OK, ABM_EINVAL, ABM_ENOMEM, ABM_ECUDA, ABM_ESTATE, ABM_ELIMIT = 0, -1, -2, -3, -4, -5
ABM_FP32, ABM_FP64 = 0, 1
ABM_EULER_MARUYAMA, ABM_HEUN = 0, 1
ABM_ACCURACY_AUTO, ABM_ACCURACY_FAST, ABM_ACCURACY_PRECISE = 0, 1, 2
ABM_ACCURACY_BEYOND_TOLERANCE = 0x100
ABM_RNG_PHILOX, ABM_RNG_XORSHIFT128 = 0, 1
ABM_STEP_KERNEL_AUTO, ABM_STEP_KERNEL_PER_THREAD, ABM_STEP_KERNEL_SPLIT_WARPS = 0, 1, 2
ABM_N_SUMS = 8
ABM_STATIC_MAX_SLICES = 65536        # partial records in the built-in scratch of abm_frame_moment_sums_static

# abm_params.step_kernel of records built by make_params when the caller names none.  The GPU tests flip it
# to run every case through both step kernels (results are bit-identical whichever runs).
DEFAULT_STEP_KERNEL = ABM_STEP_KERNEL_AUTO


class abm_params(C.Structure):
    """Mirror of `abm_params` (include/abm.h)."""
    _fields_ = [
        ("struct_size", C.c_uint32), ("precision", C.c_uint32), ("integrator", C.c_uint32),
        ("init_v", C.c_uint32), ("snapshot_every", C.c_uint32), ("accuracy", C.c_uint32),
        ("rng", C.c_uint32), ("step_kernel", C.c_uint32),
        ("dt", C.c_double), ("gamma0", C.c_double), ("q", C.c_double), ("c", C.c_double),
        ("d", C.c_double), ("D", C.c_double), ("F0", C.c_double), ("A", C.c_double),
        ("omega", C.c_double), ("L", C.c_double), ("A1", C.c_double), ("A2", C.c_double),
        ("phi", C.c_double), ("v0", C.c_double), ("e0", C.c_double),
        ("traj_base", C.c_uint64), ("traj_set_stride", C.c_uint64), ("stream", C.c_void_p),
    ]


class abm_moment(C.Structure):
    """Mirror of `abm_moment` (include/abm.h), 80 bytes."""
    _fields_ = [("n", C.c_uint64), ("step", C.c_uint64), ("mean_x", C.c_double),
                ("var_x", C.c_double), ("mean_v", C.c_double), ("var_v", C.c_double),
                ("mean_e", C.c_double), ("mean_dx", C.c_double), ("mean_dx2", C.c_double),
                ("mean_x2", C.c_double)]


MOMENT_DTYPE = np.dtype([("n", "<u8"), ("step", "<u8"), ("mean_x", "<f8"), ("var_x", "<f8"),
                         ("mean_v", "<f8"), ("var_v", "<f8"), ("mean_e", "<f8"),
                         ("mean_dx", "<f8"), ("mean_dx2", "<f8"), ("mean_x2", "<f8")])

EXPORTS = ["abm_create", "abm_step", "abm_snapshot", "abm_snapshot_host", "abm_moments", "abm_moments_async",
           "abm_moment_sums", "abm_moment_sums_dev", "abm_moments_from_sums", "abm_time_averaged_velocity",
           "abm_frame_moment_sums_static", "abm_raster", "abm_get_step", "abm_get_accuracy", "abm_destroy", "abm_trim", "abm_philox_blocks",
           "abm_philox_blocks_loop", "abm_strerror", "abm_abi_version"]

_lib = None


class AbmError(RuntimeError):
    def __init__(self, fn, status):
        self.status = status
        msg = lib().abm_strerror(status).decode() if _lib is not None else str(status)
        super().__init__(f"{fn} failed: {status} ({msg})")


def lib():
    """Load libabm_b200.so (built by paper_1104_2499_b200/build.py).  No fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1104_2499_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, u64, u32 = C.c_void_p, C.c_uint64, C.c_uint32
        L.abm_create.argtypes = [C.POINTER(abm_params), u64, u32, u64, C.POINTER(vp)]
        L.abm_step.argtypes = [vp, u64]
        L.abm_snapshot.argtypes = [vp, vp, C.c_size_t]
        L.abm_snapshot_host.argtypes = [vp, vp, C.c_size_t]
        L.abm_moments.argtypes = [vp, vp]
        L.abm_moments_async.argtypes = [vp, vp]
        L.abm_moment_sums.argtypes = [vp, vp]
        L.abm_moment_sums_dev.argtypes = [vp, vp]
        L.abm_moments_from_sums.argtypes = [vp, u32, u64, vp]
        L.abm_time_averaged_velocity.argtypes = [vp, vp]
        L.abm_frame_moment_sums_static.argtypes = [vp, vp, C.c_size_t, u32, u64, u32, vp, vp]
        L.abm_raster.argtypes = [vp, vp, u32, u32, C.c_double, C.c_double, vp, u32]
        L.abm_get_step.argtypes = [vp, C.POINTER(u64)]
        L.abm_get_accuracy.argtypes = [vp, C.POINTER(u32)]
        L.abm_destroy.argtypes = [vp]
        L.abm_trim.argtypes = []
        L.abm_philox_blocks.argtypes = [u64, u64, u64, u64, u64, vp, vp]
        L.abm_philox_blocks_loop.argtypes = [u64, u64, u64, u64, u64, u32, u32, vp, vp]
        for n in EXPORTS[:-2]:
            getattr(L, n).restype = C.c_int
        L.abm_strerror.argtypes = [C.c_int]
        L.abm_strerror.restype = C.c_char_p
        L.abm_abi_version.argtypes = []
        L.abm_abi_version.restype = C.c_uint32
        _lib = L
    return _lib


_PARAM_KEYS = ["precision", "integrator", "init_v", "snapshot_every", "accuracy", "rng", "step_kernel", "dt", "gamma0", "q", "c", "d",
               "D", "F0", "A", "omega", "L", "A1", "A2", "phi", "v0", "e0", "traj_base",
               "traj_set_stride"]


def make_params(param_sets, stream=0, **common):
    """list of dicts (one per parameter set) -> ctypes array of abm_params."""
    arr = (abm_params * len(param_sets))()
    for s, d in enumerate(param_sets):
        p = arr[s]
        p.struct_size = C.sizeof(abm_params)
        p.step_kernel = DEFAULT_STEP_KERNEL
        for k in _PARAM_KEYS:
            if k in common:
                setattr(p, k, common[k])
            elif k in d:
                setattr(p, k, d[k])
        p.stream = stream or None
    return arr


def _check(fn, status):
    if status != ABM_OK:
        raise AbmError(fn, status)


# ---- the calls, one-to-one -------------------------------------------------------------------

def abm_create(params, n_particles, n_param_sets, seed):
    h = C.c_void_p()
    _check("abm_create", lib().abm_create(params, n_particles, n_param_sets, seed, C.byref(h)))
    return h


def abm_step(ctx, n_steps):
    _check("abm_step", lib().abm_step(ctx, n_steps))


def abm_snapshot(ctx, dev_ptr, stride_bytes):
    _check("abm_snapshot", lib().abm_snapshot(ctx, dev_ptr, stride_bytes))


def abm_moments_async(ctx, n_param_sets, out):
    """Enqueue the reduction and the copy into `out` (caller-owned record array [n_param_sets], pinned for a
    true asynchronous copy) without waiting; `out` is defined once the caller has synchronised the stream."""
    assert out.dtype == MOMENT_DTYPE and out.shape == (n_param_sets,) and out.flags.c_contiguous
    _check("abm_moments_async", lib().abm_moments_async(ctx, out.ctypes.data))
    return out


def abm_snapshot_host(ctx, host_array, stride_bytes):
    _check("abm_snapshot_host", lib().abm_snapshot_host(ctx, host_array.ctypes.data, stride_bytes))


def abm_moments(ctx, n_param_sets, out=None):
    """`out`: optional caller-owned record array [n_param_sets] (e.g. a view of pinned host memory, which
    makes the device->host copy a true DMA); a fresh pageable array otherwise."""
    if out is None:
        out = np.zeros(n_param_sets, MOMENT_DTYPE)
    assert out.dtype == MOMENT_DTYPE and out.shape == (n_param_sets,) and out.flags.c_contiguous
    _check("abm_moments", lib().abm_moments(ctx, out.ctypes.data))
    return out


def abm_moment_sums(ctx, n_param_sets, out=None):
    if out is None:
        out = np.zeros((n_param_sets, ABM_N_SUMS), np.float64)
    assert out.dtype == np.float64 and out.shape == (n_param_sets, ABM_N_SUMS) and out.flags.c_contiguous
    _check("abm_moment_sums", lib().abm_moment_sums(ctx, out.ctypes.data))
    return out


def abm_moment_sums_dev(ctx, dev_ptr):
    """Enqueue the reduction and a device-to-device copy of the raw sums [n_param_sets][8] to `dev_ptr`."""
    _check("abm_moment_sums_dev", lib().abm_moment_sums_dev(ctx, dev_ptr))


def abm_moments_from_sums(sums, step):
    sums = np.ascontiguousarray(sums, np.float64)
    out = np.zeros(sums.shape[0], MOMENT_DTYPE)
    _check("abm_moments_from_sums",
           lib().abm_moments_from_sums(sums.ctypes.data, sums.shape[0], step, out.ctypes.data))
    return out


def abm_frame_moment_sums_static(dev_frame, dev_frame0, stride_bytes, precision, n_particles, n_param_sets,
                                 dev_out, stream=0):
    """The eight moment sums per set of a caller-owned device frame, written to caller-owned device memory
    [n_param_sets][8], without any device allocation by the library (its scratch is a fixed array inside the
    library image: at most ABM_STATIC_MAX_SLICES slices of 4096 trajectories, else ABM_ELIMIT).  For
    callers that own all device memory themselves or may not allocate once their loop runs.  Calls
    share that scratch: keep them on one stream.  The first call per GPU belongs to start-up."""
    _check("abm_frame_moment_sums_static",
           lib().abm_frame_moment_sums_static(dev_frame, dev_frame0 or None, stride_bytes, precision, n_particles,
                                              n_param_sets, dev_out, stream or None))


def abm_time_averaged_velocity(ctx, n_param_sets):
    out = np.zeros(n_param_sets, np.float64)
    _check("abm_time_averaged_velocity", lib().abm_time_averaged_velocity(ctx, out.ctypes.data))
    return out


def abm_raster(ctx, dev_counts, width, height, v_min, v_max, dev_rgba=None, saturation=1):
    _check("abm_raster", lib().abm_raster(ctx, dev_counts, width, height, v_min, v_max, dev_rgba, saturation))


def abm_get_step(ctx):
    n = C.c_uint64()
    _check("abm_get_step", lib().abm_get_step(ctx, C.byref(n)))
    return n.value


def abm_get_accuracy(ctx):
    m = C.c_uint32()
    _check("abm_get_accuracy", lib().abm_get_accuracy(ctx, C.byref(m)))
    return m.value


def abm_destroy(ctx):
    _check("abm_destroy", lib().abm_destroy(ctx))


def abm_trim():
    _check("abm_trim", lib().abm_trim())


def abm_philox_blocks_loop(seed, traj_first, n_traj, block_first, n_blocks, loop_shape, frame_every_blocks,
                           dev_ptr, stream=0):
    _check("abm_philox_blocks_loop",
           lib().abm_philox_blocks_loop(seed, traj_first, n_traj, block_first, n_blocks, loop_shape,
                                        frame_every_blocks, dev_ptr, stream or None))


def abm_philox_blocks(seed, traj_first, n_traj, block_first, n_blocks, dev_ptr, stream=0):
    _check("abm_philox_blocks",
           lib().abm_philox_blocks(seed, traj_first, n_traj, block_first & 0xffffffffffffffff,
                                   n_blocks, dev_ptr, stream or None))


def pinned_moment_buffers(n_param_sets):
    """(records, sums) numpy views of pinned host memory (torch owns it) for abm_moments / abm_moment_sums."""
    import torch
    rec = torch.zeros(n_param_sets * MOMENT_DTYPE.itemsize, dtype=torch.uint8, pin_memory=True)
    sums = torch.zeros((n_param_sets, ABM_N_SUMS), dtype=torch.float64, pin_memory=True)
    out = rec.numpy().view(MOMENT_DTYPE)
    out_s = sums.numpy()
    out.flags.writeable = True
    return (out, rec), (out_s, sums)


# ---- convenience wrapper (owns the handle and the torch snapshot buffer) ----------------------

class Ensemble:
    """A context plus the caller-owned device snapshot buffer (a torch tensor).

    `param_sets`: list of parameter dicts (workloads.Workload.set_params), or an abm_params
    array from make_params (then stream / snapshot_every / traj_base must already be set in it).
    Marshalling only.
    """

    def __init__(self, param_sets, n_particles, seed, snapshot_every=0, stream=None,
                 traj_base=0, traj_set_stride=0, accuracy=ABM_ACCURACY_AUTO, rng=None, step_kernel=None):
        import torch
        self._torch = torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1104_2499_b200 needs a CUDA device (no CPU fallback)")
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self.n_sets = len(param_sets)
        self.n_particles = n_particles
        self.n_traj = n_particles * self.n_sets
        if isinstance(param_sets, C.Array):      # already marshalled (make_params) by the caller
            params = param_sets
        else:
            common = dict(snapshot_every=snapshot_every, traj_base=traj_base,
                          traj_set_stride=traj_set_stride, accuracy=accuracy)
            if rng is not None:          # else the parameter records decide (default Philox)
                common["rng"] = rng
            if step_kernel is not None:  # else the parameter records, else DEFAULT_STEP_KERNEL
                common["step_kernel"] = step_kernel
            params = make_params(param_sets, stream=self.stream.cuda_stream, **common)
        self.fp64 = int(params[0].precision) == 1
        self.ctx = abm_create(params, n_particles, self.n_sets, seed)
        self.frame = None

    def bind_snapshot(self, with_e=False):
        """Allocate (once) and bind a device frame: [n_traj, 2] (x, v) or [n_traj, 4] (x, v, e, 1)."""
        torch = self._torch
        cols = 4 if with_e else 2
        dtype = torch.float64 if self.fp64 else torch.float32
        if self.frame is None or self.frame.shape[1] != cols:
            with torch.cuda.stream(self.stream):
                self.frame = torch.empty((self.n_traj, cols), dtype=dtype, device="cuda")
        abm_snapshot(self.ctx, self.frame.data_ptr(), cols * self.frame.element_size())
        return self.frame

    def unbind_snapshot(self):
        abm_snapshot(self.ctx, None, 0)

    def step(self, n):
        abm_step(self.ctx, n)

    def moments(self, out=None):
        return abm_moments(self.ctx, self.n_sets, out)

    def moments_async(self, out):
        return abm_moments_async(self.ctx, self.n_sets, out)

    def moment_sums(self, out=None):
        return abm_moment_sums(self.ctx, self.n_sets, out)

    def moment_sums_dev(self, out):
        """Raw sums into rows of a caller-owned float64 CUDA tensor [n_sets, 8] (no host round trip)."""
        assert out.is_cuda and out.dtype == self._torch.float64 and out.is_contiguous() \
            and tuple(out.shape) == (self.n_sets, ABM_N_SUMS)
        abm_moment_sums_dev(self.ctx, out.data_ptr())
        return out

    def raster(self, width, height, v_min, v_max, saturation=0):
        """-> (counts int32-viewed uint32 tensor [height, width], rgba uint8 tensor [height, width, 4] or None);
        device tensors owned by the caller, written on this ensemble's stream."""
        torch = self._torch
        with torch.cuda.stream(self.stream):
            counts = torch.empty((height, width), dtype=torch.int32, device="cuda")
            rgba = torch.empty((height, width, 4), dtype=torch.uint8, device="cuda") if saturation else None
        abm_raster(self.ctx, counts.data_ptr(), width, height, v_min, v_max,
                   rgba.data_ptr() if rgba is not None else None, saturation or 1)
        return counts, rgba

    def time_averaged_velocity(self):
        return abm_time_averaged_velocity(self.ctx, self.n_sets)

    def state(self):
        """Current (x, v, e) of all trajectories as a float64 numpy array [n_traj, 3] (host)."""
        cols, item = 4, (8 if self.fp64 else 4)
        host = np.empty((self.n_traj, cols), np.float64 if self.fp64 else np.float32)
        abm_snapshot_host(self.ctx, host, cols * item)
        return host[:, :3].astype(np.float64)

    @property
    def accuracy(self):
        return abm_get_accuracy(self.ctx) & 0xff

    @property
    def beyond_tolerance(self):
        return bool(abm_get_accuracy(self.ctx) & ABM_ACCURACY_BEYOND_TOLERANCE)

    @property
    def step_count(self):
        return abm_get_step(self.ctx)

    def close(self):
        if self.ctx is not None:
            abm_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
