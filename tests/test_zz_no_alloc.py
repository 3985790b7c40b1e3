"""abm_frame_moment_sums_static: the moment sums for callers that cannot allocate device memory.

Some users of this library may not call cudaMalloc where they need the moments: a host program that owns
every device allocation itself and gives libraries no budget of their own (the frame sits in ITS tensor),
a service that has claimed the whole GPU at start-up, a latency-critical loop in which allocator calls --
they may lock the driver and synchronise the device -- are banned once it runs.  For them the library has
one entry point whose only scratch is a fixed array built into the library image.  This file checks it
against the ordinary, context-owned reduction (abm_moment_sums_dev): same state in, the same eight sums
out -- bit for bit, since both add in the same order -- on two calls in a row, because the array is
shared by all calls and keeps the previous call's contents.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  It has to pass alone in a fresh process (then its first call does the per-GPU address
look-up) as well as after all other tests.
"""
import ctypes as C

import numpy as np
import pytest

from paper_1104_2499_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def abm():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1104_2499_b200 import binding
    binding.lib()
    return binding


def _frames_and_reference(abm, torch, ens, with_e, steps):
    """Step `ens`; return (frame at step 0, frame now, sums of the context-owned reduction) -- all on the device."""
    cols = 4 if with_e else 2
    frame = ens.bind_snapshot(with_e=with_e)            # caller-owned tensor, written now (step 0)
    frame0 = frame.clone()
    ens.unbind_snapshot()
    ens.step(steps)
    abm.abm_snapshot(ens.ctx, frame.data_ptr(), cols * frame.element_size())
    ens.unbind_snapshot()
    ref = torch.empty((ens.n_sets, abm.ABM_N_SUMS), dtype=torch.float64, device="cuda")
    ens.moment_sums_dev(ref)
    return frame0, frame, ref


CASES = [
    # id, workload, n_particles, n_sets, steps, with_e
    ("cfg0_f32_one_set_ragged", "config0", 4096 * 3 + 77, None, 40, True),     # 4 slices, the last one ragged
    ("cfg2_f32_sweep_64_per_set", "config2", 64, 300, 24, True),               # one short CTA per set
    ("cfg3_f32_heun_precise_xv", "config3", 9000, None, 16, False),            # (x, v) frames: no e column
    ("cfg4_f64", "config4", 5000, None, 12, True),
]


@pytest.mark.parametrize("name,cfg,n_particles,n_sets,steps,with_e", CASES, ids=[c[0] for c in CASES])
def test_static_scratch_sums_equal_the_context_reduction_twice(abm, name, cfg, n_particles, n_sets, steps, with_e):
    import torch
    wl = getattr(W, cfg)()
    sets = range(wl.n_param_sets) if n_sets is None else np.linspace(0, wl.n_param_sets - 1, n_sets).astype(int)
    params = [wl.set_params(int(s)) for s in sets]
    stream = torch.cuda.current_stream().cuda_stream
    with abm.Ensemble(params, n_particles, wl.seed) as ens:
        precision = abm.ABM_FP64 if ens.fp64 else abm.ABM_FP32
        frame0, frame, ref = _frames_and_reference(abm, torch, ens, with_e, steps)
        stride = frame.shape[1] * frame.element_size()
        out = torch.full((ens.n_sets, abm.ABM_N_SUMS), float("nan"), dtype=torch.float64, device="cuda")
        # call 1
        abm.abm_frame_moment_sums_static(frame.data_ptr(), frame0.data_ptr(), stride, precision, n_particles,
                                         ens.n_sets, out.data_ptr(), stream)
        got1 = out.cpu().numpy()
        want1 = ref.cpu().numpy()
        if not with_e:
            want1[:, 5] = 0.0                            # the short frame has no e column: sum e is defined as 0
        assert np.array_equal(got1, want1), np.abs(got1 - want1).max()
        # a different, LARGER job in between leaves its records in the shared array ...
        junk = torch.randn((70_000, frame.shape[1]), dtype=frame.dtype, device="cuda")
        junk_out = torch.empty((1, abm.ABM_N_SUMS), dtype=torch.float64, device="cuda")
        abm.abm_frame_moment_sums_static(junk.data_ptr(), None, stride, precision, 70_000, 1, junk_out.data_ptr(),
                                         stream)
        j = junk_out.cpu().numpy()[0]
        jd = junk.double()
        assert j[0] == 70_000 and j[6] == 0.0 and j[7] == 0.0          # no step-0 frame: dx sums are 0
        np.testing.assert_allclose(j[1:5], [jd[:, 0].sum().item(), (jd[:, 0] ** 2).sum().item(),
                                            jd[:, 1].sum().item(), (jd[:, 1] ** 2).sum().item()],
                                   rtol=1e-12, atol=1e-9)
        # ... and call 2, after more steps, must again equal the context's own reduction
        ens.step(steps + 4)
        abm.abm_snapshot(ens.ctx, frame.data_ptr(), stride)
        ens.unbind_snapshot()
        ens.moment_sums_dev(ref)
        out.fill_(float("nan"))
        abm.abm_frame_moment_sums_static(frame.data_ptr(), frame0.data_ptr(), stride, precision, n_particles,
                                         ens.n_sets, out.data_ptr(), stream)
        got2 = out.cpu().numpy()
        want2 = ref.cpu().numpy()
        if not with_e:
            want2[:, 5] = 0.0
        assert np.array_equal(got2, want2), np.abs(got2 - want2).max()
        assert not np.array_equal(got1, got2)            # the state did move between the calls
        # the host-side finalisation of these sums is the record abm_moments gives
        m = abm.abm_moments_from_sums(got2, ens.step_count)
        rec = ens.moments()
        for f in ("n", "step", "mean_x", "var_x", "mean_v", "var_v", "mean_dx", "mean_dx2", "mean_x2") + \
                 (("mean_e",) if with_e else ()):
            assert np.array_equal(m[f], rec[f]), f


def test_static_scratch_allocates_nothing(abm):
    """Device memory in use does not change over calls of the entry point (the first call on this GPU
    included when this file runs alone), and torch's allocator is not asked for anything either."""
    import torch
    n = 100_000
    frame = torch.randn((n, 4), dtype=torch.float32, device="cuda")
    out = torch.empty((1, abm.ABM_N_SUMS), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    reserved_before = torch.cuda.memory_reserved()
    for _ in range(3):
        abm.abm_frame_moment_sums_static(frame.data_ptr(), None, 16, abm.ABM_FP32, n, 1, out.data_ptr(), stream)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert torch.cuda.memory_reserved() == reserved_before
    assert free_after == free_before, (free_before, free_after)
    got = out.cpu().numpy()[0]
    fd = frame.double()
    np.testing.assert_allclose(got[:6], [n, fd[:, 0].sum().item(), (fd[:, 0] ** 2).sum().item(), fd[:, 1].sum().item(),
                                         (fd[:, 1] ** 2).sum().item(), fd[:, 2].sum().item()], rtol=1e-12, atol=1e-9)


def test_static_scratch_limit_and_argument_errors(abm):
    import torch
    L = abm.lib()
    buf = torch.zeros(4096, dtype=torch.float64, device="cuda")
    out = torch.zeros((4, abm.ABM_N_SUMS), dtype=torch.float64, device="cuda")
    p, o = buf.data_ptr(), out.data_ptr()
    f = L.abm_frame_moment_sums_static
    cap = abm.ABM_STATIC_MAX_SLICES
    # beyond the built-in scratch: refused before anything is read or launched (the buffers are far too small)
    assert f(p, None, 16, abm.ABM_FP32, 4096 * cap + 1, 1, o, None) == abm.ABM_ELIMIT
    assert f(p, None, 16, abm.ABM_FP32, 64, cap + 1, o, None) == abm.ABM_ELIMIT
    assert f(p, None, 32, abm.ABM_FP64, 2**60, 1, o, None) == abm.ABM_ELIMIT
    assert b"scratch" in L.abm_strerror(abm.ABM_ELIMIT)
    # argument errors
    assert f(None, None, 16, abm.ABM_FP32, 64, 1, o, None) == abm.ABM_EINVAL
    assert f(p, None, 16, abm.ABM_FP32, 64, 1, None, None) == abm.ABM_EINVAL
    assert f(p, None, 12, abm.ABM_FP32, 64, 1, o, None) == abm.ABM_EINVAL          # no such layout
    assert f(p, None, 8, abm.ABM_FP64, 64, 1, o, None) == abm.ABM_EINVAL           # fp64 frames are 16 / 32
    assert f(p + 4, None, 16, abm.ABM_FP32, 64, 1, o, None) == abm.ABM_EINVAL      # misaligned frame
    assert f(p, p + 8, 16, abm.ABM_FP32, 64, 1, o, None) == abm.ABM_EINVAL         # misaligned step-0 frame
    assert f(p, None, 16, 7, 64, 1, o, None) == abm.ABM_EINVAL
    assert f(p, None, 16, abm.ABM_FP32, 0, 1, o, None) == abm.ABM_EINVAL
    assert f(p, None, 16, abm.ABM_FP32, 64, 0, o, None) == abm.ABM_EINVAL
    # exactly at the limit of sets is accepted (65,536 sets of one trajectory each need 65,536 records)
    big = torch.ones((cap, 2), dtype=torch.float32, device="cuda")
    big_out = torch.empty((cap, abm.ABM_N_SUMS), dtype=torch.float64, device="cuda")
    assert f(big.data_ptr(), None, 8, abm.ABM_FP32, 1, cap, big_out.data_ptr(),
             C.c_void_p(torch.cuda.current_stream().cuda_stream)) == abm.ABM_OK
    got = big_out.cpu().numpy()
    assert np.array_equal(got, np.tile(np.array([1, 1, 1, 1, 1, 0, 0, 0], np.float64), (cap, 1)))
