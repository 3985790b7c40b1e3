"""Host-side checks of the C-ABI boundary (no GPU): the library builds, loads, exports every
function include/abm.h declares, the ctypes mirrors match the C layout, and the error paths
answer as documented.  No kernel is launched here."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "abm.h")


@pytest.fixture(scope="module")
def abm():
    from paper_1104_2499_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(abm_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(abm):
    names = _declared_functions()
    assert set(names) == set(abm.EXPORTS), (names, abm.EXPORTS)
    L = abm.lib()
    for n in names:
        assert getattr(L, n) is not None
    assert L.abm_abi_version() == 6


def test_header_is_plain_c_and_layout_matches_ctypes(abm, tmp_path):
    """Compile a C99 probe against include/abm.h with gcc: the header must be usable from C, and
    sizeof/offsetof must agree with the ctypes mirrors the tests and bench use."""
    fields = [f[0] for f in abm.abm_params._fields_]
    mfields = [f[0] for f in abm.abm_moment._fields_]
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "abm.h"', 'int main(void){',
             'printf("%zu\\n", sizeof(abm_params));', 'printf("%zu\\n", sizeof(abm_moment));']
    lines += [f'printf("%zu\\n", offsetof(abm_params, {f}));' for f in fields]
    lines += [f'printf("%zu\\n", offsetof(abm_moment, {f}));' for f in mfields]
    lines += ['return 0;}']
    src = tmp_path / "probe.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "probe"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"),
                    "-o", str(exe), str(src)], check=True)
    vals = [int(v) for v in subprocess.run([str(exe)], check=True, capture_output=True,
                                           text=True).stdout.split()]
    assert vals[0] == C.sizeof(abm.abm_params)
    assert vals[1] == C.sizeof(abm.abm_moment) == 80 == abm.MOMENT_DTYPE.itemsize
    want = [getattr(abm.abm_params, f).offset for f in fields] + \
           [getattr(abm.abm_moment, f).offset for f in mfields]
    assert vals[2:] == want


def test_error_paths_without_device(abm):
    L = abm.lib()
    h = C.c_void_p()
    from paper_1104_2499_b200 import workloads as W
    good = abm.make_params([W.config0().set_params(0)])
    # argument validation comes first and needs no device
    assert L.abm_create(None, 16, 1, 1, C.byref(h)) == abm.ABM_EINVAL
    assert L.abm_create(good, 0, 1, 1, C.byref(h)) == abm.ABM_EINVAL
    assert L.abm_create(good, 16, 0, 1, C.byref(h)) == abm.ABM_EINVAL
    assert L.abm_create(good, 16, 1, 1, None) == abm.ABM_EINVAL
    bad = abm.make_params([W.config0().set_params(0)])
    bad[0].struct_size = 8
    assert L.abm_create(bad, 16, 1, 1, C.byref(h)) == abm.ABM_EINVAL
    for key, val in [("dt", 0.0), ("dt", float("nan")), ("L", -1.0), ("D", -0.1), ("precision", 7),
                     ("integrator", 2), ("step_kernel", 3), ("rng", 2), ("accuracy", 3)]:
        bad = abm.make_params([dict(W.config0().set_params(0), **{key: val})])
        assert L.abm_create(bad, 16, 1, 1, C.byref(h)) == abm.ABM_EINVAL, key
    # run-control fields must agree between sets
    two = abm.make_params([W.config0().set_params(0), dict(W.config0().set_params(0), dt=2e-3)])
    assert L.abm_create(two, 16, 2, 1, C.byref(h)) == abm.ABM_EINVAL
    assert h.value is None                                  # *out untouched on error
    # the global trajectory index range must not wrap 2^64 (it keys the Philox counter)
    one = W.config0().set_params(0)
    wrap = abm.make_params([one], traj_base=2**64 - 10)
    assert L.abm_create(wrap, 16, 1, 1, C.byref(h)) == abm.ABM_EINVAL
    wrap3 = abm.make_params([one] * 3, traj_set_stride=2**63)
    assert L.abm_create(wrap3, 16, 3, 1, C.byref(h)) == abm.ABM_EINVAL
    fits = abm.make_params([one], traj_base=2**64 - 16)      # last index = 2^64 - 1: legal
    rc = L.abm_create(fits, 16, 1, 1, C.byref(h))
    assert rc in (abm.ABM_OK, abm.ABM_ECUDA)                # ECUDA: no device on this box
    if rc == abm.ABM_OK:
        assert L.abm_destroy(h) == abm.ABM_OK
        h = C.c_void_p()
    junk = (C.c_char * 4096)()                              # an address that never was a context
    assert L.abm_destroy(C.addressof(junk)) == abm.ABM_ESTATE
    assert L.abm_step(C.addressof(junk), 1) == abm.ABM_ESTATE
    assert L.abm_moment_sums_dev(None, None) == abm.ABM_ESTATE
    assert L.abm_philox_blocks_loop(1, 0, 1, 0, 1, 2, 0, None, None) == abm.ABM_EINVAL
    # null / never-created contexts
    assert L.abm_step(None, 1) == abm.ABM_ESTATE
    assert L.abm_destroy(None) == abm.ABM_ESTATE
    assert L.abm_moments(None, None) == abm.ABM_ESTATE
    assert L.abm_moments_async(None, None) == abm.ABM_ESTATE
    assert L.abm_snapshot(None, None, 8) == abm.ABM_ESTATE
    assert L.abm_philox_blocks(1, 0, 0, 0, 1, None, None) == abm.ABM_EINVAL
    for code in (0, -1, -2, -3, -4, -99):
        assert len(L.abm_strerror(code)) > 0


def test_no_cpu_fallback(abm):
    """On a box without a CUDA device a valid abm_create must fail loudly (ABM_ECUDA), never
    compute on the host."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present; the GPU tests cover the success path")
    from paper_1104_2499_b200 import workloads as W
    good = abm.make_params([W.config0().set_params(0)])
    h = C.c_void_p()
    assert abm.lib().abm_create(good, 16, 1, 1, C.byref(h)) == abm.ABM_ECUDA
    with pytest.raises(abm.AbmError):
        abm.abm_create(good, 16, 1, 1)
    with pytest.raises(RuntimeError):
        abm.Ensemble([W.config0().set_params(0)], 16, 1)


def test_moments_from_sums_matches_numpy(abm):
    """abm_moments_from_sums is pure host arithmetic (the shard-combination step)."""
    rng = np.random.default_rng(3)
    x, v, e, x0 = rng.normal(2, 3, 500), rng.normal(0, 1, 500), rng.uniform(0, 2, 500), rng.uniform(0, 1, 500)
    dx = x - x0
    sums = np.array([[x.size, x.sum(), (x * x).sum(), v.sum(), (v * v).sum(), e.sum(), dx.sum(),
                      (dx * dx).sum()]])
    m = abm.abm_moments_from_sums(sums, 77)[0]
    assert m["n"] == 500 and m["step"] == 77
    assert m["mean_x"] == pytest.approx(x.mean(), rel=1e-12)
    assert m["var_x"] == pytest.approx(x.var(), rel=1e-10)
    assert m["mean_v"] == pytest.approx(v.mean(), rel=1e-10, abs=1e-14)
    assert m["var_v"] == pytest.approx(v.var(), rel=1e-10)
    assert m["mean_e"] == pytest.approx(e.mean(), rel=1e-12)
    assert m["mean_dx"] == pytest.approx(dx.mean(), rel=1e-12)
    assert m["mean_dx2"] == pytest.approx((dx * dx).mean(), rel=1e-12)
    assert m["mean_x2"] == pytest.approx((x * x).mean(), rel=1e-12)
    with pytest.raises(abm.AbmError):
        abm.abm_moments_from_sums(np.zeros((1, 8)), 0)


def test_library_reads_no_environment_variable():
    """The kernel choice is a field of abm_params (step_kernel), not an environment variable."""
    src = open(os.path.join(ROOT, "paper_1104_2499_b200", "csrc", "abm.cu")).read()
    assert "getenv" not in src


def test_product_never_imports_oracle():
    """The oracle is test infrastructure: nothing under the package may import or load it."""
    pkg = os.path.join(ROOT, "paper_1104_2499_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"import\s+oracle|from\s+oracle|abm_oracle|abo_", txt), (dirpath, f)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_1104_2499_b200", txt, flags=re.M)
            assert '#include "abm.h"' not in txt and "abm_device" not in txt


def _build_c_demo(tmp_path):
    exe = tmp_path / "abm_demo"
    pkg = os.path.join(ROOT, "paper_1104_2499_b200")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-o", str(exe),
                    os.path.join(pkg, "examples", "abm_demo.c"), "-L", pkg, "-labm_b200",
                    "-Wl,-rpath," + pkg], check=True)
    return exe


def test_plain_c_caller_links_and_fails_loudly_without_a_device(abm, tmp_path):
    """The boundary is a C library: a C99 program with no CUDA headers links against it.  Without a
    device it must report ABM_ECUDA (exit code 3 of the demo), never compute on the CPU."""
    import torch
    exe = _build_c_demo(tmp_path)
    r = subprocess.run([str(exe), "8", "4"], capture_output=True, text=True)
    if torch.cuda.is_available():
        assert r.returncode == 0, r.stderr
    else:
        assert r.returncode == 3 and "abm_create: -3" in r.stderr, (r.returncode, r.stderr)


@pytest.mark.gpu
def test_plain_c_caller_matches_the_oracle(abm, tmp_path):
    """The same program on the GPU box: its printed state and moments against the CPU oracle."""
    import numpy as np
    from paper_1104_2499_b200 import workloads as W
    from oracle import abm_oracle as orc
    exe = _build_c_demo(tmp_path)
    n, steps = 300, 100
    r = subprocess.run([str(exe), str(n), str(steps)], capture_output=True, text=True, check=True)
    lines = r.stdout.strip().splitlines()
    got = np.array([[float(t) for t in ln.split()[2:5]] for ln in lines[1:]])
    assert got.shape == (n, 3)
    p = W.config0().set_params(0)
    x, v, e = orc.init_many(p, 42, n)
    orc.run(p, 42, x, v, e, 0, steps)
    want = np.stack([x, v, e], 1)
    rms = np.sqrt((want**2).mean(0))
    assert np.all(np.abs(got - want) / np.maximum(np.abs(want), rms) <= 1e-5)
    mom = dict(zip(lines[0].split()[1::2], lines[0].split()[2::2]))
    assert int(mom["n"]) == n and int(mom["step"]) == steps
    assert abs(float(mom["mean_v"]) - got[:, 1].mean()) <= 1e-6
