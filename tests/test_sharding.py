"""Multi-GPU host logic on the CPU: shard plans, and the one exchange of the
path -- the all-reduce of the per-set raw moment sums -- with two `gloo` ranks.

No GPU here: each rank's shard is integrated by the CPU oracle (the tests may use it) on exactly the
global trajectory indices the plan gives the rank's context; the raw sums are then combined by the product's
`sharding.reduce_moments` (torch.distributed + the C ABI's host-side `abm_moments_from_sums`) and compared
with the oracle's moments of the undivided ensemble.
"""
import os
import socket

import numpy as np
import pytest

from paper_1104_2499_b200 import sharding, workloads as W


# ---- shard plans -------------------------------------------------------------------------------

@pytest.mark.parametrize("n_particles,n_sets,world", [(4096, 1, 2), (1000, 1, 3), (64, 65536, 8), (64, 7, 4),
                                                      (5, 2, 4), (1, 3, 2)])
def test_strong_plans_partition_the_ensemble(n_particles, n_sets, world):
    whole = sharding.shard_plan(n_particles, n_sets, 0, 1, "strong").global_indices()
    assert np.array_equal(whole, np.arange(n_particles * n_sets, dtype=np.uint64))
    parts = [sharding.shard_plan(n_particles, n_sets, r, world, "strong") for r in range(world)]
    got = np.concatenate([p.global_indices() for p in parts])
    assert got.size == whole.size and np.array_equal(np.sort(got), whole)      # disjoint cover
    if n_sets >= world:
        assert all(p.split == "sets" and p.n_particles == n_particles for p in parts)
        assert sum(p.n_sets for p in parts) == n_sets
    else:
        assert all(p.split == "particles" and p.n_sets == n_sets for p in parts)
        assert sum(p.n_particles for p in parts) == n_particles
        # a trajectory keeps its global index: set s, realisation r -> s * n_particles + r
        p = parts[-1]
        assert p.traj_set_stride == n_particles and p.global_indices()[0] == p.traj_base


def test_weak_plans_are_disjoint_replicas():
    parts = [sharding.shard_plan(64, 10, r, 4, "weak") for r in range(4)]
    got = np.concatenate([p.global_indices() for p in parts])
    assert np.array_equal(got, np.arange(4 * 640, dtype=np.uint64))
    assert all(p.n_sets == 10 and p.n_particles == 64 for p in parts)


def test_bad_requests():
    with pytest.raises(ValueError):
        sharding.shard_plan(10, 1, 2, 2)
    with pytest.raises(ValueError):
        sharding.shard_plan(1, 1, 1, 2, "strong")       # rank 1 would be empty
    with pytest.raises(ValueError):
        sharding.shard_plan(10, 1, 0, 2, "diagonal")


# ---- two gloo ranks ----------------------------------------------------------------------------

def _raw_sums(x, v, e, x0):
    dx = x - x0
    return np.array([x.size, x.sum(), (x * x).sum(), v.sum(), (v * v).sum(), e.sum(), dx.sum(), (dx * dx).sum()])


def _integrate_shard(plan, sets, seed, n_steps):
    """Oracle stand-in for one rank's device context: raw sums [n_sets_local, 8] of its shard."""
    from oracle import abm_oracle as orc
    stride = plan.traj_set_stride or plan.n_particles
    out = np.zeros((plan.n_sets, 8))
    for j in range(plan.n_sets):
        p = sets[plan.set_first + j]
        first = plan.traj_base + j * stride
        x, v, e = orc.init_many(p, seed, plan.n_particles, first)
        x0 = x.copy()
        orc.run(p, seed, x, v, e, 0, n_steps, first)
        out[j] = _raw_sums(x, v, e, x0)
    return out


def _rank_main(rank, world, port, case, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n_particles, sets, seed, n_steps, scaling = case
        plan = sharding.shard_plan(n_particles, len(sets), rank, world, scaling)
        sums = _integrate_shard(plan, sets, seed, n_steps)
        m = sharding.reduce_moments(sums, n_steps, plan)
        q.put((rank, plan.split, m.tobytes()))
    finally:
        dist.destroy_process_group()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _cases():
    wl = W.config2(n_D=2, n_q=3, realisations=40, n_steps=50)          # 6 sets >= 2 ranks -> split by sets
    sweep = [wl.set_params(s) for s in range(wl.n_param_sets)]
    one = [W.config0().set_params(0)]
    return {
        "strong_particles": (301, one, 42, 60, "strong"),               # ragged split 151 + 150
        "strong_sets": (40, sweep, 1234, 50, "strong"),
        "weak_replicas": (128, one, 7, 40, "weak"),
    }


@pytest.mark.parametrize("name", list(_cases()))
def test_two_gloo_ranks_reduce_to_the_undivided_ensemble(name, oracle):
    import torch.multiprocessing as mp
    from paper_1104_2499_b200 import binding
    case = _cases()[name]
    n_particles, sets, seed, n_steps, scaling = case
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_main, args=(r, world, port, case, q)) for r in range(world)]
    for p in procs:
        p.start()
    results = [q.get(timeout=180) for _ in range(world)]
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    got = {r: np.frombuffer(b, binding.MOMENT_DTYPE) for r, _, b in results}
    assert got[0].tobytes() == got[1].tobytes()                         # every rank holds the job's moments
    m = got[0]
    # the undivided ensemble, one process
    n_tot = n_particles * (world if scaling == "weak" else 1)
    assert m.shape[0] == len(sets)
    for s, p in enumerate(sets):
        first = s * n_particles if scaling == "strong" else 0
        if scaling == "weak":
            assert len(sets) == 1
        x, v, e = oracle.init_many(p, seed, n_tot, first)
        x0 = x.copy()
        oracle.run(p, seed, x, v, e, 0, n_steps, first)
        want = oracle.moments(x, v, e, x0)
        assert int(m[s]["n"]) == n_tot and int(m[s]["step"]) == n_steps
        for k, val in want.items():
            assert abs(m[s][k] - val) <= 1e-12 * max(1.0, abs(val)), (name, s, k, m[s][k], val)


# ---- the device-side exchange (MomentExchange) with two ranks on the GPU box -----------------------

def _gpu_rank_main(rank, world, port, case, q):
    import torch
    import torch.distributed as dist
    from paper_1104_2499_b200 import binding as abm
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)      # one GPU on the box: the ranks share it
    try:
        torch.cuda.set_device(0)
        n_particles, sets, seed, chunks, scaling = case
        plan = sharding.shard_plan(n_particles, len(sets), rank, world, scaling)
        ex = sharding.MomentExchange(plan, n_slots=len(chunks), backend="gloo")
        mine = sets[plan.set_first:plan.set_first + plan.n_sets]
        with abm.Ensemble(mine, plan.n_particles, seed, traj_base=plan.traj_base,
                          traj_set_stride=plan.traj_set_stride) as ens:
            for j, n in enumerate(chunks):
                ens.step(n)
                ex.enqueue(ens, j)                                     # nothing waits here
            torch.cuda.current_stream().synchronize()
        q.put((rank, [ex.result(j).tobytes() for j in range(len(chunks))]))
    finally:
        dist.destroy_process_group()


@pytest.mark.gpu
@pytest.mark.parametrize("name", ["strong_particles", "strong_sets", "weak_replicas"])
def test_two_ranks_device_side_exchange_equals_one_context(name):
    """The sharded job's moments (two contexts on disjoint index ranges, sums exchanged by MomentExchange) against
    ONE context holding the whole ensemble: same trajectories bit for bit, so the moments agree to the rounding
    of the differently ordered fp64 sums."""
    import torch
    import torch.multiprocessing as mp
    from paper_1104_2499_b200 import binding as abm
    assert torch.cuda.is_available()
    n_particles, sets, seed, n_steps, scaling = _cases()[name]
    chunks = [n_steps // 2, n_steps - n_steps // 2]
    case = (n_particles, sets, seed, chunks, scaling)
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_gpu_rank_main, args=(r, world, port, case, q)) for r in range(world)]
    for p in procs:
        p.start()
    results = dict(q.get(timeout=300) for _ in range(world))
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert results[0] == results[1]                                    # every rank holds the job's moments
    n_tot = n_particles * (world if scaling == "weak" else 1)
    with abm.Ensemble(sets, n_tot, seed) as whole:
        for j, n in enumerate(chunks):
            whole.step(n)
            want = whole.moments()
            got = np.frombuffer(results[0][j], abm.MOMENT_DTYPE)
            assert np.array_equal(got["n"], want["n"]) and np.array_equal(got["step"], want["step"])
            for k in ("mean_x", "var_x", "mean_v", "var_v", "mean_e", "mean_dx", "mean_dx2", "mean_x2"):
                assert np.allclose(got[k], want[k], rtol=1e-12, atol=1e-13), (name, j, k)


# ---- MomentExchange on a stream that is not torch's current one ---------------------------

@pytest.mark.gpu
@pytest.mark.parametrize("scaling", ["weak", "strong"])
def test_exchange_is_ordered_on_the_ensembles_own_stream(scaling):
    """The context enqueues its reduction on the stream it was created with; MomentExchange must put its own
    torch operations (zero fill, copy to the host) on that same stream even when the caller's current stream is
    another one.  The default stream is kept busy meanwhile, so work wrongly issued there would run late."""
    import torch
    from paper_1104_2499_b200 import binding as abm
    wl = W.config2()
    sets = [wl.set_params(s) for s in range(0, wl.n_param_sets, wl.n_param_sets // 37)]
    chunks = [40, 24, 36, 8]
    side = torch.cuda.Stream()
    plan = sharding.shard_plan(200, len(sets), 0, 1, scaling)
    ex = sharding.MomentExchange(plan, n_slots=len(chunks), always_collective=False)
    ballast = torch.empty(1 << 28, dtype=torch.float32, device="cuda")     # 1 GiB fills on the default stream
    with abm.Ensemble(sets, 200, wl.seed, stream=side) as ens:
        assert torch.cuda.current_stream() != side
        for j, n in enumerate(chunks):
            ballast.fill_(float(j))
            ens.step(n)
            ex.enqueue(ens, j)                                             # called OUTSIDE any stream block
        ens.stream.synchronize()
        got = [ex.result(j) for j in range(len(chunks))]
    torch.cuda.synchronize()
    with abm.Ensemble(sets, 200, wl.seed) as twin:                          # same trajectories, waiting calls
        for j, n in enumerate(chunks):
            twin.step(n)
            assert got[j].tobytes() == twin.moments().tobytes(), j


# ---- the NCCL calls of the N-rank job, executed with a one-rank group on the box's one GPU -------------

def _nccl_one_rank_main(port, q):
    import torch
    import torch.distributed as dist
    from paper_1104_2499_b200 import binding as abm
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        wl = W.config2()
        sets = [wl.set_params(s) for s in range(0, wl.n_param_sets, wl.n_param_sets // 19)]
        chunks = [20, 12, 40]
        out = {}
        for scaling in ("weak", "strong"):                                # "replica" and "sets" splits
            plan = sharding.shard_plan(128, len(sets), 0, 1, scaling)
            ex = sharding.MomentExchange(plan, n_slots=len(chunks), backend="nccl", always_collective=True)
            side = torch.cuda.Stream()
            with abm.Ensemble(sets, 128, wl.seed, stream=side) as ens:
                for j, n in enumerate(chunks):
                    ens.step(n)
                    ex.enqueue(ens, j)                                     # abm_moment_sums_dev -> ncclAllReduce -> D2H
                ens.stream.synchronize()
                got = [ex.result(j).tobytes() for j in range(len(chunks))]
            with abm.Ensemble(sets, 128, wl.seed) as twin:
                want = []
                for n in chunks:
                    twin.step(n)
                    want.append(twin.moments().tobytes())
            out[scaling] = (got == want)
        q.put(("ok", out, dist.get_backend(), dist.get_world_size()))
    except Exception as exc:                                               # report instead of hanging the parent
        q.put(("error", repr(exc), None, None))
    finally:
        dist.destroy_process_group()


@pytest.mark.gpu
def test_nccl_branch_runs_with_a_one_rank_group():
    """`dist.init_process_group("nccl", device_id=...)` and the in-place all-reduce of the CUDA tensor between
    `abm_step` calls -- the branch bench.py takes under torchrun -- executed for real: a one-rank NCCL
    communicator on cuda:0.  The sum over one rank is the identity, so the moments equal abm_moments bit for bit."""
    import torch
    import torch.multiprocessing as mp
    assert torch.cuda.is_available()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    p = ctx.Process(target=_nccl_one_rank_main, args=(_free_port(), q))
    p.start()
    status, out, backend, world = q.get(timeout=300)
    p.join(60)
    assert status == "ok", out
    assert p.exitcode == 0
    assert backend == "nccl" and world == 1
    assert out == {"weak": True, "strong": True}
