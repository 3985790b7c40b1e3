"""Sharding one ensemble over several GPUs -- host logic only.

Trajectories are independent and the random stream depends only on the GLOBAL
trajectory index, so a shard is just an index range: no collective runs during integration.  The
one exchange is the sum of the per-set raw moment sums (8 doubles per set), after which every
rank finalises the same `abm_moment` records with `abm_moments_from_sums`.

    plan = shard_plan(n_particles, n_param_sets, rank, world, scaling="strong")
    ens  = Ensemble(sets[plan.set_first:plan.set_first + plan.n_sets], plan.n_particles, seed,
                    traj_base=plan.traj_base, traj_set_stride=plan.traj_set_stride)
    ...
    m = reduce_moments(ens.moment_sums(), ens.step_count, plan)     # identical on every rank

or, without any host round trip between the reduction kernel and the collective (NCCL):

    ex = MomentExchange(plan, n_slots=20)                           # device + pinned host buffers
    for j in range(20):
        ens.step(1000); ex.enqueue(ens, j)                          # reduction, all-reduce, async copy: no wait
    ens.stream.synchronize()
    m = [ex.result(j) for j in range(20)]
"""
from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class ShardPlan:
    rank: int
    world: int
    scaling: str           # "weak" | "strong"
    split: str             # "replica" | "sets" | "particles"
    n_particles: int       # per set, on this rank
    set_first: int         # first parameter set of this rank
    n_sets: int            # parameter sets on this rank
    n_sets_total: int
    traj_base: int         # abm_params.traj_base of this rank's context
    traj_set_stride: int   # abm_params.traj_set_stride (0 = n_particles)

    def global_indices(self) -> np.ndarray:
        """Global stream indices of this shard in local order k = set * n_particles + r."""
        stride = self.traj_set_stride or self.n_particles
        s = np.arange(self.n_sets, dtype=np.uint64)[:, None]
        r = np.arange(self.n_particles, dtype=np.uint64)[None, :]
        return (np.uint64(self.traj_base) + s * np.uint64(stride) + r).reshape(-1)


def _split(n: int, rank: int, world: int):
    """Contiguous near-equal split of range(n): (first, count); the first n % world ranks get one more."""
    base, rem = divmod(n, world)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def shard_plan(n_particles: int, n_param_sets: int, rank: int, world: int,
               scaling: str = "strong") -> ShardPlan:
    """Index range of `rank`.

    weak:    every rank integrates a full copy of the workload on its own indices
             [rank * T, (rank + 1) * T), T = n_particles * n_param_sets: the job is a `world` times
             larger ensemble with `world * n_particles` realisations per set.
    strong:  the ensemble is divided.  With at least `world` parameter sets, whole sets go to a
             rank (its moments are final without any exchange, only gathered); otherwise the
             realisations of every set are divided and the raw sums are all-reduced.
    """
    if not (0 <= rank < world) or n_particles <= 0 or n_param_sets <= 0:
        raise ValueError("bad shard request")
    T = n_particles * n_param_sets
    if scaling == "weak":
        return ShardPlan(rank, world, scaling, "replica", n_particles, 0, n_param_sets, n_param_sets,
                         rank * T, 0)
    if scaling != "strong":
        raise ValueError("scaling must be 'weak' or 'strong'")
    if n_param_sets >= world:
        first, count = _split(n_param_sets, rank, world)
        return ShardPlan(rank, world, scaling, "sets", n_particles, first, count, n_param_sets,
                         first * n_particles, 0)
    first, count = _split(n_particles, rank, world)
    if count == 0:
        raise ValueError("more ranks than realisations")
    return ShardPlan(rank, world, scaling, "particles", count, 0, n_param_sets, n_param_sets,
                     first, n_particles)


def reduce_moment_sums(sums: np.ndarray, plan: ShardPlan, group=None, device=None) -> np.ndarray:
    """All ranks' raw sums [n_sets_local, 8] -> the job's raw sums [n_sets_total, 8] on every rank.

    "replica" / "particles": element-wise sum (one all-reduce).  "sets": the ranks own disjoint sets;
    their rows are placed into a zero matrix and summed (same collective, no special casing).
    world == 1 returns the input.  `device`: where the collective's tensor lives ("cuda" for NCCL).
    """
    sums = np.ascontiguousarray(sums, np.float64)
    if plan.world == 1:
        return sums
    import torch
    import torch.distributed as dist
    full = np.zeros((plan.n_sets_total, sums.shape[1]), np.float64)
    full[plan.set_first:plan.set_first + plan.n_sets] = sums
    t = torch.from_numpy(full)
    if device is not None:
        t = t.to(device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return t.cpu().numpy()


def reduce_moments(sums: np.ndarray, step: int, plan: ShardPlan, group=None, device=None):
    """Raw sums of this rank -> finalised moments of the whole job (abm_moment records)."""
    from . import binding
    return binding.abm_moments_from_sums(reduce_moment_sums(sums, plan, group, device), step)


class MomentExchange:
    """The exchange of the sharded path kept on the device: `abm_moment_sums_dev` writes this
    rank's raw sums into its rows of a [n_sets_total, 8] float64 CUDA tensor, one `all_reduce` (NCCL over
    NVLink) sums the tensor in place across ranks, and an asynchronous copy brings it to pinned host memory --
    nothing waits, so moments every M steps do not stall the integration.
    `result(slot)` finalises on the host (`abm_moments_from_sums`) after the caller has synchronised.

    Stream order: the library enqueues the reduction on the ensemble's stream (`ens.stream`, the one its context
    was created with), so `enqueue` issues every torch operation -- the zero fill, the collective, the copy to
    the host -- on THAT stream as well, whatever torch's current stream is at the call.  The buffers are
    zero-filled at construction on the then-current stream, which the constructor waits for.  Synchronise
    `ens.stream` before `result`.

    backend gloo (rehearsal with ranks sharing one GPU; gloo reduces host tensors): the sums take a synchronous
    detour through the host, everything else is the same code.  world == 1 skips the collective unless
    `always_collective` is set (a one-rank NCCL group is legal and exercises the very calls of the N-rank job).
    """

    def __init__(self, plan: ShardPlan, n_slots: int = 1, group=None, backend: str = "nccl",
                 always_collective: bool = False):
        import torch
        self._torch, self.plan, self.group, self.backend = torch, plan, group, backend
        self.collective = plan.world > 1 or always_collective
        shape = (n_slots, plan.n_sets_total, 8)
        self.dev = torch.zeros(shape, dtype=torch.float64, device="cuda")
        self.host = torch.zeros(shape, dtype=torch.float64, pin_memory=True)
        torch.cuda.current_stream().synchronize()   # the fills are done before any other stream touches the buffers
        self.steps = [0] * n_slots

    def enqueue(self, ens, slot: int):
        torch, plan = self._torch, self.plan
        buf = self.dev[slot]
        with torch.cuda.stream(ens.stream):        # the stream abm_moment_sums_dev enqueues on
            if plan.split == "sets" and self.collective:
                buf.zero_()                       # rows of the other ranks' sets: filled by the all-reduce
            rows = buf[plan.set_first:plan.set_first + plan.n_sets]
            ens.moment_sums_dev(rows)
            self.steps[slot] = ens.step_count
            if self.collective:
                import torch.distributed as dist
                if self.backend == "nccl":
                    dist.all_reduce(buf, op=dist.ReduceOp.SUM, group=self.group)
                else:
                    t = buf.cpu()
                    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=self.group)
                    buf.copy_(t)
            self.host[slot].copy_(buf, non_blocking=True)

    def result(self, slot: int):
        """Finalised moments of the whole job (valid once the ensemble's stream has been synchronised)."""
        from . import binding
        return binding.abm_moments_from_sums(self.host[slot].numpy(), self.steps[slot])
