#!/usr/bin/env python
"""bench.py -- particle-steps/s of the hot path on BASELINE.json's config[1] (default), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl ours|reference]
                    [--scaling weak|strong] [--all-configs PASSES]

One bench "step" = one pass of the whole hot path over one batch of synthetic input
(SURVEY.md 8(a) rows S0-S7): create + init the ensemble from its Philox init blocks, bind the
snapshot buffer, integrate all n_steps of the config (one frame every K_snap steps), reduce the
ensemble moments, destroy.  `value` times that on the device (CUDA events on the launching
stream, parameters already marshalled); `e2e` times the same pass by wall clock through the
C ABI from HOST parameter records to HOST results, including a device->host copy of the final
frame into pinned memory and of the moments.

N > 1: one process per GPU.  Under torchrun (WORLD_SIZE set) this process is one rank; a bare
`python bench.py --gpus N` re-executes itself under `python -m torch.distributed.run --nproc-per-node N`
(127.0.0.1 rendezvous) and fails loudly if the box has fewer than N devices.  Each rank integrates its
own shard of a N-times larger ensemble (weak scaling, the default; trajectory indices rank*T ... via
traj_base) or, with --scaling strong, its part [gT/G, (g+1)T/G) of the ONE ensemble (whole parameter sets
per rank when there are at least N, else the realisations of every set divided), and the only exchange
is one all-reduce of the per-set raw moment sums (8 doubles per set) over NCCL on the device
(sharding.MomentExchange: no host round trip), inside the timed region.

The default run (config 1, one GPU) then also times configs 0, 2, 3, 4 -- after the headline's timed regions,
same protocol, 3 passes each -- and reports them under "all_configs" (value, kernel_ms, frac, frac_executed,
e2e, clocks per config), so one driver-run line carries all five BASELINE.json configs.

Timing protocol of the paper (PAPER.md:100 "20 steps ... last fifteen", :122 "average and standard
deviation ... zero steps ... offset time"): besides the mean, the line carries the standard deviation over
the timed passes (`ms_per_step_sd`, `roofline.kernel_ms_sd`) and `offset_ms`: 20 launches of ONE step on the
same ensemble, the last 15 averaged -- what a launch costs before any iteration is done (load + store of the
state, launch latency).

--impl reference times the CPU oracle (oracle/, plain fp64 C) on a bounded sample of the same
workload on the host cores: a deliberately slow program, reported as the baseline, not the target.
"""
import argparse
import json
import os
import statistics
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1104_2499_b200 import workloads as W  # noqa: E402

# Algorithmic (necessary) warp-lane instructions per particle-step, frozen in BASELINE.md /
# DESIGN.md before tuning.
I_ALG = {0: 29.0, 1: 29.0, 2: 29.0, 3: 45.0, 4: 60.0}
N_SM, LANES_PER_SM = 148, 128
# config[4] is bound by the FP64 pipe (64 lanes/clk/SM; 59 measured for DFMA), not by issue slots: its
# I_alg counts the ~60 DFMA-pipe operations per particle-step and its peak is 64 lanes.
LANES_FP64 = 64
# What the committed `ncu --set full` captures of the launches bench.py times say about the step kernel
# (profiles/r03_step_kernels_ncu_full.md), per launch: dram__bytes_read.sum + dram__bytes_write.sum (`traffic`)
# and what the kernel EXECUTES per particle-step -- warp-lane instructions (smsp__inst_executed.sum x 32 / particle-
# steps) for the fp32 kernels, FP64-pipe lane operations (smsp__inst_executed_pipe_fp64.sum x 32 / particle-steps)
# for config[4] -- from which `roofline.frac_executed` follows: the fraction of the issue slots (or of the FP64
# pipe) the kernel keeps busy with whatever it executes, next to `frac`, which credits the frozen I_alg.
# Each entry carries the git blob ids of the two kernel sources it was captured on: when a source has changed
# since, the figures are stale and the line says null instead (re-capture, then update the entry).
# The frame (one, overwritten) and the state stay in the 126 MB L2 during a launch, so the traffic is far BELOW
# the algorithmic bytes.  Every capture is of the full launch bench.py times (config[3]: one of the 20 launches of
# 1,000 steps a pass is made of).
_SRC = dict(kernels="846dcb59299abdf7283dcc81d6fbb01e7b906435", device="41e835be8e554d8dda9c5a0b24acdd14995b1e13",
            summary="profiles/r03_step_kernels_ncu_full.md")
NCU_CAPTURE = {
    # cfg: dict(traffic=bytes per launch, executed=per particle-step, kernels=blob of csrc/abm_kernels.cuh,
    #           device=blob of csrc/abm_device.cuh, summary=file under profiles/)
    0: dict(traffic=80_128, executed=40.89, **_SRC),
    1: dict(traffic=12_692_480, executed=30.78, **_SRC),
    2: dict(traffic=56_665_600, executed=30.29, **_SRC),
    # one of the 20 launches (1,000 steps each) of a pass
    3: dict(traffic=21_009_408, executed=50.36, **_SRC),
    # FP64-pipe operations (146 per Philox block in the loop; ncu: sm__pipe_fp64_cycles_active 71.55 %); the fp64
    # kernel is the one of round 2 (same instruction count, 576.4 ms), so the operation count is carried over
    4: dict(traffic=157_319_168, executed=36.5, **_SRC),
}
# Warp-lane instructions per particle-step of the xorshift variant are not frozen anywhere: no `frac` for it.


def git_blob(path):
    """What `git hash-object` prints for the file."""
    import hashlib
    data = open(path, "rb").read()
    return hashlib.sha1(b"blob %d\0" % len(data) + data).hexdigest()


def ncu_capture(cfg_id):
    """-> (entry or None, where it comes from / why there is none)"""
    ent = NCU_CAPTURE.get(cfg_id)
    if not ent:
        return None, "no committed capture of this launch"
    csrc = os.path.join(ROOT, "paper_1104_2499_b200", "csrc")
    now = (git_blob(os.path.join(csrc, "abm_kernels.cuh")), git_blob(os.path.join(csrc, "abm_device.cuh")))
    if now != (ent["kernels"], ent["device"]):
        return None, f"stale: kernel sources changed since the capture in {ent['summary']}"
    return ent, f"ncu --set full, per launch, {ent['summary']}"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return json.load(open(path)), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback (B200_PROFILING.md)"


# ---------------------------------------------------------------------------------------------
# clocks sampled DURING the timed region
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    def __init__(self, index=0, period=0.2):
        self.index, self.period = index, period
        self.sm, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20,
                 "hw_thermal_slowdown": 0x40, "hw_power_brake": 0x80, "sync_boost": 0x10,
                 "app_clocks": 0x2}
        while not self._stop.is_set():
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr:
            self._thr.join()

    def summary(self):
        if not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["unavailable"]}
        return {"sm_mhz": float(statistics.median(self.sm)), "sm_max_mhz": float(self.max_mhz),
                "reasons": sorted(self.reasons), "samples": len(self.sm)}


# ---------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline and --impl reference): the ONLY places bench.py touches oracle/
# ---------------------------------------------------------------------------------------------
def oracle_sample(wl, every, n_steps, threads):
    """Oracle on every `every`-th trajectory of set 0 for the first n_steps steps -> (psteps, seconds)."""
    from oracle import abm_oracle as orc
    p = wl.set_params(0)
    n = max(wl.n_particles // every, 1)
    x, v, e = orc.init_many(p, wl.seed, n, 0, every)
    t0 = time.perf_counter()
    orc.run(p, wl.seed, x, v, e, 0, n_steps, 0, every, threads=threads)
    dt = time.perf_counter() - t0
    assert np.isfinite(x).all()
    return n * n_steps, dt


def cpu_baseline(wl, budget_s=6.0):
    """Oracle as it stands on the host cores: one thread, then the same loop split over all cores."""
    from oracle import abm_oracle as orc
    cores = orc.host_threads()
    every1 = max(wl.n_particles // 2048, 1)
    ps, dt = oracle_sample(wl, every1, 200, 1)            # calibrate
    rate1 = ps / dt
    n1 = int(max(200, min(wl.n_steps, budget_s * rate1 / (wl.n_particles // every1))))
    ps1, dt1 = oracle_sample(wl, every1, n1, 1)
    everyN = max(wl.n_particles // (2048 * cores), 1)
    psN, dtN = oracle_sample(wl, everyN, n1, cores)
    return {
        "value": psN / dtN, "unit": "particle-steps/s", "cores": cores, "kind": "oracle",
        "single_thread_value": ps1 / dt1,
        "sample": f"{wl.name}: every {everyN}th trajectory ({wl.n_particles // everyN}) x first {n1} "
                  f"steps on {cores} threads ({psN:.3g} particle-steps in {dtN:.2f} s); single thread: "
                  f"every {every1}th x {n1} steps in {dt1:.2f} s; fp64, plain C, not tuned",
    }


def run_reference(args, wl):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import abm_oracle as orc
    cores = orc.host_threads()
    every = max(wl.n_particles // (2048 * cores), 1)
    n_steps = 1000
    for _ in range(args.warmup):
        oracle_sample(wl, every, 100, cores)
    tot_ps, tot_t = 0, 0.0
    for _ in range(args.steps):
        ps, dt = oracle_sample(wl, every, n_steps, cores)
        tot_ps += ps
        tot_t += dt
    val = tot_ps / tot_t
    sample = (f"each step = every {every}th trajectory ({wl.n_particles // every}) x first {n_steps} steps "
              f"of {wl.name} on {cores} host threads")
    print(json.dumps({
        "impl": "reference", "metric": "particle-steps/sec", "value": val, "unit": "particle-steps/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "sample": sample},
        "cpu_baseline": {"value": val, "unit": "particle-steps/s", "cores": cores, "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": val, "unit": "particle-steps/s", "h2d_bytes_per_step": 0,
                "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
def run_ours(args, wl, cfg_id):
    import torch
    import torch.distributed as dist
    from paper_1104_2499_b200 import binding as abm, sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference "
                         "for the oracle)")
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE is {world}: launch one rank per GPU "
                         f"(torchrun --nproc-per-node {args.gpus}, or the bare `python bench.py --gpus N`)")
    n_dev = torch.cuda.device_count()
    if args.backend == "nccl" and n_dev < world:
        raise SystemExit(f"bench.py: --gpus {world} needs {world} CUDA devices, this box has {n_dev} "
                         "(--backend gloo rehearses the multi-rank flow with ranks sharing a GPU)")
    torch.cuda.set_device(local_rank % n_dev)
    if world > 1:
        if args.backend == "nccl":
            # the communicator's own log lines (rank count, transport: NVLS / P2P over NVLink) go to stderr
            os.environ.setdefault("NCCL_DEBUG", "INFO")
            os.environ.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
            dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        else:   # gloo: exercises the multi-rank flow where ranks must share one GPU (NCCL refuses that)
            dist.init_process_group("gloo")
    coll_dev = "cuda" if args.backend == "nccl" else "cpu"
    print(f"[bench rank {rank}/{world}] cuda:{torch.cuda.current_device()} "
          f"{torch.cuda.get_device_name()} backend {args.backend if world > 1 else 'none'}",
          file=sys.stderr, flush=True)
    abm.lib()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    peaks, peak_src = load_peaks()
    f_max = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")  # > 126 MB L2

    def measure(wl, cfg_id, steps, warmup, with_offset=True):
        """`warmup` untimed + `steps` device-timed + `steps` end-to-end passes of one workload -> (line, moments)."""
        stream = torch.cuda.Stream()
        all_sets = [dict(wl.set_params(s), rng=1 if args.rng == "xorshift" else 0) for s in range(wl.n_param_sets)]
        # weak: rank r integrates a full copy of the workload on global trajectories [r*T, (r+1)*T);
        # strong: the one ensemble is divided (whole sets per rank, else realisations), SURVEY.md 8(e)
        plan = sharding.shard_plan(wl.n_particles, wl.n_param_sets, rank, world, args.scaling)
        sets = all_sets[plan.set_first:plan.set_first + plan.n_sets]
        n_particles = plan.n_particles
        T = n_particles * len(sets)                      # trajectories of THIS rank
        n_steps, M = wl.n_steps, (wl.moments_every or wl.n_steps)
        fp64 = sets[0]["precision"] == 1
        frame_cols = 2
        frame_item = 8 if fp64 else 4
        host_frame = torch.empty((T, frame_cols), dtype=torch.float64 if fp64 else torch.float32,
                                 pin_memory=True)
        (mom_out, _mom_keep), (sums_out, _sums_keep) = abm.pinned_moment_buffers(len(sets))  # pinned: true DMA
        # one pinned record array per intermediate reduction of a pass (config[3]: 19)
        mom_slots = [abm.pinned_moment_buffers(len(sets))[0] for _ in range(max(n_steps // M - 1, 0))]
        # N > 1: device + pinned buffers of the one exchange, a slot per reduction of a pass
        exchange = sharding.MomentExchange(plan, n_slots=n_steps // M, backend=args.backend) if world > 1 else None
        launches = {"n": 0}
        ens_tilt = any(p["A"] != 0.0 for p in sets)
        step_launches = (2 if ens_tilt else 1) * -(-M // (65536 if ens_tilt else 2**30))
        # parameter records marshalled once (host side); abm_create copies them to the device
        params = abm.make_params(sets, stream=stream.cuda_stream, snapshot_every=wl.snapshot_every,
                                 traj_base=plan.traj_base, traj_set_stride=plan.traj_set_stride)
        params_bytes = len(sets) * abm.C.sizeof(abm.abm_params)

        def one_pass(e2e, ev=None):
            """The whole hot path once.  Returns the moments (host)."""
            with torch.cuda.stream(stream):
                ens = abm.Ensemble(params, n_particles, wl.seed, stream=stream)    # S0 (1 kernel)
                launches["n"] += 1
                if wl.snapshot_every:
                    ens.bind_snapshot()                                            # S5 (1 kernel)
                    launches["n"] += 1
                m = None
                for j in range(n_steps // M):
                    if ev is not None:
                        ev[j][0].record(stream)
                    ens.step(M)                                                    # S1-S5, S7
                    if ev is not None:
                        ev[j][1].record(stream)
                    launches["n"] += step_launches
                    if world > 1:                          # S6 (2 kernels) + all-reduce, enqueued: no host round trip
                        exchange.enqueue(ens, j)
                    elif j + 1 < n_steps // M:     # intermediate reductions: enqueued, no host round trip
                        ens.moments_async(mom_slots[j][0])                         # S6 (2 kernels)
                    else:                          # the last one waits: every record is on the host now
                        m = ens.moments(mom_out)                                   # S6 (2 kernels)
                    launches["n"] += 2
                if e2e:
                    abm.abm_snapshot_host(ens.ctx, host_frame.numpy(), frame_cols * frame_item)
                    launches["n"] += 1
                ens.close()                                # waits for the stream: every record is on the host
                if world > 1:
                    m = exchange.result(n_steps // M - 1)
            return m

        for _ in range(max(warmup, 0)):
            one_pass(False)
            one_pass(True)
        barrier()

        # ---- device-timed arm -------------------------------------------------------------------
        ev_pass = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                   for _ in range(steps)]
        ev_kern = [[(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                    for _ in range(n_steps // M)] for _ in range(steps)]   # around every abm_step
        launches["n"] = 0
        barrier()
        wall0 = time.perf_counter()
        with ClockSampler(torch.cuda.current_device()) as clk:
            for i in range(steps):
                flush.fill_(i & 0xff)                       # L2 flush between timed iterations
                torch.cuda.synchronize()
                ev_pass[i][0].record(stream)
                m = one_pass(False, ev_kern[i])
                ev_pass[i][1].record(stream)
            barrier()
        wall = time.perf_counter() - wall0
        gpu_launches = launches["n"]
        t_pass_ms = [a.elapsed_time(b) for a, b in ev_pass]
        t_dev = sum(t_pass_ms) * 1e-3
        t_kern_ms = [sum(a.elapsed_time(b) for a, b in evs) for evs in ev_kern]   # per pass, all abm_step calls

        # ---- end-to-end arm (host params -> host frame + moments), wall clock ---------------------
        barrier()
        t0 = time.perf_counter()
        for i in range(steps):
            one_pass(True)
        barrier()
        t_e2e = time.perf_counter() - t0

        # ---- the paper's "offset time": 20 launches of one step, the last 15 ----
        t_off = None
        if with_offset:
            with torch.cuda.stream(stream):
                ens = abm.Ensemble(params, n_particles, wl.seed, stream=stream)
                if wl.snapshot_every:
                    ens.bind_snapshot()
                ev_off = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
                          for _ in range(20)]
                for a, b in ev_off:
                    a.record(stream)
                    ens.step(1)
                    b.record(stream)
                stream.synchronize()
                ens.close()
            t_off = [a.elapsed_time(b) for a, b in ev_off][5:]

        tt = torch.tensor([t_dev, t_e2e], dtype=torch.float64, device=coll_dev)
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_dev, t_e2e = float(tt[0]), float(tt[1])

        # particle-steps of the whole job: weak = `world` copies of the workload, strong = the one workload
        psteps_rank = T * n_steps
        psteps_job = wl.particle_steps * (world if args.scaling == "weak" else 1) * steps
        value = psteps_job / t_dev
        clocks = clk.summary()

        out = {
            "metric": "particle-steps/sec", "value": value, "unit": "particle-steps/s",
            "n_gpus": world, "steps": steps, "warmup": warmup,
            "ms_per_step": 1e3 * t_dev / steps, "higher_is_better": True, "scaling": args.scaling,
            "ms_per_step_sd": statistics.pstdev(t_pass_ms) if len(t_pass_ms) > 1 else None,   # this rank's passes
            "offset_ms": {"mean": statistics.mean(t_off), "sd": statistics.pstdev(t_off),
                          "protocol": "20 launches of 1 step, last 15 (PAPER.md:100, :122)"} if t_off else None,
            "vs_baseline": None,   # the paper states no throughput for this path
            "dtype": "f64" if fp64 else "f32", "data": "synthetic",
            "config": {"workload": wl.name, "baseline_config": cfg_id, "trajectories_per_gpu": T,
                       "param_sets": wl.n_param_sets, "sim_steps": n_steps,
                       "snapshot_every": wl.snapshot_every, "moments_every": M,
                       "integrator": "heun" if sets[0]["integrator"] else "euler-maruyama", "rng": args.rng,
                       "scaling": args.scaling, "shard": plan.split if world > 1 else "none",
                       "l2": "flushed between timed iterations (256 MiB fill)",
                       "pass": "create+init, bind frame, integrate, moments, destroy"},
            "e2e": {"value": psteps_job / t_e2e, "unit": "particle-steps/s",
                    "h2d_bytes_per_step": int(params_bytes),
                    "d2h_bytes_per_step": int(host_frame.numel() * host_frame.element_size()
                                              + 80 * len(sets) * (n_steps // M)),
                    "timer": "wall clock, host parameter records -> pinned host frame + moments"},
            "gpu_launches": gpu_launches,
            "clocks": clocks,
            "wall_s_timed_region": wall,
        }
        if t_kern_ms:
            t_k = statistics.mean(t_kern_ms) * 1e-3
            lane_instr = I_ALG[cfg_id] * psteps_rank
            lanes = LANES_FP64 if fp64 else LANES_PER_SM
            peak = N_SM * lanes * f_max
            achieved = lane_instr / t_k
            sm_mhz = clocks.get("sm_mhz") or (f_max / 1e6)
            cap, cap_src = ncu_capture(cfg_id) if (not args.sim_steps and args.rng == "philox" and world == 1) else \
                (None, "no capture of this launch (--sim-steps / --rng xorshift / sharded)")
            philox = args.rng == "philox"
            out["roofline"] = {
                "bound": "alu",
                "kernel": "abm::step_kernel_small" if (not fp64 and args.rng == "philox" and
                                                        T <= 96 * torch.cuda.get_device_properties(0).multi_processor_count)
                else "abm::step_kernel",   # AUTO: up to three 32-trajectory CTAs per SM (include/abm.h)
                "achieved": achieved / 1e12 if philox else None,
                "peak": peak / 1e12,
                "unit": "Tinstr/s (FP64-pipe lane operations)" if fp64 else "Tinstr/s (warp-lane instructions)",
                "frac": achieved / peak if philox else None,     # I_alg is frozen for the Philox path only
                "frac_at_sustained_clock": achieved / (N_SM * lanes * sm_mhz * 1e6) if philox else None,
                "i_alg_per_particle_step": I_ALG[cfg_id] if philox else None,
                # the same with what the kernel executes per particle-step in place of I_alg (ncu capture): how busy
                # the issue slots (fp64: the FP64 pipe) are, whatever the instructions are worth
                "frac_executed": cap["executed"] * psteps_rank / t_k / peak if cap else None,
                "executed_per_particle_step": cap["executed"] if cap else None,
                "particle_steps_per_pass": psteps_rank,
                "kernel_ms": 1e3 * t_k, "kernel_ms_sd": statistics.pstdev(t_kern_ms) if len(t_kern_ms) > 1 else None,
                "kernel_launches_per_pass": step_launches * (n_steps // M),
                "kernel_share_of_pass": sum(t_kern_ms) / sum(t_pass_ms),
                "peak_source": f"148 SMs x {lanes} lanes x sm_max_mhz {f_max / 1e6:.0f} MHz, {peak_src}",
                "traffic": cap["traffic"] if cap else None, "traffic_source": cap_src,
                "hbm_algorithmic_bytes_per_launch": int(T * (24 + 8 * (n_steps // wl.snapshot_every
                                                                       if wl.snapshot_every else 0))),
            }
        return out, m

    out, m = measure(wl, cfg_id, args.steps, args.warmup)
    # The other BASELINE.json configs, measured AFTER the headline's timed regions (which they cannot disturb) with
    # the same protocol and fewer passes, so that the one line the driver runs carries all five.
    if world == 1 and args.all_configs and cfg_id == 1 and not args.sim_steps and args.rng == "philox":
        extra = {}
        for other in (0, 2, 3, 4):
            o, _ = measure(W.CONFIGS[other](), other, args.all_configs, 1, with_offset=False)
            r = o["roofline"]
            extra[o["config"]["workload"]] = {
                "value": o["value"], "ms_per_step": o["ms_per_step"], "steps": o["steps"], "dtype": o["dtype"],
                "kernel": r["kernel"], "kernel_ms": r["kernel_ms"], "kernel_ms_sd": r["kernel_ms_sd"],
                "frac": r["frac"], "frac_executed": r["frac_executed"], "unit": r["unit"],
                "e2e": o["e2e"]["value"], "clocks": o["clocks"]}
        out["all_configs"] = extra
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(wl)
        m0 = m[0]
        out["result"] = {"step": int(m0["step"]), "mean_v": float(m0["mean_v"]),
                         "var_x": float(m0["var_x"]), "mean_e": float(m0["mean_e"])}
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def launcher_command(argv, n_gpus, port=None):
    """The command a bare `python bench.py --gpus N` (N > 1, no WORLD_SIZE) re-executes: one rank per GPU."""
    if port is None:
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n_gpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, help="BASELINE.json config index (default 1)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="collective backend for N > 1 (gloo only to rehearse the flow with ranks sharing a GPU)")
    ap.add_argument("--rng", default="philox", choices=["philox", "xorshift"],
                    help="generator A/B (SURVEY.md 8(f) NEXT-4); the headline and the roofline are Philox")
    ap.add_argument("--sim-steps", type=int, default=0, help="override the config's step count")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: every rank a full copy on its own trajectory indices (weak, default), or the one "
                         "ensemble divided over the ranks (strong: [gT/G, (g+1)T/G), SURVEY.md 8(e))")
    ap.add_argument("--all-configs", type=int, default=3, metavar="PASSES",
                    help="after the headline (config 1, N = 1) also time configs 0, 2, 3, 4 with this many passes "
                         "each -> \"all_configs\" in the line; 0 = skip")
    args = ap.parse_args()
    wl = W.CONFIGS[args.config]()
    if args.sim_steps:
        wl.n_steps = args.sim_steps
        if wl.moments_every:
            wl.moments_every = min(wl.moments_every, wl.n_steps)
    if args.impl == "reference":
        run_reference(args, wl)
        return
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not under torchrun: start the N ranks ourselves (one process per GPU)
        import subprocess
        cmd = launcher_command(sys.argv[1:], args.gpus)
        print("bench.py: launching " + " ".join(cmd), file=sys.stderr, flush=True)
        raise SystemExit(subprocess.call(cmd))
    run_ours(args, wl, args.config)


if __name__ == "__main__":
    main()
