"""The paper's two measurement campaigns, re-run on one B200 through the C ABI.

    python -m paper_1104_2499_b200.studies scaling      [--out profiles/rNN_scaling]
    python -m paper_1104_2499_b200.studies presentation [--out profiles/rNN_presentation]
    python -m paper_1104_2499_b200.studies fig2         [--out profiles/rNN_fig2]

scaling       PAPER.md:100-136 (Figs. 3-4): time of one launch against the number of work items, for
              0, 10^3 and 10^4 iterations per launch; 20 launches per size, the last 15 averaged (:100);
              per-iteration time and offset from a linear fit over the iteration counts (:174).  Work items =
              trajectories of the paper's F0 sweep (one per parameter set, :74).  Sizes: powers of two
              2^0 .. 2^22; the paper's own fine sweep, 50 .. 3,500 work items in steps of 50 (:122, Fig. 4), which on
              148 SMs lies inside the flat region; and a fine sweep in steps of one eighth of a wave that shows
              where the paper's "bands" (:122-134) would fall on this machine.
presentation  PAPER.md:138-194 (Tab. 1): what showing a frame costs, in "iterations lost" = cost / time of
              one iteration at that size.  No graphics stack exists on this box, so the three columns are:
              the device-resident frame (the shared-buffer analogue, :156-162), a device->host copy of the
              frame (the non-shared buffer, :152-154), text formatting of the copied frame (the gnuplot
              pipe, :144-150; formatting only, nothing is drawn), plus the CUDA rasteriser (abm_raster).

fig2          PAPER.md:72-74, :94-96 (Fig. 2): the paper's example result, <v> against the opposing force F0.

All write a .csv and a .md (with the command) next to each other.  Timing: CUDA events on the launching
stream for device work, perf_counter around synchronous host work.
"""
import argparse
import io
import os
import statistics
import sys
import time

import numpy as np

from . import binding as abm, workloads as W

REPS, KEEP = 20, 15


def _events(torch):
    return torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)


def _launch_times(torch, ens, stream, n_iter, reps=REPS, keep=KEEP):
    """ms per abm_step(n_iter) launch: `reps` launches, the last `keep` averaged.  n_iter = 0 measures the
    offset the way the paper does (a launch that reads and writes the state but iterates zero times) with
    the smallest launch the ABI has: one step."""
    ts = []
    for _ in range(reps):
        a, b = _events(torch)
        a.record(stream)
        ens.step(max(n_iter, 1))
        b.record(stream)
        b.synchronize()
        ts.append(a.elapsed_time(b))
    ts = ts[-keep:]
    return statistics.mean(ts), (statistics.stdev(ts) if len(ts) > 1 else 0.0)


def _sweep_ensemble(torch, n_items, stream):
    wl = W.paper_f0_sweep(n_F0=n_items, realisations=1)
    if n_items <= 65_536:
        sets = [wl.set_params(s) for s in range(n_items)]
        return abm.Ensemble(sets, 1, wl.seed, stream=stream)
    # beyond the paper's 2^16 parameter values: 65,536 values x realisations
    reals = n_items // 65_536
    wl = W.paper_f0_sweep(n_F0=65_536, realisations=reals)
    sets = [wl.set_params(s) for s in range(65_536)]
    return abm.Ensemble(sets, reals, wl.seed, stream=stream)


def scaling(out):
    import torch
    torch.cuda.set_device(0)
    stream = torch.cuda.Stream()
    iters = [0, 1000, 10_000]
    sizes = [2 ** k for k in range(0, 23)]
    wave = 148 * 128 * 8                 # trajectories resident at once (one-set fp32 EM kernel: 8 CTAs/SM)
    fine = [wave * j // 8 for j in range(1, 33)]   # realisations of ONE parameter set (config[1]'s model)
    paper_fine = list(range(50, 3501, 50))         # "from 50 to 3500 with step 50"
    rows = []
    with torch.cuda.stream(stream):
        for kind, ns in (("pow2", sizes), ("paper_fine", paper_fine), ("fine", fine)):
            for n in ns:
                if kind == "fine":
                    n_eff = n
                    wl = W.config1(n_particles=n)
                    ens = abm.Ensemble([wl.set_params(0)], n, wl.seed, stream=stream)
                else:
                    n_eff = n if n <= 65_536 else (n // 65_536) * 65_536
                    ens = _sweep_ensemble(torch, n_eff, stream)
                ens.step(8)              # warm-up launch
                t = {}
                for it in iters:
                    if kind == "fine" and it != 10_000:
                        continue
                    t[it] = _launch_times(torch, ens, stream, it)
                ens.close()
                if kind != "fine":
                    xs = np.array([max(i, 1) for i in iters], float)
                    ys = np.array([t[i][0] for i in iters])
                    slope, offset = np.polyfit(xs, ys, 1)
                else:
                    slope, offset = t[10_000][0] / 10_000, float("nan")
                rows.append((kind, n_eff, t.get(0, (float("nan"),) * 2), t.get(1000, (float("nan"),) * 2),
                             t[10_000], slope * 1e3, offset * 1e3))
                print(f"{kind} N={n_eff}: " + "  ".join(f"{k}:{v[0]:.4f}ms" for k, v in t.items()), flush=True)
    with open(out + ".csv", "w") as f:
        f.write("kind,work_items,ms_0it,sd_0it,ms_1e3it,sd_1e3it,ms_1e4it,sd_1e4it,us_per_iteration,offset_us,"
                "particle_steps_per_s_at_1e4\n")
        for kind, n, t0, t3, t4, slope, off in rows:
            f.write(f"{kind},{n},{t0[0]:.5f},{t0[1]:.5f},{t3[0]:.5f},{t3[1]:.5f},{t4[0]:.5f},{t4[1]:.5f},"
                    f"{slope:.5f},{off:.3f},{n * 10_000 / (t4[0] * 1e-3):.4e}\n")
    return rows


def presentation(out):
    import torch
    torch.cuda.set_device(0)
    stream = torch.cuda.Stream()
    rows = []
    with torch.cuda.stream(stream):
        for n in (2 ** 6, 2 ** 13, 2 ** 16, 2 ** 20):
            ens = _sweep_ensemble(torch, n, stream)
            ens.step(1000)
            t_it = _launch_times(torch, ens, stream, 10_000, reps=8, keep=5)[0] / 10_000      # ms per iteration
            frame = ens.bind_snapshot(with_e=True)                                             # float4 vertex, :162
            host = np.empty((ens.n_traj, 4), np.float32)
            res = {}
            # (a) device-resident frame: one rewrite of the bound buffer (what abm_step does every K steps)
            ts = []
            for _ in range(REPS):
                a, b = _events(torch)
                a.record(stream)
                abm.abm_snapshot(ens.ctx, frame.data_ptr(), 16)
                b.record(stream)
                b.synchronize()
                ts.append(a.elapsed_time(b))
            res["device_frame"] = statistics.mean(ts[-KEEP:])
            # (b) frame copied to the host
            ts = []
            for _ in range(REPS):
                t0 = time.perf_counter()
                abm.abm_snapshot_host(ens.ctx, host, 16)
                ts.append(1e3 * (time.perf_counter() - t0))
            res["host_copy"] = statistics.mean(ts[-KEEP:])
            # (c) text formatting of the copied frame ("x v" per line, as for a gnuplot pipe); nothing is drawn
            ts = []
            for _ in range(3 if n > 2 ** 16 else REPS):
                t0 = time.perf_counter()
                abm.abm_snapshot_host(ens.ctx, host, 16)
                buf = io.StringIO()
                np.savetxt(buf, host[:, :2], fmt="%.6g")
                ts.append(1e3 * (time.perf_counter() - t0))
            res["text"] = statistics.mean(ts[-KEEP:])
            # (d) CUDA rasteriser: 1024 x 1024 histogram + RGBA8
            counts, rgba = ens.raster(1024, 1024, -4.0, 4.0, saturation=4)
            ts = []
            for _ in range(REPS):
                a, b = _events(torch)
                a.record(stream)
                abm.abm_raster(ens.ctx, counts.data_ptr(), 1024, 1024, -4.0, 4.0, rgba.data_ptr(), 4)
                b.record(stream)
                b.synchronize()
                ts.append(a.elapsed_time(b))
            res["raster_1024"] = statistics.mean(ts[-KEEP:])
            ens.close()
            rows.append((n, t_it, res))
            print(n, f"{t_it * 1e3:.3f} us/iteration", {k: round(v, 4) for k, v in res.items()}, flush=True)
    with open(out + ".csv", "w") as f:
        f.write("work_items,us_per_iteration,device_frame_ms,host_copy_ms,text_ms,raster_1024_ms,"
                "device_frame_iters,host_copy_iters,text_iters,raster_1024_iters\n")
        for n, t_it, r in rows:
            keys = ["device_frame", "host_copy", "text", "raster_1024"]
            f.write(f"{n},{t_it * 1e3:.4f}," + ",".join(f"{r[k]:.5f}" for k in keys) + "," +
                    ",".join(f"{r[k] / t_it:.1f}" for k in keys) + "\n")
    return rows


def fig2(out):
    """The paper's example plot (Fig. 2): mean velocity against the opposing load F0, averaged
    over time and launches (:74).  1,024 values of F0 in [-1, 0] x 1,024 realisations on the Eq. 3 potential
    (h = 1; depot parameters of BASELINE.json configs[0] -- the paper prints none), ten launches of 10^4 iterations
    (:122); after every launch the running average <x(t) - x(0)> / t of each work item, as the paper's display
    loop shows it.  The standard error comes from the same device reduction (mean_dx, mean_dx2)."""
    import torch
    torch.cuda.set_device(0)
    stream = torch.cuda.Stream()
    wl = W.paper_f0_sweep(n_F0=1024, F0_min=-1.0, F0_max=0.0, realisations=1024, n_steps=100_000)
    sets = [wl.set_params(s) for s in range(wl.n_param_sets)]
    dt = sets[0]["dt"]
    cols = []
    with torch.cuda.stream(stream):
        ens = abm.Ensemble(sets, wl.n_particles, wl.seed, stream=stream)
        a, b = _events(torch)
        a.record(stream)
        for launch in range(10):
            ens.step(10_000)
            cols.append(ens.time_averaged_velocity())
        b.record(stream)
        b.synchronize()
        m = ens.moments()
        ens.close()
    t = 100_000 * dt
    se = np.sqrt(np.maximum(m["mean_dx2"] - m["mean_dx"] ** 2, 0.0) / wl.n_particles) / t
    with open(out + ".csv", "w") as f:
        f.write("F0," + ",".join(f"vbar_after_{(k + 1) * 10_000}_steps" for k in range(10)) + ",standard_error\n")
        for s in range(wl.n_param_sets):
            f.write(f"{sets[s]['F0']:.6f}," + ",".join(f"{c[s]:.6f}" for c in cols) + f",{se[s]:.6f}\n")
    print(f"fig2: {wl.n_trajectories} trajectories x 100000 steps in {a.elapsed_time(b):.1f} ms "
          f"(10 launches + 10 reductions); <v>(F0=-1) = {cols[-1][0]:+.4f}, <v>(F0=0) = {cols[-1][-1]:+.4f} "
          f"+- {se[-1]:.4f}", flush=True)
    return [None] * wl.n_param_sets


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("study", choices=["scaling", "presentation", "fig2"])
    ap.add_argument("--out", default=None)
    args = ap.parse_args()
    out = args.out or f"gpurun_out/{args.study}"
    os.makedirs(os.path.dirname(out) or ".", exist_ok=True)
    rows = {"scaling": scaling, "presentation": presentation, "fig2": fig2}[args.study](out)
    with open(out + ".md", "w") as f:
        f.write(f"# {args.study} study (SURVEY.md 8(f))\n\nCommand (B200, through gpurun):\n\n"
                f"    python -m paper_1104_2499_b200.studies {args.study} --out {out}\n\n"
                f"Data: `{os.path.basename(out)}.csv` ({len(rows)} rows). See the module docstring of "
                "`paper_1104_2499_b200/studies.py` for what each column is and which passage of the paper it follows.\n")
    print("wrote", out + ".csv")


if __name__ == "__main__":
    sys.exit(main())
