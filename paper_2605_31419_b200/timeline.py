"""Per-job timeline of the fused tracking kernel (ts_render_track_l1), for the work-distribution argument of DESIGN.md.

    python -m paper_2605_31419_b200.timeline --config 2 --out profiles/r03_timeline_config2

builds a PROFILING build of the same CUDA sources (-DTS_JOB_TIMELINE: every persistent warp stamps %globaltimer at the
start and at the end of each job it runs; libts_timeline.so, the product library is not touched), runs warm-up tracking
iterations of the BASELINE config on cuda:0, then one stamped launch, and writes
  <out>_jobs.csv    one row per job: ticket, tile, block, list length, warp, start_us, duration_us
  <out>_warps.csv   one row per persistent warp: jobs run, first start, last end, busy time
  <out>.md          the figures the bound is made of: launch span, instant until which every warp is busy, drain, the
                    longest jobs, and span >= max(longest job, total busy time / number of warps).
The stamps cost two timer reads and one 16-byte store per job (25 800 jobs at config 2) and the stamped launch is slower
than the product kernel (config 2: about 100 us against 89 us by CUDA events), so its time is reported and never used as
a benchmark value: what the stamps show is how the work is DISTRIBUTED over the warps.  --define NAME=VALUE adds compile
definitions to the profiling build, e.g. the ticket policy before round 3 (every warp requests its next ticket at the
start of the current job):  --define TS_PREFETCH_MAX_LEN=0x40000000u --define TS_TAIL_ROUNDS=0u --tag prefetch_always.
Argument marshalling and bookkeeping only: nothing of the method is computed here.
"""
from __future__ import annotations

import argparse
import os
import sys

import numpy as np


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2, choices=[1, 2])
    ap.add_argument("--out", default="gpurun_out/timeline")
    ap.add_argument("--warmup", type=int, default=40)
    ap.add_argument("--define", action="append", default=[], help="extra NAME=VALUE compile definition (repeatable)")
    ap.add_argument("--tag", default="", help="suffix of the profiling build's name when --define is used")
    args = ap.parse_args()

    from paper_2605_31419_b200 import build
    os.environ["TS_LIBTS"] = build.build_variant("timeline" + ("_" + args.tag if args.tag else ""), ["TS_JOB_TIMELINE", *args.define])
    import torch
    from paper_2605_31419_b200 import scenes, ts

    assert torch.cuda.is_available(), "needs a CUDA device"
    torch.cuda.set_device(0)
    sc = scenes.make_config(args.config)
    ctx = ts.Context(0)
    d = lambda a: torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float32).cuda()
    scene = ts.Scene(d(sc.pos), d(sc.color), d(sc.opacity))
    cam, prm = ts.make_camera(sc.cam), ts.make_params(sc.params)
    W, H = sc.cam.width, sc.cam.height
    frame = ts.Frame(ctx, scene.M, W, H, pair_capacity=max(2 * scene.M, 1 << 16))
    Chat, Dhat = torch.zeros(3, H, W, device="cuda"), torch.zeros(H, W, device="cuda")
    # target frame = the render at the ground-truth pose, as in bench.py
    ts.ts_project(ctx, scene, cam, prm, d(sc.T_gt[0].reshape(-1)), frame)
    ts.ts_bin_sort(ctx, frame)
    ts.ts_render_fwd(ctx, scene, frame, Chat, Dhat, None)
    T = d(sc.T_start[0].reshape(-1))
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    evs = []
    for _ in range(args.warmup + 1):                          # the stamps that are read back are those of the last launch
        ts.ts_project(ctx, scene, cam, prm, T, frame)
        ts.ts_bin_sort(ctx, frame)
        flush.fill_(1)                                        # cold L2, as in the benchmark protocol
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        ts.ts_render_track_l1(ctx, scene, frame, None, None, None, Chat, Dhat, sc.params.lambda_dep)
        ev1.record()
        evs.append((ev0, ev1))
    torch.cuda.synchronize()
    launch_us = evs[-1][0].elapsed_time(evs[-1][1]) * 1e3
    median_us = float(np.median([a.elapsed_time(b) for a, b in evs[len(evs) // 2:]])) * 1e3
    jobs = ts.ts_frame_view(ctx, frame, ts.VIEW_JOBS).cpu().numpy().reshape(-1, 4).view(np.uint32).astype(np.int64)
    tl = ts.ts_frame_view(ctx, frame, ts.VIEW_TIMELINE).cpu().numpy().reshape(-1, 4).view(np.uint32).astype(np.int64)
    n = jobs.shape[0]
    t0 = tl[:, 0].min()
    start = ((tl[:, 0] - t0) % (1 << 32)) * 1e-3              # us since the first job started (32-bit ns stamps)
    dur = ((tl[:, 1] - tl[:, 0]) % (1 << 32)) * 1e-3
    end = start + dur
    length, warp = tl[:, 2], tl[:, 3]
    assert np.array_equal(length, jobs[:, 2] - jobs[:, 1]), "timeline rows are not in ticket order"
    os.makedirs(os.path.dirname(args.out) or ".", exist_ok=True)
    with open(args.out + "_jobs.csv", "w") as fh:
        fh.write("ticket,tile,block,list_len,warp,start_us,duration_us\n")
        for j in range(n):
            fh.write(f"{j},{jobs[j, 0] & 0x0fffffff},{(jobs[j, 0] >> 28) & 7},{length[j]},{warp[j]},{start[j]:.3f},{dur[j]:.3f}\n")
    n_warps = int(warp.max()) + 1
    w_jobs = np.bincount(warp, minlength=n_warps)
    w_busy = np.bincount(warp, weights=dur, minlength=n_warps)
    w_first = np.full(n_warps, np.inf)
    w_last = np.zeros(n_warps)
    np.minimum.at(w_first, warp, start)
    np.maximum.at(w_last, warp, end)
    with open(args.out + "_warps.csv", "w") as fh:
        fh.write("warp,jobs,first_start_us,last_end_us,busy_us\n")
        for w in range(n_warps):
            fh.write(f"{w},{w_jobs[w]},{w_first[w]:.3f},{w_last[w]:.3f},{w_busy[w]:.3f}\n")
    span, all_busy = float(end.max()), float(w_last[w_jobs > 0].min())
    order = np.argsort(-dur)[:20]
    with open(args.out + ".md", "w") as fh:
        fh.write(f"# Job timeline of render_track_kernel, config {args.config} ({sc.M} faces, {W}x{H})\n\n")
        extra = "".join(f" --define {d}" for d in args.define) + (f" --tag {args.tag}" if args.tag else "")
        fh.write(f"Command: `python -m paper_2605_31419_b200.timeline --config {args.config}{extra} --out {args.out}` "
                 f"(profiling build -DTS_JOB_TIMELINE; rows: `{os.path.basename(args.out)}_jobs.csv`, "
                 f"`{os.path.basename(args.out)}_warps.csv`).\n\n")
        fh.write("| quantity | value |\n|---|---|\n")
        fh.write(f"| jobs / persistent warps that ran one | {n} / {int((w_jobs > 0).sum())} of {n_warps} |\n")
        fh.write(f"| stamped launch, CUDA events (us) | {launch_us:.1f} (median of the later half of {len(evs)} launches: {median_us:.1f}) |\n")
        fh.write(f"| span first job start -> last job end (us) | {span:.1f} |\n")
        fh.write(f"| every warp still busy until (us) | {all_busy:.1f} |\n")
        fh.write(f"| drain = span - that instant (us) | {span - all_busy:.1f} |\n")
        fh.write(f"| longest job (us) / its list length / its start (us) | {dur[order[0]]:.1f} / {length[order[0]]} / {start[order[0]]:.1f} |\n")
        fh.write(f"| sum of job durations / warps = busy time per warp (us) | {dur.sum() / max(1, int((w_jobs > 0).sum())):.1f} |\n")
        fh.write(f"| mean job (us) / mean list length | {dur.mean():.2f} / {length.mean():.2f} |\n")
        fh.write(f"| jobs with an empty list | {int((length == 0).sum())} |\n\n")
        fh.write("The launch cannot end before its longest job does, nor before the warps have worked off the total job time "
                 "between them: span >= max(longest job end, busy time per warp).\n\n")
        fh.write("Twenty longest jobs:\n\n| ticket | tile | block | list length | start (us) | duration (us) | us per entry |\n|---|---|---|---|---|---|---|\n")
        for j in order:
            fh.write(f"| {j} | {jobs[j, 0] & 0x0fffffff} | {(jobs[j, 0] >> 28) & 7} | {length[j]} | {start[j]:.1f} | {dur[j]:.1f} | "
                     f"{dur[j] / max(1, length[j]):.2f} |\n")
        fh.write("\nDuration against list length (all jobs):\n\n| list length | jobs | mean duration (us) | share of total job time |\n|---|---|---|---|\n")
        edges = [0, 1, 2, 4, 8, 16, 32, 64, 128, 1 << 30]
        for a, b in zip(edges[:-1], edges[1:]):
            m = (length >= a) & (length < b)
            if m.any():
                fh.write(f"| {a}{'' if b == a + 1 else '-' + (str(b - 1) if b < (1 << 30) else '')} | {int(m.sum())} | {dur[m].mean():.2f} | "
                         f"{dur[m].sum() / dur.sum():.3f} |\n")
    print(open(args.out + ".md").read())
    frame.release()
    ctx.close()


if __name__ == "__main__":
    sys.exit(main())
