#!/usr/bin/env python
"""bench.py -- fwd+bwd render throughput of the triangle-splatting rasteriser hot path (BASELINE.json metric:
"fwd+bwd render Mpix/s @1200x680, 500k tris; tracking iters/s; % of roofline").

A step = ONE tracking iteration on BASELINE.json configs[2] (Replica-shaped, 1200x680, 500k faces, seed 2):
ts_project -> ts_bin_sort -> ts_render_track_l1 (= ts_render_fwd + ts_l1_loss_grad + ts_render_bwd(pose-only) in one
launch; C, D, A and the cotangent images are still written) ->
ts_pose_reduce_step (= ts_pose_jacobian_reduce + ts_pose_step in one launch), i.e. every row a1..a8 of DESIGN.md section 2, on synthetic data.
L2 is flushed between timed steps (the 18 MB map would otherwise stay L2-resident across iterations); the extra
"tracking_iters_per_s" figure is the 100-iteration block of one frame WITHOUT flushes (the real tracking loop).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

FP32_LANES_PER_SM = 128


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return {"hbm_gbs": d["hbm_gbs"], "sm_max_mhz": d.get("sm_max_mhz", 1965.0), "src": "measured"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "src": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) >= 7 and r[3 + i].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def algorithmic_work(cnt, HW, NT, M, p_sort, mode="pose"):
    """algorithmic bytes / FP32 flops per step from the measured counters, per bench stage
    (render_fwd = a3 + a4 fused: + 16 B/px of target read and 16 B/px of cotangents written)."""
    nv, P, nr, nh = cnt["n_visible"], cnt["n_pairs"], cnt["n_rect"], cnt["n_hit"]
    B = {"project": 36 * M + 4 * nv + 48 * nv,
         "bin_sort": 12 * nv + P * (12 + 8 + 24 * p_sort + 4) + 8 * NT,
         "render_fwd": 84 * nv + 24 * HW + 32 * HW,
         "render_bwd": 84 * nv + 28 * HW + (24 * NT if mode == "pose" else 168 * nv) + (0 if mode == "pose" else 144 * nv),
         "pose_reduce": 24 * NT}
    F = {"project": 130 * M, "bin_sort": 0, "render_fwd": 100 * P + 15 * nr + 40 * nh + 8 * HW,
         "render_bwd": 100 * P + 15 * nr + (170 if mode == "pose" else 190) * nh + 60 * nv, "pose_reduce": 60 * nv}
    B["render_track"] = B["render_fwd"] + B["render_bwd"]       # a3 + a4 + a5 in one launch: same rows, same work
    F["render_track"] = F["render_fwd"] + F["render_bwd"]
    return B, F


STEP_ROWS = ("project", "bin_sort", "render_fwd", "render_bwd", "pose_reduce")   # every row once


def load_traffic():
    """dram bytes per launch of each stage's kernels from the committed ncu --set full capture (profiles/)."""
    p = os.path.join(ROOT, "profiles", "r01_traffic.json")
    return json.load(open(p)) if os.path.exists(p) else {}


def rank_seed(config, rank):
    """Replicas / weak scaling: rank r tracks its own frame of the same scene family."""
    return config + 100 * rank


def max_over_ranks(dist, value, device):
    """Max over ranks of a scalar (device-timed milliseconds): one all-reduce outside the timed region."""
    import torch
    if dist is None:
        return float(value)
    t = torch.tensor([float(value)], device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the same config / metric (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import tso
    from paper_2605_31419_b200 import scenes
    sc = scenes.make_config(args.config)
    HW = sc.cam.width * sc.cam.height
    tgt_o = tso.Oracle(sc.pos, sc.color, sc.opacity, None, sc.T_gt[0], sc.cam, sc.params, "f32").forward("tiled")
    T = sc.T_start[0].copy()
    state = np.zeros(13, np.float32)
    lr = [1e-3] * 3 + [3e-3] * 3

    def step(T, state):
        o = tso.Oracle(sc.pos, sc.color, sc.opacity, None, T, sc.cam, sc.params, "f32")
        f = o.forward("tiled")
        L, gC, gD = o.l1_loss(f.color, f.depth, tgt_o.color, tgt_o.depth, sc.params.lambda_dep)
        g = o.backward(gC, gD, None, want=("pose",))
        return tso.pose_step_f32(T, g.dL_dtau, state, lr)

    for _ in range(args.warmup):
        T, state = step(T, state)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        T, state = step(T, state)
    dt = (time.perf_counter() - t0) / max(1, args.steps)
    val = HW / dt / 1e6
    cpu = {"value": val, "unit": "Mpix/s", "cores": 1, "kind": "oracle",
           "sample": f"{args.steps} full tracking iterations of {sc.name} (float32 tiled oracle, single thread)"}
    print(json.dumps({"impl": "reference", "metric": "fwd+bwd render Mpix/s", "value": val, "unit": "Mpix/s",
                      "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3,
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
                      "data": "synthetic", "config": {"workload": sc.name, "faces": sc.M, "image": [sc.cam.width, sc.cam.height]},
                      "cpu_baseline": cpu,
                      "e2e": {"value": val, "unit": "Mpix/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


class Tracker:
    """Device state of one tracking problem + the call sequence of one iteration (argument marshalling only)."""

    def __init__(self, sc, device, count_flags=0):
        import torch
        from paper_2605_31419_b200 import ts
        self.torch, self.ts, self.sc = torch, ts, sc
        self.ctx = ts.Context(device)
        d = lambda a, dt=torch.float32: torch.as_tensor(np.ascontiguousarray(a), dtype=dt).cuda()
        self.scene = ts.Scene(d(sc.pos), d(sc.color), d(sc.opacity))
        self.cam, self.prm = ts.make_camera(sc.cam), ts.make_params(sc.params, count_flags)
        self.W, self.H = sc.cam.width, sc.cam.height
        self.frame = ts.Frame(self.ctx, self.scene.M, self.W, self.H, pair_capacity=max(2 * self.scene.M, 1 << 16))
        H, W = self.H, self.W
        z = lambda *s: torch.zeros(*s, device="cuda")
        self.C, self.D, self.A = z(3, H, W), z(H, W), z(H, W)
        self.Chat, self.Dhat = z(3, H, W), z(H, W)
        self.gC, self.gD = z(3, H, W), z(H, W)
        self.T, self.tau, self.state, self.loss = d(sc.T_start[0].reshape(-1)), z(6), z(13), z(1)
        self.T0 = self.T.clone()
        self.lr = [1e-3] * 3 + [3e-3] * 3          # PAPER.md:440-441 (trans 0.001, rot 0.003)
        # target RGB-D frame = our own render at the ground-truth pose (synthetic stand-in for the dataset frame)
        Tgt = d(sc.T_gt[0].reshape(-1))
        ts.ts_project(self.ctx, self.scene, self.cam, self.prm, Tgt, self.frame)
        ts.ts_bin_sort(self.ctx, self.frame)
        ts.ts_render_fwd(self.ctx, self.scene, self.frame, self.Chat, self.Dhat, None)
        torch.cuda.synchronize()

    launches_per_iter = 1 + 2 + 1 + 1   # project, bin + sort, fwd+loss+bwd (ts_render_track_l1), reduce+step

    def forward(self):
        ts = self.ts
        ts.ts_project(self.ctx, self.scene, self.cam, self.prm, self.T, self.frame)
        ts.ts_bin_sort(self.ctx, self.frame)
        ts.ts_render_fwd_l1(self.ctx, self.scene, self.frame, self.C, self.D, self.A, self.Chat, self.Dhat,
                            self.sc.params.lambda_dep, self.gC, self.gD, self.loss)

    def iteration(self):
        """One tracking iteration, every row a1..a8: project, bin + sort, forward + L1 + pose-only backward (one fused
        launch; C, D, A and the cotangent images are still written), pose reduction + step."""
        ts = self.ts
        ts.ts_project(self.ctx, self.scene, self.cam, self.prm, self.T, self.frame)
        ts.ts_bin_sort(self.ctx, self.frame)
        ts.ts_render_track_l1(self.ctx, self.scene, self.frame, self.C, self.D, self.A, self.Chat, self.Dhat,
                              self.sc.params.lambda_dep, self.gC, self.gD, self.loss)
        ts.ts_pose_reduce_step(self.ctx, self.frame, self.tau, self.T, self.state, self.lr)

    def reset(self):
        self.T.copy_(self.T0)
        self.state.zero_()
        self.loss.zero_()

    def stages(self):
        """The iteration split at its API calls; the last two entries time the unfused forward and backward, which
        the fused ts_render_track_l1 replaces (reported for the roofline of the individual kernels)."""
        ts = self.ts
        lam = self.sc.params.lambda_dep
        return [("project", lambda: ts.ts_project(self.ctx, self.scene, self.cam, self.prm, self.T, self.frame)),
                ("bin_sort", lambda: ts.ts_bin_sort(self.ctx, self.frame)),
                ("render_track", lambda: ts.ts_render_track_l1(self.ctx, self.scene, self.frame, self.C, self.D, self.A,
                                                               self.Chat, self.Dhat, lam, self.gC, self.gD, self.loss)),
                ("pose_reduce", lambda: ts.ts_pose_reduce_step(self.ctx, self.frame, self.tau, self.T, self.state, self.lr)),
                ("render_fwd", lambda: ts.ts_render_fwd_l1(self.ctx, self.scene, self.frame, self.C, self.D, self.A, self.Chat,
                                                           self.Dhat, lam, self.gC, self.gD, self.loss)),
                ("render_bwd", lambda: ts.ts_render_bwd(self.ctx, self.scene, self.frame, self.gC, self.gD, None, None,
                                                        None, None, ts.GRAD_POSE))]


def cpu_baseline(sc, budget_iters=3):
    """The oracle as it stands, single thread, on the same frame (bounded: a few full iterations)."""
    from oracle import tso
    tgt = tso.Oracle(sc.pos, sc.color, sc.opacity, None, sc.T_gt[0], sc.cam, sc.params, "f32").forward("tiled")
    t0 = time.perf_counter()
    for _ in range(budget_iters):
        o = tso.Oracle(sc.pos, sc.color, sc.opacity, None, sc.T_start[0], sc.cam, sc.params, "f32")
        f = o.forward("tiled")
        L, gC, gD = o.l1_loss(f.color, f.depth, tgt.color, tgt.depth, sc.params.lambda_dep)
        o.backward(gC, gD, None, want=("pose",))
    dt = (time.perf_counter() - t0) / budget_iters
    return {"value": sc.cam.width * sc.cam.height / dt / 1e6, "unit": "Mpix/s", "cores": 1, "kind": "oracle",
            "sample": f"{budget_iters} full fwd+bwd tracking iterations of {sc.name}, float32 tiled oracle, 1 thread",
            "ms_per_step": dt * 1e3}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-graph", action="store_true")
    ap.add_argument("--skip-extras", action="store_true", help="only the timed region (for ncu launch lists)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3)
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2605_31419_b200 import scenes, ts
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks = load_peaks()
    # replicas / weak scaling: every rank tracks its own frame of the same scene family (seed offset by rank)
    sc = scenes.make_config(args.config, seed=rank_seed(args.config, rank)) if rank else scenes.make_config(args.config)
    HW, M = sc.cam.width * sc.cam.height, sc.M

    # counters (debug instantiation, outside the timed region)
    trc = Tracker(sc, local, count_flags=ts.PARAM_COUNTERS)
    trc.forward()
    fl, nvis, npairs = ts.ts_frame_status(trc.ctx, trc.frame)
    cn = ts.ts_frame_view(trc.ctx, trc.frame, ts.VIEW_COUNTERS).cpu().numpy()
    # the counting instantiation ran once, for the target render in Tracker.__init__ (the fused forward does not count)
    cnt = {"n_visible": int(nvis), "n_pairs": int(npairs), "n_warp_visits": int(cn[0]), "n_rect": int(cn[1]), "n_hit": int(cn[2]),
           "note": "n_rect / n_hit / n_warp_visits: one forward render (ground-truth pose); n_visible / n_pairs: start pose"}
    del trc
    torch.cuda.empty_cache()

    tr = Tracker(sc, local)
    NT = tr.frame_nt = ((sc.cam.width + 15) // 16) * ((sc.cam.height + 15) // 16)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.Stream()
    graph = None
    with torch.cuda.stream(stream):
        for _ in range(3):
            tr.iteration()
        stream.synchronize()
        if not args.no_graph:
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=stream):
                tr.iteration()
    run = (lambda: graph.replay()) if graph is not None else tr.iteration

    def timed(k, do_flush=True):
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(k)]
        with torch.cuda.stream(stream):
            for a, b in ev:
                if do_flush:
                    flush.fill_(1)
                a.record(stream)
                run()
                b.record(stream)
        stream.synchronize()
        return [a.elapsed_time(b) for a, b in ev]

    tr.reset()
    timed(args.warmup)
    tr.reset()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    clk = ClockSampler(local)
    clk.start()
    t_wall0 = time.perf_counter()
    ms = timed(args.steps)
    torch.cuda.synchronize()
    t_wall = time.perf_counter() - t_wall0
    total_ms = float(sum(ms))
    total_ms = max_over_ranks(dist, total_ms, "cuda")
    if dist is not None:
        dist.barrier()
    ms_per_step = total_ms / args.steps

    if args.skip_extras:
        if rank == 0:
            print(json.dumps({"metric": "fwd+bwd render Mpix/s", "value": world * HW / (ms_per_step * 1e-3) / 1e6,
                              "unit": "Mpix/s", "ms_per_step": ms_per_step, "steps": args.steps, "partial": True}))
        return
    # one frame = 100 tracking iterations back to back, no flush
    tr.reset()
    with torch.cuda.stream(stream):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(100):
            run()
        b.record(stream)
    stream.synchronize()
    frame_ms = a.elapsed_time(b)
    loss_after = None

    # per-stage device times: every stage captured into its own CUDA graph (so that host launch overhead does not
    # leak into the numbers), events between the graph launches; flush between steps
    tr.reset()
    stage_graphs = []
    with torch.cuda.stream(stream):
        for name, fn in tr.stages():
            if args.no_graph:
                stage_graphs.append((name, fn))
            else:
                gr = torch.cuda.CUDAGraph()
                with torch.cuda.graph(gr, stream=stream):
                    fn()
                stage_graphs.append((name, gr.replay))
    tr.reset()
    stage_ms = {}
    with torch.cuda.stream(stream):
        for it in range(args.steps):
            flush.fill_(1)
            evs = [torch.cuda.Event(enable_timing=True) for _ in range(len(stage_graphs) + 1)]
            evs[0].record(stream)
            for i, (name, fn) in enumerate(stage_graphs):
                fn()
                evs[i + 1].record(stream)
            for i, (name, fn) in enumerate(stage_graphs):
                stage_ms.setdefault(name, []).append((evs[i], evs[i + 1]))
    stream.synchronize()
    stage_ms = {k: float(np.median([a.elapsed_time(b) for a, b in v])) for k, v in stage_ms.items()}
    clocks = clk.stop()

    # extra, informational: one MAPPING view of the same scene (BASELINE.json configs[3]'s step is 8 of these on 1 M
    # faces): project + bin/sort + forward with L1 + full-gradient backward (positions, colours, opacities), one graph
    V = tr.scene.V
    gpos, gcol, gopa = torch.zeros(V, 3, device="cuda"), torch.zeros(V, 3, device="cuda"), torch.zeros(V, device="cuda")
    lam = sc.params.lambda_dep

    def map_view():
        ts.ts_project(tr.ctx, tr.scene, tr.cam, tr.prm, tr.T, tr.frame)
        ts.ts_bin_sort(tr.ctx, tr.frame)
        ts.ts_render_map_l1(tr.ctx, tr.scene, tr.frame, tr.C, tr.D, tr.A, tr.Chat, tr.Dhat, lam, tr.gC, tr.gD, tr.loss,
                            gpos, gcol, gopa, ts.GRAD_POS | ts.GRAD_COLOR | ts.GRAD_OPACITY)

    tr.reset()
    with torch.cuda.stream(stream):
        for _ in range(2):
            map_view()
        stream.synchronize()
        mrun = map_view
        if not args.no_graph:
            mg = torch.cuda.CUDAGraph()
            with torch.cuda.graph(mg, stream=stream):
                map_view()
            mrun = mg.replay
        mev = []
        for _ in range(max(10, args.steps // 2)):
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            mrun()
            b.record(stream)
            mev.append((a, b))
    stream.synchronize()
    map_ms = float(np.median([a.elapsed_time(b) for a, b in mev]))

    # e2e: same iteration through the C ABI with HOST buffers: every step the frame's target RGB-D (pinned, 16 B/pixel)
    # and the pose go up and dL/dtau and the loss come back, all inside the timed region.  The uploads run on a copy
    # stream into one of two device buffers while the previous step computes (what a tracking front-end does with the
    # next camera frame); the L2 flush of the protocol is part of every step here, on the compute stream.
    hC, hD = tr.Chat.cpu().pin_memory(), tr.Dhat.cpu().pin_memory()
    hT = tr.T0.cpu().pin_memory()
    n_e2e = args.warmup + args.steps
    h_out = torch.empty(n_e2e, 7).pin_memory()
    bufs = [(tr.Chat, tr.Dhat), (torch.empty_like(tr.Chat), torch.empty_like(tr.Dhat))]
    runs = [run]
    with torch.cuda.stream(stream):
        tr.Chat, tr.Dhat = bufs[1]
        if args.no_graph:
            def run_b():
                tr.Chat, tr.Dhat = bufs[1]
                tr.iteration()
                tr.Chat, tr.Dhat = bufs[0]
            runs.append(run_b)
        else:
            g2 = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g2, stream=stream):
                tr.iteration()
            runs.append(g2.replay)
        tr.Chat, tr.Dhat = bufs[0]
    stream.synchronize()
    tr.reset()
    copy_stream = torch.cuda.Stream()
    copied = [torch.cuda.Event() for _ in range(n_e2e)]
    done = [torch.cuda.Event() for _ in range(n_e2e)]

    def e2e_steps(i0, i1):
        for i in range(i0, i1):
            b = i & 1
            with torch.cuda.stream(copy_stream):
                if i >= 2:
                    copy_stream.wait_event(done[i - 2])           # the buffer's previous user has finished
                bufs[b][0].copy_(hC, non_blocking=True)
                bufs[b][1].copy_(hD, non_blocking=True)
                copied[i].record(copy_stream)
            with torch.cuda.stream(stream):
                flush.fill_(1)
                tr.T.copy_(hT, non_blocking=True)
                stream.wait_event(copied[i])
                runs[b]()
                h_out[i, :6].copy_(tr.tau, non_blocking=True)
                h_out[i, 6:].copy_(tr.loss, non_blocking=True)
                done[i].record(stream)

    e2e_steps(0, args.warmup)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    e2e_steps(args.warmup, n_e2e)
    torch.cuda.synchronize()
    e2e_step = (time.perf_counter() - t0) * 1e3 / args.steps
    e2e_step = max_over_ranks(dist, e2e_step, "cuda")

    value = world * HW / (ms_per_step * 1e-3) / 1e6
    p_sort = (32 + max(0, (NT - 1).bit_length()) + 7) // 8
    B, F = algorithmic_work(cnt, HW, NT, M, p_sort, "pose")
    p_fp32 = 148 * FP32_LANES_PER_SM * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12        # TFLOP/s, nominal
    t_hbm = sum(B[k] for k in STEP_ROWS) / (peaks["hbm_gbs"] * 1e9)
    t_alu = sum(F[k] for k in STEP_ROWS) / (p_fp32 * 1e12)
    t_roof = max(t_hbm, t_alu)
    in_step = ("project", "bin_sort", "render_track", "pose_reduce")          # the launches of the timed iteration
    dom = max((k for k in in_step if k in stage_ms), key=lambda k: stage_ms[k])
    dom_t = stage_ms[dom] * 1e-3
    if F[dom] / (p_fp32 * 1e12) > B[dom] / (peaks["hbm_gbs"] * 1e9):
        roof = {"bound": "alu", "kernel": dom, "achieved": F[dom] / dom_t / 1e12, "peak": p_fp32, "unit": "TFLOP/s",
                "peak_source": "nominal 148 SM x 128 FP32 lanes x 2 x sm_max_mhz (DESIGN.md section 8)"}
    else:
        roof = {"bound": "hbm", "kernel": dom, "achieved": B[dom] / dom_t / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "peak_source": peaks["src"]}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["traffic"] = load_traffic().get(dom)
    roof["algorithmic_bytes"] = B[dom]
    roof["algorithmic_flops"] = F[dom]
    roof["launch_ms"] = stage_ms[dom]

    out = {"metric": "fwd+bwd render Mpix/s", "value": value, "unit": "Mpix/s", "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f32", "data": "synthetic",
           "config": {"workload": sc.name, "faces": M, "image": [sc.cam.width, sc.cam.height], "sigma": sc.params.sigma,
                      "mode": "tracking iteration, pose-only gradients", "l2": "flushed between timed steps (256 MiB write)",
                      "cuda_graph": graph is not None},
           "clocks": clocks, "gpu_launches": Tracker.launches_per_iter * args.steps,
           "e2e": {"value": world * HW / (e2e_step * 1e-3) / 1e6, "unit": "Mpix/s", "h2d_bytes_per_step": 16 * HW + 48,
                   "d2h_bytes_per_step": 28, "ms_per_step": e2e_step,
                   "how": "K steps timed as a whole by the host clock; every step uploads its target RGB-D frame and pose from "
                          "pinned memory (copy stream, two device buffers, overlapping the previous step's kernels), flushes L2, "
                          "runs the iteration and reads dL/dtau + loss back"},
           "roofline": roof,
           "step_roofline": {"t_hbm_us": t_hbm * 1e6, "t_alu_us": t_alu * 1e6, "t_roof_us": t_roof * 1e6,
                             "frac": t_roof / (ms_per_step * 1e-3), "algorithmic_bytes": sum(B[k] for k in STEP_ROWS),
                             "algorithmic_flops": sum(F[k] for k in STEP_ROWS), "hbm_peak_gbs": peaks["hbm_gbs"], "fp32_peak_tflops": p_fp32},
           "mapping_view": {"ms": map_ms, "Mpix_per_s": HW / (map_ms * 1e-3) / 1e6,
                            "what": "project + bin/sort + ts_render_map_l1 (forward, L1, backward wrt positions, colours, "
                                    "opacities) of ONE view of this scene, one CUDA graph, L2 flushed (informational; not the "
                                    "headline metric)"},
           "tracking_iters_per_s": world * 100.0 / (frame_ms * 1e-3), "frame_100_iters_ms": frame_ms,
           "stage_ms": stage_ms, "counters": cnt, "wall_s_timed_region": t_wall}
    if rank == 0:
        if not args.no_cpu_baseline and world >= 1:
            out["cpu_baseline"] = cpu_baseline(sc)
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
