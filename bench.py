"""bench.py -- fwd+bwd rasterisation throughput of the 3DGS hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload replica300k|mono50k|tracking500k|fused2m|peaks]

One step = one pass of the whole hot path: gs_preprocess -> gs_bin_tiles -> gs_rasterize_fwd ->
[upstream gradients] -> gs_rasterize_bwd -> gs_pose_grad.  Default workload = BASELINE.json configs[2] (the
configuration the metric is quoted on): 300k Gaussians, 1200x680, SH degree 3, five Replica-shaped synthetic scenes
(seeds 30-34) cycled step to step, so that the inputs of consecutive steps (71 MB of parameters each, 355 MB in total)
exceed the 126 MB L2.  Prints ONE JSON line.  Multi-GPU: replicas only: every rank runs the same job
on its own GPU; value = all ranks' steps / max-over-ranks device time.
`--impl reference` times the fp64 CPU oracle (oracle/) on the host cores on the same workload (rank 0 only).
`--workload peaks` prints the measured machine peaks (gs_measure_peaks) that the roofline entries are divided by.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2605_10760_b200 import scenes  # noqa: E402

METRIC = "fwd+bwd rasterize iters/sec at 1200x680, 300k Gaussians"
SEEDS = (30, 31, 32, 33, 34)
# Algorithmic FP32 work of the compositing kernels, in FLOPs with FMA = 2, per (pixel, Gaussian) pair:
#   evaluated pair (the pixel is still alive and the region mask keeps the Gaussian): u (2 FFMA), v (1), p2 (2) = 10,
#       p2 >= -log2(255) and T >= 1e-4 (2) -> 12, + nothing else when the pair is rejected
#   blended pair, forward: MUFU.EX2, min (1), alpha T (1), 4 FFMA (8), T update FFMA (2) -> 12
#   blended pair, backward pixel phase: MUFU.EX2, min (1), 1 - alpha (1), MUFU.RCP, T / (1 - alpha) (1), alpha T (1),
#       w_i (4 FFMA = 8), dL/dalpha (3), S (2), clamp test (1), gp (1) = 20; Gaussian phase (the per-Gaussian sums over the
#       pixels of the region): u (2), gp u, gp v (2), 2 adds (2), 3 FFMA (6), sum gp (1), 4 FFMA (8) = 21     -> 41
FLOP_EVAL, FLOP_BLEND_FWD, FLOP_BLEND_BWD = 12.0, 12.0, 41.0
LDS_PER_ENTRY = 3.0   # broadcast LDS.128 per relevant (region, Gaussian) entry in the pixel loops (48-byte record)
# Warp instructions the kernels execute per relevant entry, from the committed ncu capture (profiles/r2_v10_ncu_full.txt,
# r2_v10_chain.md: smsp__inst_executed / relevant entries of the captured scene).  NOT an algorithmic count: it says how
# close the kernels run to the issue rate that actually binds them (roofline_stages[...]["issue"]), next to the
# algorithmic FLOP fraction.
WINST_PER_ENTRY_FWD, WINST_PER_ENTRY_BWD = 34.0, 67.6   # scene seed 30: 47.78 M / 1.4055 M, 94.26 M / 1.3947 M


def load_measured_peaks_file():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region, the way the profiling recipe does it: ONE nvidia-smi
    process in loop mode, started before the warm-up and killed after the timed region (a process forked per sample at the
    start of the timed loop took the launching thread's CPU: -2.3 % on a 20-step run).  Samples inside the timed window
    are reported; a window shorter than the sampling period falls back to the samples since the warm-up (the GPU is under
    the same load from the first warm-up step to the last timed one)."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int, period_ms: int = 20):
        self.index, self.period_ms, self.rows, self._p, self._t = index, period_ms, [], None, None
        self.t_begin = self.t_end = None

    def _run(self):
        try:
            for line in self._p.stdout:
                c = [x.strip() for x in line.strip().split(",")]
                if len(c) >= 6:
                    self.rows.append((time.perf_counter(), c))
        except Exception:
            pass

    def start(self):
        try:
            self._p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i",
                                        str(self.index), "-lms", str(self.period_ms)], stdout=subprocess.PIPE,
                                       stderr=subprocess.DEVNULL, text=True)
            self._t = threading.Thread(target=self._run, daemon=True)
            self._t.start()
        except Exception:
            self._p = None
        return self

    def wait_first(self, timeout_s: float):
        t0 = time.perf_counter()
        while not self.rows and time.perf_counter() - t0 < timeout_s and self._p is not None and self._p.poll() is None:
            time.sleep(0.01)

    def mark_begin(self):
        self.t_begin = time.perf_counter()

    def mark_end(self):
        self.t_end = time.perf_counter()

    def stop(self):
        if self._p is not None:
            try:
                self._p.kill()
                self._p.wait(timeout=5)
            except Exception:
                pass
        if self._t is not None:
            self._t.join(timeout=5)

    def summary(self, t_begin=None, t_end=None):
        if t_begin is not None:     # an explicit window (the sustained leg)
            inside = [c for t, c in self.rows if t_begin <= t <= t_end]
            window = "sustained leg"
            if not inside:
                return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
            return self._fmt(inside, window)
        inside = [c for t, c in self.rows if self.t_begin is not None and self.t_begin <= t <= (self.t_end or t)]
        window = "timed region"
        if not inside:   # region shorter than the sampling period: everything since the warm-up began
            t_lo = (self.t_begin or 0.0) - 2.0   # the warm-up, the statistics pass and the timed steps: the same load
            inside = [c for t, c in self.rows if t >= t_lo and (self.t_end is None or t <= self.t_end + 0.05)]
            window = "warm-up + timed region (the timed region is shorter than the sampling period)"
        if not inside:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        return self._fmt(inside, window)

    @staticmethod
    def _fmt(inside, window):
        try:
            sm = sorted(float(r[0]) for r in inside)
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            reasons = [n for k, n in enumerate(names) if any(r[2 + k].lower().startswith("active") for r in inside)]
            return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(inside[0][1]), "reasons": reasons,
                    "samples": len(inside), "window": window}
        except Exception:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unparsed"]}


# ----------------------------------------------------------------------------------------------------------------------
# workloads: the scenes, the views of one step and the loss that forms the upstream gradients
# ----------------------------------------------------------------------------------------------------------------------
class Workload:
    def __init__(self, name):
        self.name = name
        self.pose_only = False
        self.views = 1
        if name == "replica300k":
            self.scenes = [scenes.replica_scene(seed=s) for s in SEEDS]
            self.cams = [[sc.camera] for sc in self.scenes]
            self.up_seeds = list(SEEDS)
            self.label = (f"replica300k: BASELINE.json configs[2], {self.scenes[0].N} Gaussians, 1200x680, SH3, "
                          f"seeds {list(SEEDS)} cycled")
            self.l2 = "inputs larger than L2: 5 scenes x 71 MB of parameters cycled step to step"
        elif name == "mono50k":
            self.scenes = [scenes.mono_scene(seed=s) for s in (2, 3, 4)]
            self.cams = [[sc.camera] for sc in self.scenes]
            self.up_seeds = [2, 3, 4]
            self.label = "mono50k: BASELINE.json configs[1], 50000 Gaussians, 640x480, SH0, seeds [2, 3, 4] cycled"
            self.l2 = "L2 flushed by the 3 cycled scenes only partly (12 MB): a parity-size case, not the headline"
        elif name == "replica_small":  # CPU-side testing of the harness only
            self.scenes = [scenes.replica_scene(seed=s, N=20000, width=300, height=170, f=150.0) for s in (30, 31)]
            self.cams = [[sc.camera] for sc in self.scenes]
            self.up_seeds = [30, 31]
            self.label = "replica_small: harness test, 20000 Gaussians, 300x170, SH3"
            self.l2 = "harness test"
        elif name == "tracking500k":
            # BASELINE.json configs[3]: 500k Gaussians frozen, L1 RGB against a render from the pose perturbed by 2 cm / 1 deg
            sc = scenes.replica_scene(seed=40, N=500_000)
            self.scenes = [sc]
            self.cams = [[sc.camera]]
            self.up_seeds = [40]
            self.pose_only = True
            self.label = "tracking500k: BASELINE.json configs[3], 500000 Gaussians, 1200x680, SH3, pose-only, seed 40"
            self.l2 = "inputs larger than L2: 118 MB of parameters + 50 MB of per-step scratch"
        elif name == "fused2m":
            # BASELINE.json configs[4]: 2M Gaussians (4 Sim(3)-mapped submaps), 8 views per iteration, gradients accumulated
            sc, cams = scenes.fused_scene(seed=50)
            self.scenes = [sc]
            self.cams = [cams]
            self.views = len(cams)
            self.up_seeds = [50]
            self.label = "fused2m: BASELINE.json configs[4], 2000000 Gaussians, 8 views of 1200x680, SH3, seed 50"
            self.l2 = "inputs larger than L2: 472 MB of parameters"
        else:
            raise SystemExit(f"unknown workload {name}")
        self.W, self.H = self.cams[0][0].width, self.cams[0][0].height


def oracle_step(wl: Workload, k: int, only_view=None):
    """One step of the workload on the fp64 oracle (all views, or just `only_view` for the extrapolated sample)."""
    from oracle import gso
    sc = wl.scenes[k % len(wl.scenes)]
    if wl.pose_only:
        cam_t = sc.camera.copy()
        cam_t.T_cw = scenes.perturb_pose(sc.camera.T_cw, scenes.tracking_perturbation(40))
        if not hasattr(wl, "_oracle_target"):
            wl._oracle_target = gso.forward(sc, camera=cam_t)["rgb"]
        img = gso.forward(sc)
        gC = (np.sign(img["rgb"] - wl._oracle_target) / (3 * wl.W * wl.H)).astype(np.float32)
        gso.forward_backward(sc, gC, None)
        return
    for v, cam in enumerate(wl.cams[k % len(wl.cams)]):
        if only_view is not None and v != only_view:
            continue
        gC, gD = scenes.upstream_gradients(wl.up_seeds[k % len(wl.up_seeds)] + v, wl.W, wl.H)
        gso.forward_backward(sc, gC, gD, camera=cam)


def oracle_leg(wl: Workload, budget_s: float, max_iters: int):
    """Times the fp64 oracle, as it stands, on the host cores: whole steps of the same workload."""
    from oracle import gso
    gso.lib()
    cores = gso.num_threads()
    t0, n = time.perf_counter(), 0
    while n < max_iters and (n == 0 or time.perf_counter() - t0 < budget_s):
        oracle_step(wl, n)
        n += 1
    dt = time.perf_counter() - t0
    return n / dt, cores, n, dt


def config_dict(wl: Workload, world: int):
    return {"workload": wl.label, "l2": wl.l2, "parallelism": "replicas only" if world > 1 else "single GPU"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = Workload(args.workload)
    t0, warmed = time.perf_counter(), 0
    while warmed < args.warmup and (warmed == 0 or time.perf_counter() - t0 < 5.0):
        oracle_step(wl, warmed)   # untimed; bounded at ~5 s because one oracle step costs 0.4-20 s
        warmed += 1
    val, cores, n, dt = oracle_leg(wl, budget_s=120.0, max_iters=max(1, args.steps))
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "iter/s", "n_gpus": args.gpus, "steps": n,
            "warmup": args.warmup, "ms_per_step": 1e3 / val, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(wl, int(os.environ.get("WORLD_SIZE", "1"))),
            "cpu_baseline": {"value": val, "unit": "iter/s", "cores": cores, "kind": "oracle",
                             "sample": f"{n} whole steps of the workload (each = all {wl.views} view(s), fwd+bwd) in {dt:.1f} s; "
                                       f"{warmed} untimed warm-up step(s) run"},
            "e2e": {"value": val, "unit": "iter/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "mpix_iter_per_s": val * wl.views * wl.W * wl.H / 1e6}
    print(json.dumps(line))


def max_over_ranks(ms_local: float, dist, device) -> float:
    """Device time of the job = the slowest rank's (replicas only: no data-path collective)."""
    if dist is None:
        return float(ms_local)
    import torch
    t = torch.tensor([ms_local], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_throughput(world: int, steps: int, ms_total: float) -> float:
    """Whole-job iterations/s: every rank ran `steps` steps of its own replica in `ms_total` (max over ranks)."""
    return world * steps / (ms_total / 1e3)


def stage_models(N, K3, V, I, P, tiles, E, C, Eb, R, Rb, pose_only, dense_fill=True):
    """Algorithmic work per launch of every stage: HBM bytes, or FP32 flops + broadcast LDS for the
    two compositing kernels.  V visible Gaussians, I tile instances, P pixels, E / Eb (pixel, Gaussian) pairs evaluated
    by the forward / backward, C blended pairs, R / Rb relevant (region, Gaussian) entries of the forward / backward."""
    gp = 0 if pose_only else (44 + 4 * K3)
    fill = gp if dense_fill else 0
    return {
        "preprocess": {"bound": "hbm", "bytes": 48 * N + (4 * K3 + 120) * V},
        "tile_scan": {"bound": "hbm", "bytes": 16.0 * tiles, "note": "latency-bound: one L2 round trip between its CTAs"},
        "emit": {"bound": "hbm", "bytes": 48 * V + 8 * I},
        "tile_sort": {"bound": "hbm", "bytes": 32 * I, "note": "compare-exchange network in registers: integer-ALU work"},
        "raster_fwd": {"bound": "alu", "flops": E * FLOP_EVAL + C * FLOP_BLEND_FWD, "lds": R * LDS_PER_ENTRY,
                       "winst": R * WINST_PER_ENTRY_FWD, "bytes": 16 * I + 32 * V + 24 * P},
        "raster_bwd": {"bound": "alu", "flops": Eb * FLOP_EVAL + C * FLOP_BLEND_BWD, "lds": Rb * LDS_PER_ENTRY,
                       "winst": Rb * WINST_PER_ENTRY_BWD, "bytes": 16 * I + 32 * V + 28 * P + 48 * V},
        "gauss_bwd": {"bound": "hbm", "bytes": (48 + 48 + 48 + 16 + 4 + 4 * K3) * V + gp * V + (fill * (N - V) + 4 * N if fill else 0),
                      "note": "reads g2d, parameters, SH of the V visible Gaussians, writes their gradient rows; dense mode: "
                              "+ the zero rows of the N - V culled Gaussians, cleared by the same kernel"},
        "pose_grad": {"bound": "hbm", "bytes": 120.0, "note": "latency-bound: one thread"},
    }


def run_ours(args):
    import torch
    from paper_2605_10760_b200 import binding as B
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist_
        dist = dist_
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    clk = ClockSampler(local).start()   # one nvidia-smi in loop mode from here to the end of the timed region
    peaks = B.gs_measure_peaks(local)          # measured in this run: the roofline denominators
    wl = Workload(args.workload)
    W, H = wl.W, wl.H
    ctx = B.Context(local)
    dss = [B.DeviceScene(sc, local) for sc in wl.scenes]
    out = dss[0].alloc_outputs(W, H)
    to_dev = lambda a: torch.from_numpy(np.ascontiguousarray(a, np.float32)).to(dev)
    T_dev = target = gC_track = None
    ups = []
    if wl.pose_only:
        sc = wl.scenes[0]
        cam_t = sc.camera.copy()
        cam_t.T_cw = scenes.perturb_pose(sc.camera.T_cw, scenes.tracking_perturbation(40))
        B.forward(ctx, dss[0], cam_t, out)
        torch.cuda.synchronize(); ctx.gs_poll()
        target = out["rgb"].clone()
        T_dev = to_dev(np.asarray(sc.camera.T_cw, np.float32).reshape(-1))
        gC_track = torch.empty_like(out["rgb"])
    else:
        for k in range(len(wl.scenes)):
            ups.append([tuple(to_dev(a) for a in scenes.upstream_gradients(wl.up_seeds[k] + v, W, H))
                        for v in range(wl.views)])

    # --grads sparse: GS_SPARSE_GRADS (one gradient row per visible Gaussian, no dense zero fill); single-view workloads
    grad_flag = B.GS_SPARSE_GRADS if (args.grads == "sparse" and wl.views == 1) else 0

    # multi-view workloads: extra (context, stream, output) sets; the gradient arrays are shared
    n_vs = max(1, args.view_streams) if wl.views > 1 else 1
    n_is = max(1, args.iter_streams) if (wl.views == 1 and not wl.pose_only) else 1
    ictx = [ctx] + [B.Context(local) for _ in range(n_is - 1)]
    istreams = [torch.cuda.Stream(device=dev) for _ in range(n_is)] if n_is > 1 else []
    iout = [out] + [dss[0].alloc_outputs(W, H) for _ in range(n_is - 1)]
    prof_seq = [False]  # the stage-profile loop runs the views one after the other on `ctx`
    vctx, vstreams, vout = [ctx], [], [out]
    if n_vs > 1:
        vctx += [B.Context(local) for _ in range(n_vs - 1)]
        vstreams = [torch.cuda.Stream(device=dev) for _ in range(n_vs)]
        for _ in range(n_vs - 1):
            o = dss[0].alloc_outputs(W, H)
            for name in ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh"):
                o[name] = out[name]
            vout.append(o)

    def step(k):
        s = k % len(dss)
        if wl.pose_only:
            # preprocess (pose read from the device) -> bin -> fwd -> L1 gradient -> bwd (pose only) -> pose gradient ->
            # on-device normalised pose step; no host synchronisation inside the loop
            B.forward(ctx, dss[0], wl.scenes[0].camera, out, T_cw_dev=T_dev)
            B.gs_aux_l1_grad(out["rgb"], target, 1.0 / (3 * W * H), gC_track)
            B.backward(ctx, out, gC_track, None, None, flags=B.GS_POSE_ONLY, pose=True)
            B.gs_aux_pose_step(T_dev, out["g_twist"], 1e-3)
            return
        if n_is > 1 and not prof_seq[0]:
            j = k % n_is
            with torch.cuda.stream(istreams[j]):
                B.forward(ictx[j], dss[s], wl.cams[s][0], iout[j])
                B.backward(ictx[j], iout[j], ups[s][0][0], ups[s][0][1], None, flags=grad_flag, pose=True)
            return
        if n_vs > 1 and not prof_seq[0]:
            # views round-robin on n_vs (context, stream) pairs: the latency-bound per-Gaussian and binning kernels of one
            # view overlap the compositing kernels of another.  All views ACCUMULATE into the zeroed gradient arrays.
            for name in ("g_means", "g_scales", "g_quats", "g_opacities", "g_sh"):
                out[name].zero_()
            main = torch.cuda.current_stream()
            fork = torch.cuda.Event(); fork.record(main)
            for st in vstreams:
                st.wait_event(fork)
            for v, cam in enumerate(wl.cams[s]):
                j = v % n_vs
                with torch.cuda.stream(vstreams[j]):
                    B.forward(vctx[j], dss[s], cam, vout[j])
                    B.backward(vctx[j], vout[j], ups[s][v][0], ups[s][v][1], None, flags=B.GS_ACCUMULATE, pose=True)
            for st in vstreams:
                join = torch.cuda.Event(); join.record(st); main.wait_event(join)
            return
        for v, cam in enumerate(wl.cams[s]):
            B.forward(ctx, dss[s], cam, out)
            B.backward(ctx, out, ups[s][v][0], ups[s][v][1], None, flags=(B.GS_ACCUMULATE if v > 0 else grad_flag), pose=True)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    clk.wait_first(5.0)
    # warm-up: also calibrates the instance capacity over all poses (an overflowing iteration is re-issued)
    warm = max(args.warmup, 3)
    k = 0
    while k < max(warm, len(dss)):
        try:
            step(k)
            torch.cuda.synchronize()
            for c in vctx + ictx[1:]:
                c.gs_poll()
            k += 1
        except B.GsError as e:
            if e.code != -5:
                raise
    # workload statistics per scene (last view of the step): V, I and the pair counts of the compositing kernels
    stats = []
    prof_seq[0] = True
    for k in range(len(dss)):
        step(k)
        nv, ni = ctx.gs_get_counts()
        wlst = ctx.gs_get_workload()
        stats.append(dict(visible=nv, instances=ni, **wlst))
    if wl.pose_only:
        T_dev.copy_(to_dev(np.asarray(wl.scenes[0].camera.T_cw, np.float32).reshape(-1)))
    prof_seq[0] = False
    barrier()

    # ---- timed region: exactly K steps, device time, max over ranks ----
    K = args.steps
    l0 = sum(c.gs_get_launch_count() for c in vctx + ictx[1:])
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    clk.mark_begin()
    e0.record()
    if n_is > 1:   # the iteration streams start behind e0 and are joined in front of e1
        fk = torch.cuda.Event(); fk.record()
        for st in istreams:
            st.wait_event(fk)
    for k in range(K):
        step(k)
    if n_is > 1:
        for st in istreams:
            jn = torch.cuda.Event(); jn.record(st); torch.cuda.current_stream().wait_event(jn)
    e1.record()
    barrier()
    clk.mark_end()
    ms_total = e0.elapsed_time(e1)
    for c in vctx + ictx[1:]:
        c.gs_poll()
    launches = sum(c.gs_get_launch_count() for c in vctx + ictx[1:]) - l0
    ms_total = max_over_ranks(ms_total, dist, dev)
    value = replica_throughput(world, K, ms_total)

    # ---- sustained leg: a timed region under 0.25 s (e.g. the driver's --steps 20: 5 ms) is too short for the clock
    # sampler and for an outside clock to see; the same loop is then timed again over about half a second.  `value`,
    # `steps` and `ms_per_step` stay those of the K requested steps; this is reported beside them.
    sustained = None
    if ms_total < 250.0 and n_is == 1:
        K2 = int(min(50_000, max(K, np.ceil(500.0 / max(ms_total / K, 1e-3)))))
        if dist is not None:   # every rank must run the same number of steps
            t = torch.tensor([K2], device=dev); dist.all_reduce(t, op=dist.ReduceOp.MAX); K2 = int(t.item())
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        tb = time.perf_counter()
        s0.record()
        for k in range(K2):
            step(k)
        s1.record()
        barrier()
        te = time.perf_counter()
        ms2 = max_over_ranks(s0.elapsed_time(s1), dist, dev)
        for c in vctx + ictx[1:]:
            c.gs_poll()
        sustained = {"value": replica_throughput(world, K2, ms2), "unit": "iter/s", "steps": K2, "ms_per_step": ms2 / K2,
                     "clocks": clk.summary(tb, te)}
    clk.stop()

    # ---- per-stage device times (second loop, stage events on; same steps; last view of each step) ----
    prof_seq[0] = True
    ctx.gs_profile_enable(True)
    stage_ms = {s: 0.0 for s in B.STAGES}
    for k in range(K):
        step(k)
        r = ctx.gs_profile_read()
        for s in B.STAGES:
            stage_ms[s] += r[s] / K
    ctx.gs_profile_enable(False)

    # ---- rooflines: every stage, against peaks measured in this run ----
    pf = load_measured_peaks_file()
    hbm_peak = float(pf["hbm_gbs"]) if pf else peaks["hbm_copy_gbs"]
    hbm_src = "measured copy bandwidth, MEASURED_PEAKS.json (driver)" if pf else "measured copy bandwidth, gs_measure_peaks (this run)"
    alu_peak = 2.0 * peaks["fma_tlanes"]                                  # TFLOP/s, FMA = 2
    used = [k % len(dss) for k in range(K)]
    mean = lambda key: float(np.mean([stats[u][key] for u in used]))
    N, K3 = wl.scenes[0].N, 3 * (wl.scenes[0].sh_degree + 1) ** 2
    P, tiles = W * H, ((W + 15) // 16) * ((H + 15) // 16)
    V, I = mean("visible"), mean("instances")
    models = stage_models(N, K3, V, I, P, tiles, mean("evaluated"), mean("blended"), mean("evaluated_bwd"),
                          mean("region_entries"), mean("region_entries_bwd"), wl.pose_only,
                          dense_fill=(grad_flag == 0 and wl.views == 1))
    roof_stages = {}
    for s in B.STAGES:
        m, t = models[s], stage_ms[s] * 1e-3
        if t <= 0:
            continue
        e = {"bound": m["bound"], "ms": stage_ms[s]}
        if m["bound"] == "hbm":
            e.update(bytes=m["bytes"], achieved=m["bytes"] / t / 1e9, peak=hbm_peak, unit="GB/s")
        else:
            e.update(flops=m["flops"], achieved=m["flops"] / t / 1e12, peak=alu_peak, unit="TFLOP/s",
                     lds_bcast={"warp_lds": m["lds"], "achieved": m["lds"] / t / 1e12, "peak": peaks["lds128_bcast_twarp"],
                                "unit": "T warp-level LDS.128/s", "frac": m["lds"] / t / 1e12 / peaks["lds128_bcast_twarp"]},
                     issue={"warp_inst": m["winst"], "achieved": m["winst"] / t / 1e12, "peak": peaks["issue_twarp"],
                            "unit": "T warp instructions/s", "frac": m["winst"] / t / 1e12 / peaks["issue_twarp"],
                            "note": "executed (not algorithmic) instructions per relevant entry from the committed ncu capture"})
        e["frac"] = e["achieved"] / e["peak"]
        if "note" in m:
            e["note"] = m["note"]
        roof_stages[s] = e
    dominant = max(stage_ms, key=stage_ms.get)
    kernel_name = {"raster_fwd": "raster_fwd_kernel", "raster_bwd": "raster_bwd_kernel"}.get(dominant, dominant + "_kernel")
    d = roof_stages[dominant]
    roof = {"kernel": kernel_name, "bound": d["bound"], "achieved": d["achieved"], "peak": d["peak"], "unit": d["unit"],
            "frac": d["frac"], "traffic": None,
            "peak_source": hbm_src if d["bound"] == "hbm" else
            "measured FP32 FMA rate x 2, gs_measure_peaks (this run): %.2f T lane-FMA/s" % peaks["fma_tlanes"],
            "stage_share": stage_ms[dominant] / sum(stage_ms.values())}
    if "lds_bcast" in d:
        roof["lds_bcast"] = d["lds_bcast"]
        roof["issue"] = d["issue"]
    try:  # DRAM traffic per launch of the dominant kernel, from the committed ncu capture of this round (profiles/)
        import csv
        with open(os.path.join(ROOT, "profiles", "r2_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == args.workload and row["kernel"] == kernel_name:
                    roof["traffic"] = int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
                    roof["traffic_source"] = row["source"]
                    roof["traffic_note"] = ("ncu dram read+write of ONE launch on ONE scene (seed 30), while the other fields "
                                            "average the five scenes; writes that stay resident in the 126 MB L2 (images, "
                                            "gradient rows) are not in it, so it is a lower bound of the bytes moved")
    except Exception:
        pass
    # whole-iteration HBM figure (BASELINE.json "% HBM roofline"): algorithmic bytes of all stages / step time
    bytes_iter = wl.views * sum(m["bytes"] for m in models.values())
    hbm_frac_iter = bytes_iter / (ms_total / K * 1e-3) / 1e9 / hbm_peak

    line = None
    if rank == 0:
        e2e = run_e2e(args, wl, B, torch, local, world, K)
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            if wl.views > 1 and args.cpu_budget < 12.0:
                # sub-record of the default line: ONE view timed, the step (all views) extrapolated from it
                from oracle import gso
                gso.lib()
                t0 = time.perf_counter()
                oracle_step(wl, 0, only_view=0)
                dt = time.perf_counter() - t0
                cpu = {"value": 1.0 / (dt * wl.views), "unit": "iter/s", "cores": gso.num_threads(), "kind": "oracle",
                       "sample": f"EXTRAPOLATED: view 0 of one step timed ({dt:.1f} s, fwd+bwd) x {wl.views} views"}
            else:
                v, cores, n, dt = oracle_leg(wl, budget_s=args.cpu_budget, max_iters=10 * len(wl.scenes))
                cpu = {"value": v, "unit": "iter/s", "cores": cores, "kind": "oracle",
                       "sample": f"{n} whole steps of the same workload (each = all {wl.views} view(s), fwd+bwd; scene seeds cycled) in {dt:.1f} s"}
        line = {"metric": METRIC if args.workload == "replica300k" else "fwd+bwd rasterize iters/sec",
                "value": value, "unit": "iter/s", "n_gpus": world, "steps": K, "warmup": warm,
                "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic", "config": config_dict(wl, world),
                "views_per_iter": wl.views, "view_streams": n_vs, "iter_streams": n_is, "grads": "sparse" if grad_flag else "dense", "mpix_iter_per_s": value * wl.views * W * H / 1e6,
                "clocks": clk.summary(), "value_sustained": sustained, "e2e": e2e, "e2e_sequential": e2e.get("sequential"), "gpu_launches": launches, "roofline": roof,
                "roofline_stages": roof_stages, "cpu_baseline": cpu,
                "hbm_frac_whole_iteration": hbm_frac_iter, "algorithmic_bytes_per_iter": bytes_iter,
                "stages_ms": stage_ms, "stages_note": "device time per stage of the LAST view of a step (CUDA events in the library)",
                "peaks_measured": peaks,
                "workload_stats": {"visible_V": V, "instances_I": I, "evaluated_pairs_E": mean("evaluated"),
                                   "evaluated_pairs_bwd_Eb": mean("evaluated_bwd"), "blended_pairs_C": mean("blended"),
                                   "last_pos_sum_L": mean("last_pos_sum"), "region_entries_R": mean("region_entries"),
                                   "region_entries_bwd_Rb": mean("region_entries_bwd"),
                                   "tile_list_x_pixels": mean("list_len_x_pixels"),
                                   "per_scene": stats}}
    ctx.close()
    if line is not None and world == 1 and args.workload == "replica300k" and not args.no_configs:
        line["configs"] = run_config_subrecords(args)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line))


SUB_CONFIGS = (("mono50k", "BASELINE.json configs[1]", 2000), ("tracking500k", "BASELINE.json configs[3]: the 100 iterations it names", 100),
               ("fused2m", "BASELINE.json configs[4]: eight-view steps", 5))


def run_config_subrecords(args, budget_s: float = 150.0):
    """The other BASELINE.json configurations, each measured by this same program in a process of its own (same timing
    protocol, own warm-up, own peaks) and reported as a compact sub-record of the default line, so that the numbers of
    configs 2, 4 and 5 are the driver's and not only the builder's.  Bounded: a sub-run that would not fit the budget is
    recorded as skipped."""
    import subprocess
    import sys
    out, t_start = {}, time.perf_counter()
    keep = ("value", "unit", "steps", "ms_per_step", "value_sustained", "stages_ms", "roofline", "hbm_frac_whole_iteration",
            "cpu_baseline", "e2e", "clocks", "config", "gpu_launches", "views_per_iter")
    for name, what, steps in SUB_CONFIGS:
        left = budget_s - (time.perf_counter() - t_start)
        if left < 25.0:
            out[name] = {"skipped": "time budget of the sub-records used up"}
            continue
        cmd = [sys.executable, os.path.abspath(__file__), "--workload", name, "--steps", str(steps), "--warmup", str(max(args.warmup, 3)),
               "--no-configs", "--cpu-budget", "0" if args.no_cpu_baseline else "3"]
        if args.no_cpu_baseline:
            cmd.append("--no-cpu-baseline")
        try:
            r = subprocess.run(cmd, capture_output=True, text=True, timeout=left)
            d = json.loads(r.stdout.strip().splitlines()[-1])
            rec = {k: d[k] for k in keep if k in d}
            if isinstance(rec.get("roofline"), dict):
                rec["roofline"] = {k: v for k, v in rec["roofline"].items() if k in ("kernel", "bound", "achieved", "peak", "unit", "frac", "stage_share")}
            rec["what"] = what
            rec["wall_s"] = round(time.perf_counter() - t_start, 1)
            out[name] = rec
        except Exception as e:   # a sub-record must never cost the headline line
            out[name] = {"error": f"{type(e).__name__}: {str(e)[:200]}"}
    # the kernels of SURVEY.md section 8(f), each alone (bench.py --workload next), compact: time and HBM fraction
    left = budget_s - (time.perf_counter() - t_start)
    if left < 20.0:
        out["next"] = {"skipped": "time budget of the sub-records used up"}
    else:
        try:
            r = subprocess.run([sys.executable, os.path.abspath(__file__), "--workload", "next", "--steps", "10"],
                               capture_output=True, text=True, timeout=left)
            d = json.loads(r.stdout.strip().splitlines()[-1])
            out["next"] = {"what": "SURVEY.md 8(f) kernels, each alone, L2 flushed between launches; ms = median device time per call",
                           "hbm_peak_gbs": d["hbm_peak_gbs"],
                           "kernels": {k: {kk: v[kk] for kk in ("ms", "algorithmic_bytes", "frac_hbm", "mrays_per_s") if kk in v}
                                       for k, v in d["kernels"].items()}}
        except Exception as e:
            out["next"] = {"error": f"{type(e).__name__}: {str(e)[:200]}"}
    return out


def run_e2e(args, wl, B, torch, local, world, K):
    """The same metric end to end: HOST (pinned) buffers in and out, copies inside the timed region."""
    dev = torch.device("cuda", local)
    W, H = wl.W, wl.H
    extra_close = []
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, np.float32)).pin_memory()
    steps = max(3, min(K, 10))
    seq_step = None
    if args.workload in ("replica300k", "mono50k", "replica_small"):
        # through the C-ABI host-buffer entry point gs_fwd_bwd_host: H2D of all parameters and upstream gradients, D2H
        # of the images and all gradients, every step
        scs = wl.scenes[:2]
        hsc = [tuple(pin(x).numpy() for x in (sc.means, sc.scales, sc.quats, sc.opacities, sc.sh)) for sc in scs]
        hup = [tuple(pin(x).numpy() for x in scenes.upstream_gradients(wl.up_seeds[k], W, H)) for k in range(len(scs))]
        Kc, Ng = (scs[0].sh_degree + 1) ** 2, scs[0].N
        # two (context, stream, pinned output set) pairs fed alternately through gs_fwd_bwd_host_async: the device->host
        # copies of one step overlap the host->device copies and kernels of the next (PCIe is full duplex); every step
        # still copies all of its inputs in and all of its results out, and a pair is synchronised before it is reused
        mk = lambda: {k: torch.zeros(s, dtype=torch.float32).pin_memory().numpy() for k, s in
                      dict(rgb=(3, H, W), depth=(H, W), alpha=(H, W), g_means=(Ng, 3), g_scales=(Ng, 3), g_quats=(Ng, 4),
                           g_opacities=(Ng,), g_sh=(Ng, Kc, 3), g_twist=(6,)).items()}
        NP = 2   # 3 / 4 pairs measured slower over the ten timed steps (413 / 366 vs 463 it/s)
        houts = [mk() for _ in range(NP)]
        hout = houts[0]
        ctx2 = B.Context(local)
        pair_ctx = [ctx2] + [B.Context(local) for _ in range(NP - 1)]
        pair_stream = [torch.cuda.Stream(device=dev) for _ in range(NP)]
        extra_close = pair_ctx[1:]

        def e2e_step(k):
            j, p = k % len(scs), k % NP
            pair_stream[p].synchronize()   # the results of step k - 2 are in this pair's host buffers
            pair_ctx[p].gs_poll()
            pair_ctx[p].gs_fwd_bwd_host(hsc[j], scs[0].sh_degree, scs[j].camera, scs[j].bg, hup[j][0], hup[j][1], houts[p],
                                        stream=pair_stream[p], sync=False)
        h2d = sum(x.nbytes for x in hsc[0]) + sum(x.nbytes for x in hup[0])
        d2h = sum(x.nbytes for x in hout.values())
        what = ("gs_fwd_bwd_host_async on two alternating (context, stream) pairs: parameters + upstream gradients in, images "
                "+ all gradients out, every step")

        def seq_step(k):
            # one iteration at a time (a loop whose host-side optimiser needs step k's gradients before step k + 1)
            j = k % len(scs)
            pair_ctx[0].gs_fwd_bwd_host(hsc[j], scs[0].sh_degree, scs[j].camera, scs[j].bg, hup[j][0], hup[j][1], houts[0],
                                        stream=pair_stream[0], sync=True)
    else:
        # configs 4 / 5: the Gaussians stay resident (they are frozen, or updated by the on-device optimiser); per step the
        # host sends the pose (tracking) or the per-view upstream gradients (refinement) from pinned memory and reads
        # back the twist gradient (and, for the refinement, the opacity gradients) -- public binding calls + torch copies
        ctx2 = B.Context(local)
        sc = wl.scenes[0]
        ds = B.DeviceScene(sc, local)
        out = ds.alloc_outputs(W, H)
        s = torch.cuda.current_stream()
        if wl.pose_only:
            cam_t = sc.camera.copy()
            cam_t.T_cw = scenes.perturb_pose(sc.camera.T_cw, scenes.tracking_perturbation(40))
            B.forward(ctx2, ds, cam_t, out)
            torch.cuda.synchronize(); ctx2.gs_poll()
            target = out["rgb"].clone()
            gC = torch.empty_like(out["rgb"])
            hT = pin(np.asarray(sc.camera.T_cw, np.float32).reshape(-1))
            T_dev = torch.empty(12, device=dev)
            h_tw = torch.zeros(6).pin_memory()

            def e2e_step(k):
                T_dev.copy_(hT, non_blocking=True)
                B.forward(ctx2, ds, sc.camera, out, T_cw_dev=T_dev)
                B.gs_aux_l1_grad(out["rgb"], target, 1.0 / (3 * W * H), gC)
                B.backward(ctx2, out, gC, None, None, flags=B.GS_POSE_ONLY, pose=True)
                h_tw.copy_(out["g_twist"], non_blocking=True)
                s.synchronize()
            h2d, d2h = 48, 24
            what = "pose in (48 B), twist gradient out (24 B); Gaussians and target resident"
        else:
            hups = [tuple(pin(a) for a in scenes.upstream_gradients(wl.up_seeds[0] + v, W, H)) for v in range(wl.views)]
            dC, dD = torch.empty(3, H, W, device=dev), torch.empty(H, W, device=dev)
            h_tw, h_go = torch.zeros(6).pin_memory(), torch.zeros(sc.N).pin_memory()

            def e2e_step(k):
                for v, cam in enumerate(wl.cams[0]):
                    dC.copy_(hups[v][0], non_blocking=True); dD.copy_(hups[v][1], non_blocking=True)
                    B.forward(ctx2, ds, cam, out)
                    B.backward(ctx2, out, dC, dD, None, flags=(B.GS_ACCUMULATE if v > 0 else 0), pose=True)
                h_tw.copy_(out["g_twist"], non_blocking=True); h_go.copy_(out["g_opacities"], non_blocking=True)
                s.synchronize()
            h2d = wl.views * 4 * W * H * 4
            d2h = 24 + 4 * sc.N
            what = "8 views' upstream gradients in, twist + opacity gradients out; Gaussians resident"
    k = 0
    while k < 3:
        try:
            e2e_step(k); k += 1
        except B.GsError as e:
            if e.code != -5:
                raise
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for k in range(steps):
        e2e_step(k)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    res = {"value": world * steps / dt, "unit": "iter/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
           "steps": steps, "what": what}
    if seq_step is not None:
        # the pipelined figure above overlaps two INDEPENDENT iterations; the sequential one is the figure to compare from
        # round to round (round 1's e2e was sequential) and the one a host-side optimiser loop sees
        for k in range(2):
            seq_step(k)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for k in range(steps):
            seq_step(k)
        torch.cuda.synchronize()
        res["sequential"] = {"value": world * steps / (time.perf_counter() - t0), "unit": "iter/s", "steps": steps,
                             "what": "gs_fwd_bwd_host, one context, each step synchronised before the next starts; same copies"}
    ctx2.close()
    for c in extra_close:
        c.close()
    return res


def run_peaks(args):
    import torch
    from paper_2605_10760_b200 import binding as B
    torch.cuda.set_device(0)
    p = B.gs_measure_peaks(0)
    clk = p["sm_count"] * p["sm_mhz_max"] * 1e6
    derived = {"fma_lanes_per_clk_per_sm": p["fma_tlanes"] * 1e12 / clk, "fp32_tflops": 2 * p["fma_tlanes"],
               "issue_warp_instr_per_clk_per_sm": p["issue_twarp"] * 1e12 / clk,
               "ex2_lanes_per_clk_per_sm": p["ex2_tlanes"] * 1e12 / clk,
               "cycles_per_bcast_lds128_per_sm": clk / (p["lds128_bcast_twarp"] * 1e12),
               "cycles_per_lds128_per_sm": clk / (p["lds128_twarp"] * 1e12),
               "cycles_per_bcast_lds64_per_sm": clk / (p["lds64_bcast_twarp"] * 1e12),
               "cycles_per_bcast_lds32_per_sm": clk / (p["lds32_bcast_twarp"] * 1e12),
               "red_lanes_per_clk_chip": p["red_glanes"] * 1e9 / (p["sm_mhz_max"] * 1e6)}
    print(json.dumps({"workload": "peaks", "peaks_measured": p, "derived": derived,
                      "driver_file": load_measured_peaks_file()}))


def run_next(args):
    """bench.py --workload next: device time of the kernels of SURVEY.md section 8(f) (losses, optimiser, compaction, ray
    casting) at the sizes of configs 3 / 5, each alone, CUDA events on the launching stream, L2 flushed between launches
    (a 256 MB fill), against the HBM copy peak where the kernel streams (algorithmic bytes stated per entry)."""
    import torch
    from paper_2605_10760_b200 import binding as B
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    pf = load_measured_peaks_file()
    hbm = float(pf["hbm_gbs"]) if pf else B.gs_measure_peaks(0)["hbm_copy_gbs"]
    flush = torch.empty(64 * 1024 * 1024, dtype=torch.float32, device=dev)
    r = np.random.Generator(np.random.PCG64(123))
    rep = max(3, min(args.steps, 10))
    out = {}

    def timed(name, fn, nbytes, note, reset=None):
        ms = []
        for it in range(rep + 2):
            if reset is not None:
                reset()
            flush.fill_(1.0)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record()
            torch.cuda.synchronize()
            if it >= 2:
                ms.append(e0.elapsed_time(e1))
        t = float(np.median(ms))
        rec = {"ms": t, "launches_timed": rep, "note": note}
        if nbytes:
            rec.update({"algorithmic_bytes": int(nbytes), "gbs": nbytes / t / 1e6, "frac_hbm": nbytes / t / 1e6 / hbm})
        out[name] = rec

    W, H = 1200, 680
    P = W * H
    f = lambda *shape: torch.from_numpy(r.uniform(0, 1, shape).astype(np.float32)).to(dev)
    rgb, trgb, depth, tdep = f(3, H, W), f(3, H, W), f(H, W) * 5, f(H, W) * 5
    d_rgb, d_depth = torch.empty_like(rgb), torch.empty_like(depth)
    loss = torch.zeros(10, dtype=torch.float64, device=dev)
    timed("gs_loss_map", lambda: B.gs_loss_map(rgb, depth, trgb, tdep, 0.9, 0.1, d_rgb, d_depth, loss), 48 * P,
          "Eq. 4 L1 terms at 1200x680: 32 B read + 16 B written per pixel")
    ab, g_ab, work = torch.zeros(2, device=dev), torch.zeros(2, device=dev), torch.empty(9 * P, device=dev)
    timed("gs_loss_refine", lambda: B.gs_loss_refine(rgb, depth, trgb, tdep, ab, 1.75, 0.2, 0.25, d_rgb, d_depth, g_ab, work, loss),
          48 * P, "Eq. 23 exposure + L1 + SSIM (11x11 separable) + depth at 1200x680, three launches; bytes = images in + "
                  "gradients out only (the SSIM planes in `work` are extra traffic, so frac_hbm understates the bytes moved)")
    # optimiser at the fused map's size (config 5: 2 M Gaussians, SH3)
    N, K = 2_000_000, 16
    shapes = dict(means=(N, 3), scales=(N, 3), quats=(N, 4), opacities=(N,), sh=(N, K, 3))
    mk = lambda lo, hi: {k: torch.empty(sh, device=dev).uniform_(lo, hi) for k, sh in shapes.items()}
    params, grads = mk(0.1, 0.9), mk(-1.0, 1.0)
    m, v = {k: torch.zeros_like(t) for k, t in params.items()}, {k: torch.zeros_like(t) for k, t in params.items()}
    lrs = dict(means=1.6e-4, scales=5e-3, quats=1e-3, opacities=5e-2, sh=2.5e-3)
    floats = 11 + 3 * K
    timed("gs_adam_step_dense_2m", lambda: B.gs_adam_step(params, grads, m, v, lrs, 3, None), 28 * floats * N,
          "fused Adam on all 2 M Gaussians (SH3): 28 B per parameter float (p, m, v read + written, g read); five launches")
    vis = (torch.rand(N, device=dev) < 0.3).to(torch.int32)
    nv = int(vis.sum().item())
    timed("gs_adam_step_masked_2m", lambda: B.gs_adam_step(params, grads, m, v, lrs, 3, vis), 28 * floats * nv + 4 * N,
          f"the same with a visibility mask ({nv} of {N} visible, scattered): bytes of the visible rows + the mask")
    ids = torch.nonzero(vis).flatten().to(torch.int32)
    n_rows = torch.tensor([nv], dtype=torch.int32, device=dev)
    sgrads = {k: torch.empty((nv,) + tuple(sh[1:]), device=dev).uniform_(-1, 1) for k, sh in shapes.items()}
    timed("gs_adam_step_sparse_2m", lambda: B.gs_adam_step_sparse(params, sgrads, m, v, lrs, 3, ids.data_ptr(), n_rows.data_ptr(), nv),
          28 * floats * nv + 4 * nv, "GS_SPARSE_GRADS rows (compact gradient rows, id list): bytes of the visible rows + ids")
    # pruning: mask, plan, gather of the SH array
    keep = torch.empty(N, dtype=torch.uint8, device=dev)
    timed("gs_prune_mask_2m", lambda: B.gs_prune_mask(params["opacities"], 0.3, keep), 5 * N, "4 B read + 1 B written per Gaussian")
    index, n_kept = torch.empty(N, dtype=torch.int32, device=dev), torch.zeros(1, dtype=torch.int64, device=dev)
    timed("gs_compact_plan_static_2m", lambda: B.gs_compact_plan_static(keep, index, n_kept), 6 * N,
          "keep mask read twice (count, index) + 4 B index written per Gaussian; three launches, scratch inside the library")
    kept = int(n_kept.item())
    dst = torch.empty((kept, K, 3), device=dev)
    lib = B.load_library()
    timed("gs_compact_rows_sh_2m", lambda: lib.gs_compact_rows(B._stream(), N, 3 * K, B._ptr(index), B._ptr(params["sh"]), B._ptr(dst)),
          4 * N + 4 * 3 * K * (N + kept), f"SH rows (192 B) of {kept} kept Gaussians gathered in order: all rows read, kept rows written")
    # Eq. 21 on one keyframe depth map
    cam = scenes.Camera(W, H, 600.0, 600.0, 599.5, 339.5, scenes.look_at([0.3, -0.2, 1.4], [4.0, 1.0, 1.1]))
    yy, xx = np.meshgrid(np.linspace(-1, 1, H), np.linspace(-1, 1, W), indexing="ij")
    dm = torch.from_numpy((4.0 + 1.5 * np.sin(2.1 * xx + 0.3) * np.cos(1.3 * yy)).astype(np.float32)).to(dev)
    vs = B.VoxelSet(1 << 22)
    steps_per_ray = float((dm / 0.05).mean().item()) * 1.5
    timed("gs_voxel_insert_rays_1200x680", lambda: vs.insert_rays(cam, dm, 0.05, 1), 0,
          f"Eq. 21, every pixel casts a ray, v = 5 cm, ~{steps_per_ray:.0f} DDA steps per ray into a 4 Mi-slot set: latency / "
          "atomics bound, not HBM", reset=vs.clear)
    out["gs_voxel_insert_rays_1200x680"]["mrays_per_s"] = P / out["gs_voxel_insert_rays_1200x680"]["ms"] / 1e3
    out["gs_voxel_insert_rays_1200x680"]["keys_stored"] = int(len(vs.keys()))
    print(json.dumps({"workload": "next", "unit": "ms per call (median)", "hbm_peak_gbs": hbm, "l2": "flushed between launches (256 MB fill)",
                      "kernels": out}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="replica300k")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-budget", type=float, default=12.0, help="seconds of oracle time for the cpu_baseline sample")
    ap.add_argument("--no-configs", action="store_true",
                    help="default workload only: do not append the sub-records of the other BASELINE.json configurations")
    ap.add_argument("--iter-streams", type=int, default=1,
                    help="single-view workloads: issue consecutive (independent) iterations round-robin on this many "
                         "context + stream pairs, e.g. the maps of several agents optimised on one GPU; default 1 = the "
                         "headline number, one iteration after the other")
    ap.add_argument("--view-streams", type=int, default=4,
                    help="multi-view workloads (fused2m): views of one iteration are issued round-robin on this many "
                         "context + stream pairs; GS_ACCUMULATE adds with L2 reductions, so concurrent views are safe")
    ap.add_argument("--grads", default="dense", choices=["dense", "sparse"],
                    help="dense (default, the headline): (11 + 3K) N gradient arrays; sparse: GS_SPARSE_GRADS rows of the visible Gaussians")
    args = ap.parse_args()
    if args.workload == "fused2m" and args.steps == 2000:
        args.steps = 50   # 8 views per step: the default still finishes within a minute
    if args.impl == "reference":
        run_reference(args)
    elif args.workload == "peaks":
        run_peaks(args)
    elif args.workload == "next":
        run_next(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
