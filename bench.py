"""bench.py -- fwd+bwd rasterisation throughput of the 3DGS hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload replica300k|mono50k|...]

One step = one pass of the whole hot path: gs_preprocess -> gs_bin_tiles -> gs_rasterize_fwd ->
[upstream gradients: fixed seeded arrays, config 3 names no loss] -> gs_rasterize_bwd -> gs_pose_grad, on one
Replica-shaped synthetic scene of BASELINE.json configs[2] (300k Gaussians, 1200x680, SH degree 3).  The steps cycle
through five scenes (seeds 30-34; the workload varies ~3x with the pose), so the inputs of consecutive steps (71 MB of
parameters each, 355 MB in total) exceed the 126 MB L2.  Prints ONE JSON line.  Multi-GPU: replicas only:
every rank runs the same job on its own GPU; value = all ranks' steps / max-over-ranks device time.
`--impl reference` times the fp64 CPU oracle (oracle/) on the host cores on the same workload (rank 0 only).
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
SM_COUNT, FP32_LANES, SM_MAX_MHZ = 148, 128, 1965.0
# Algorithmic FP32 work of the compositing kernels, in FLOPs with FMA = 2:
#   evaluated pair: dx, dy (2) + power (fmul, fma, fmul, fmul, fma = 7) + o*G (1) + min (1) + compare (1) = 12, + 1 MUFU
#   blended pair, forward: T test (1) + alpha*T (1) + 4 fma (8) + (1-alpha) (1) + T*(.) (1) = 12
#   blended pair, backward: 1-alpha, T/oma (2 + MUFU), alpha*T, w_i (4 fma = 8), dalpha (fma + div = 3 + MUFU), S (2),
#       4 colour/depth products (4), clamp test (1), gp (1), 2 mean terms (2 fma + 2 mul + 2 mul = 8), 3 conic terms (6),
#       = 37; the reduction of the 10 sums over the pixels of the tile is 10 adds per blended pair = 10  -> 47
FLOP_EVAL, FLOP_BLEND_FWD, FLOP_BLEND_BWD = 12.0, 12.0, 47.0
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the compositing kernels, from the `ncu --set full` capture
# summarised in profiles/r1_v5_masks.md (scene seed 32); null for the other kernels
NCU_DRAM_BYTES = {"raster_bwd": 42.19e6 + 0.18e6, "raster_fwd": 14.66e6 + 0.11e6}


def load_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.index, self.rows, self._stop, self._t = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i",
                                      str(self.index)], capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.splitlines()[0].split(",")])
            except Exception:
                pass
            self._stop.wait(0.1)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[2 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]), "reasons": reasons,
                "samples": len(self.rows)}


def make_scenes(workload: str):
    if workload == "replica300k":
        return [scenes.replica_scene(seed=s) for s in SEEDS]
    if workload == "mono50k":
        return [scenes.mono_scene(seed=s) for s in (2, 3, 4)]
    if workload == "replica_small":  # CPU-side testing of the harness only
        return [scenes.replica_scene(seed=s, N=20000, width=300, height=170, f=150.0) for s in (30, 31)]
    raise SystemExit(f"unknown workload {workload}")


def oracle_leg(scs, budget_s: float, max_iters: int):
    """Times the fp64 oracle, as it stands, on the host cores: whole fwd+bwd iterations of the same workload."""
    from oracle import gso
    gso.lib()
    cores = gso.num_threads()
    t0, n = time.perf_counter(), 0
    while n < max_iters and (n == 0 or time.perf_counter() - t0 < budget_s):
        sc = scs[n % len(scs)]
        gC, gD = scenes.upstream_gradients(SEEDS[n % len(SEEDS)], sc.camera.width, sc.camera.height)
        gso.forward_backward(sc, gC, gD)
        n += 1
    dt = time.perf_counter() - t0
    return n / dt, cores, n, dt


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    scs = make_scenes(args.workload)
    sc = scs[0]
    for _ in range(min(args.warmup, 1)):
        gC, gD = scenes.upstream_gradients(SEEDS[0], sc.camera.width, sc.camera.height)
        from oracle import gso
        gso.forward_backward(sc, gC, gD)
    val, cores, n, dt = oracle_leg(scs, budget_s=120.0, max_iters=max(1, args.steps))
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "iter/s", "n_gpus": args.gpus, "steps": n,
            "warmup": min(args.warmup, 1), "ms_per_step": 1e3 / val, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.workload}: BASELINE.json configs[2], {sc.N} Gaussians, "
                                   f"{sc.camera.width}x{sc.camera.height}, SH{sc.sh_degree}, seeds {list(SEEDS)} cycled"},
            "cpu_baseline": {"value": val, "unit": "iter/s", "cores": cores, "kind": "oracle",
                             "sample": f"{n} whole fwd+bwd iterations (each step = one full iteration) in {dt:.1f} s"},
            "e2e": {"value": val, "unit": "iter/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "mpix_iter_per_s": val * sc.camera.width * sc.camera.height / 1e6}
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
    scs = make_scenes(args.workload)
    W, H = scs[0].camera.width, scs[0].camera.height
    ctx = B.Context(local)
    dss = [B.DeviceScene(sc, local) for sc in scs]
    ups = []
    for k, sc in enumerate(scs):
        gC, gD = scenes.upstream_gradients(SEEDS[k % len(SEEDS)], W, H)
        ups.append((torch.from_numpy(gC).to(dev), torch.from_numpy(gD).to(dev)))
    out = dss[0].alloc_outputs(W, H)

    def step(k):
        ds, sc = dss[k % len(dss)], scs[k % len(scs)]
        B.forward(ctx, ds, sc.camera, out)
        B.backward(ctx, out, ups[k % len(ups)][0], ups[k % len(ups)][1], None, 0, pose=True)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # warm-up: also calibrates the instance capacity over all poses (an overflowing iteration is re-issued)
    warm = max(args.warmup, 3)
    k = 0
    while k < max(warm, len(scs)):
        try:
            step(k)
            torch.cuda.synchronize()
            ctx.gs_poll()
            k += 1
        except B.GsError as e:
            if e.code != -5:
                raise
    stats = []
    for k in range(len(scs)):
        step(k)
        nv, ni = ctx.gs_get_counts()
        wl = ctx.gs_get_workload()
        stats.append(dict(visible=nv, instances=ni, **wl))
    barrier()

    # ---- timed region: exactly K steps, device time, max over ranks ----
    K = args.steps
    l0 = ctx.gs_get_launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local) as clk:
        barrier()
        e0.record()
        for k in range(K):
            step(k)
        e1.record()
        barrier()
    ms_total = e0.elapsed_time(e1)
    ctx.gs_poll()
    launches = ctx.gs_get_launch_count() - l0
    ms_total = max_over_ranks(ms_total, dist, dev)
    value = replica_throughput(world, K, ms_total)

    # ---- per-stage device times (second loop, stage events on; same steps) ----
    ctx.gs_profile_enable(True)
    stage_ms = {s: 0.0 for s in B.STAGES}
    per_scene_bwd = [0.0] * len(scs)
    per_scene_n = [0] * len(scs)
    for k in range(K):
        step(k)
        r = ctx.gs_profile_read()
        for s in B.STAGES:
            stage_ms[s] += r[s] / K
        per_scene_bwd[k % len(scs)] += r["raster_bwd"]
        per_scene_n[k % len(scs)] += 1
    ctx.gs_profile_enable(False)

    # ---- roofline of the dominant kernel ----
    dominant = max(stage_ms, key=stage_ms.get)
    hbm_peak, peak_src = load_peaks()
    alu_peak = SM_COUNT * FP32_LANES * 2 * SM_MAX_MHZ * 1e6 / 1e12  # TFLOP/s, FMA = 2
    used = [k % len(scs) for k in range(K)]
    mean = lambda key: float(np.mean([stats[u][key] for u in used]))
    if dominant == "raster_bwd":
        flops = mean("last_pos_sum") * FLOP_EVAL + mean("blended") * FLOP_BLEND_BWD
        roof = {"kernel": "raster_bwd_kernel", "bound": "alu", "achieved": flops / (stage_ms[dominant] * 1e-3) / 1e12,
                "peak": alu_peak, "unit": "TFLOP/s"}
    elif dominant == "raster_fwd":
        flops = mean("evaluated") * FLOP_EVAL + mean("blended") * FLOP_BLEND_FWD
        roof = {"kernel": "raster_fwd_kernel", "bound": "alu", "achieved": flops / (stage_ms[dominant] * 1e-3) / 1e12,
                "peak": alu_peak, "unit": "TFLOP/s"}
    else:
        N, K3 = scs[0].N, 3 * (scs[0].sh_degree + 1) ** 2
        V, I = mean("visible"), mean("instances")
        by = {"preprocess": 44 * N + 4 * K3 * V + 64 * V + 4 * N, "tile_scan": 16.0 * (W // 16 + 1) * (H // 16 + 1),
              "emit": 4 * N + 12 * V + 8 * I, "tile_sort": 20 * I,
              "gauss_bwd": (44 + 4 * K3) * V + 96 * V + (44 + 4 * K3) * N, "pose_grad": 120.0}[dominant]
        roof = {"kernel": dominant, "bound": "hbm", "achieved": by / (stage_ms[dominant] * 1e-3) / 1e9,
                "peak": hbm_peak, "unit": "GB/s"}
    roof["frac"] = roof["achieved"] / roof["peak"]
    roof["traffic"] = NCU_DRAM_BYTES.get(dominant)
    roof["traffic_unit"] = "bytes of DRAM traffic per launch (ncu, profiles/r1_v5_masks.md)"
    roof["peak_source"] = peak_src if roof["bound"] == "hbm" else \
        f"derived: {SM_COUNT} SMs x {FP32_LANES} FP32 lanes x 2 x {SM_MAX_MHZ:.0f} MHz (DESIGN.md)"
    roof["stage_share"] = stage_ms[dominant] / sum(stage_ms.values())

    # whole-iteration HBM figure (BASELINE.json "% HBM roofline"): algorithmic bytes of all stages / step time
    N, K3 = scs[0].N, 3 * (scs[0].sh_degree + 1) ** 2
    V, I, P = mean("visible"), mean("instances"), W * H
    bytes_iter = (44 * N + 4 * K3 * V + 64 * V + 4 * N) + (4 * N + 12 * V + 8 * I) + 20 * I + \
                 (4 * I + 48 * V + 24 * P) + (4 * I + 48 * V + 28 * P + 96 * V) + ((44 + 4 * K3) * V + (44 + 4 * K3) * N)
    hbm_frac_iter = bytes_iter / (ms_total / K * 1e-3) / 1e9 / hbm_peak

    line = None
    if rank == 0:
        # ---- end to end through the C-ABI with HOST buffers (pinned), copies inside the timed region ----
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a, np.float32)).pin_memory().numpy()
        e2e_steps = max(3, min(K, 10))
        hsc = [tuple(pin(x) for x in (sc.means, sc.scales, sc.quats, sc.opacities, sc.sh)) for sc in scs[:2]]
        hup = [tuple(pin(x) for x in scenes.upstream_gradients(SEEDS[k], W, H)) for k in range(2)]
        Kc = (scs[0].sh_degree + 1) ** 2
        Ng = scs[0].N
        hout = {k: torch.zeros(s, dtype=torch.float32).pin_memory().numpy() for k, s in
                dict(rgb=(3, H, W), depth=(H, W), alpha=(H, W), g_means=(Ng, 3), g_scales=(Ng, 3), g_quats=(Ng, 4),
                     g_opacities=(Ng,), g_sh=(Ng, Kc, 3), g_twist=(6,)).items()}
        ctx2 = B.Context(local)

        def e2e_step(k):
            ctx2.gs_fwd_bwd_host(hsc[k % 2], scs[0].sh_degree, scs[k % 2].camera, scs[k % 2].bg, hup[k % 2][0],
                                 hup[k % 2][1], hout)
        for k in range(3):
            try:
                e2e_step(k)
            except B.GsError as e:
                if e.code != -5:
                    raise
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for k in range(e2e_steps):
            e2e_step(k)
        torch.cuda.synchronize()
        e2e_dt = time.perf_counter() - t0
        h2d = sum(x.nbytes for x in hsc[0]) + sum(x.nbytes for x in hup[0])
        d2h = sum(x.nbytes for x in hout.values())
        ctx2.close()

        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            v, cores, n, dt = oracle_leg(scs, budget_s=12.0, max_iters=10 * len(scs))
            cpu = {"value": v, "unit": "iter/s", "cores": cores, "kind": "oracle",
                   "sample": f"{n} whole fwd+bwd iterations of the same workload (scene seeds cycled) in {dt:.1f} s"}
        sc = scs[0]
        line = {"metric": METRIC, "value": value, "unit": "iter/s", "n_gpus": world, "steps": K, "warmup": warm,
                "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": {"workload": f"{args.workload}: BASELINE.json configs[2], {sc.N} Gaussians, {W}x{H}, "
                                       f"SH{sc.sh_degree}, seeds {[30 + k for k in range(len(scs))]} cycled",
                           "l2": "inputs larger than L2: 5 scenes x 71 MB of parameters cycled step to step",
                           "parallelism": "replicas only" if world > 1 else "single GPU"},
                "mpix_iter_per_s": value * W * H / 1e6,
                "clocks": clk.summary(),
                "e2e": {"value": world * e2e_steps / e2e_dt, "unit": "iter/s", "h2d_bytes_per_step": h2d,
                        "d2h_bytes_per_step": d2h, "steps": e2e_steps},
                "gpu_launches": launches,
                "roofline": roof,
                "cpu_baseline": cpu,
                "hbm_frac_whole_iteration": hbm_frac_iter,
                "algorithmic_bytes_per_iter": bytes_iter,
                "stages_ms": stage_ms,
                "workload_stats": {"visible": mean("visible"), "instances": mean("instances"),
                                   "evaluated_pairs": mean("evaluated"), "blended_pairs": mean("blended"),
                                   "tile_list_x_pixels": mean("list_len_x_pixels")}}
    ctx.close()
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line))


def run_extra(args):
    """Configs 4 (tracking, pose only) and 5 (fused refinement, 8 views accumulated): device-resident throughput and
    stage times only (the headline line with roofline / e2e / cpu_baseline is the default workload's)."""
    import torch
    from paper_2605_10760_b200 import binding as B
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    ctx = B.Context(0)
    if args.workload == "tracking500k":
        # BASELINE.json configs[3]: 500k Gaussians frozen, L1 RGB against a render from the perturbed pose; per step:
        # preprocess (pose read from the device) -> bin -> fwd -> L1 gradient -> bwd (pose only) -> pose gradient ->
        # on-device normalised pose step; no host synchronisation inside the loop
        sc = scenes.replica_scene(seed=40, N=500_000)
        W, H = sc.camera.width, sc.camera.height
        ds = B.DeviceScene(sc, 0)
        out = ds.alloc_outputs(W, H)
        cam_t = sc.camera.copy()
        cam_t.T_cw = scenes.perturb_pose(sc.camera.T_cw, scenes.tracking_perturbation(40))
        B.forward(ctx, ds, cam_t, out)
        torch.cuda.synchronize(); ctx.gs_poll()
        target = out["rgb"].clone()
        T_dev = torch.from_numpy(np.ascontiguousarray(sc.camera.T_cw, np.float32).reshape(-1)).to(dev)
        gC = torch.empty_like(out["rgb"])

        def step(k):
            B.forward(ctx, ds, sc.camera, out, T_cw_dev=T_dev)
            B.gs_aux_l1_grad(out["rgb"], target, 1.0 / (3 * W * H), gC)
            B.backward(ctx, out, gC, None, None, flags=B.GS_POSE_ONLY, pose=True)
            B.gs_aux_pose_step(T_dev, out["g_twist"], 1e-3)
        views, label = 1, "tracking500k: BASELINE.json configs[3], 500000 Gaussians, 1200x680, SH3, pose-only, seed 40"
    else:
        # BASELINE.json configs[4]: 2M Gaussians (4 Sim(3)-mapped submaps), 8 views per iteration, gradients accumulated
        sc, cams = scenes.fused_scene(seed=50)
        W, H = cams[0].width, cams[0].height
        ds = B.DeviceScene(sc, 0)
        out = ds.alloc_outputs(W, H)
        ups = [tuple(torch.from_numpy(a).to(dev) for a in scenes.upstream_gradients(50 + v, W, H)) for v in range(len(cams))]

        def step(k):
            for v, cam in enumerate(cams):
                B.forward(ctx, ds, cam, out)
                B.backward(ctx, out, ups[v][0], ups[v][1], None, flags=(B.GS_ACCUMULATE if v > 0 else 0), pose=False)
        views, label = len(cams), "fused2m: BASELINE.json configs[4], 2000000 Gaussians, 8 views of 1200x680, SH3, seed 50"
    k = 0
    while k < max(args.warmup, 3):
        try:
            step(k); torch.cuda.synchronize(); ctx.gs_poll(); k += 1
        except B.GsError as e:
            if e.code != -5:
                raise
    K = args.steps
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(0) as clk:
        torch.cuda.synchronize()
        e0.record()
        for k in range(K):
            step(k)
        e1.record()
        torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    ctx.gs_poll()
    nv, ni = ctx.gs_get_counts()
    value = K / (ms / 1e3)
    print(json.dumps({"metric": "fwd+bwd rasterize iters/sec", "value": value, "unit": "iter/s", "n_gpus": 1, "steps": K,
                      "warmup": max(args.warmup, 3), "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": {"workload": label},
                      "views_per_iter": views, "mpix_iter_per_s": value * views * W * H / 1e6, "clocks": clk.summary(),
                      "last_view": {"visible": nv, "instances": ni}}))
    ctx.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="replica300k")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.workload in ("tracking500k", "fused2m"):
        run_extra(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
