"""CPU tests of the benchmark harness: the N>1 aggregation (world size 2, gloo), the reference arm's JSON line and the
determinism of the seeded generators."""
import json
import os
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, torch.device("cpu"))
    q.put((rank, ms, bench.replica_throughput(world, 50, ms)))
    dist.barrier()
    dist.destroy_process_group()


def test_replica_aggregation_world_size_2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, val in res:
        assert ms == 15.0                      # the slowest rank's time on every rank
        assert abs(val - 2 * 50 / 0.015) < 1e-6  # all ranks' steps / max time


def test_reference_arm_prints_one_json_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--workload",
                          "replica_small", "--steps", "2", "--warmup", "1"], capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr
    lines = [l for l in out.stdout.splitlines() if l.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "iter/s" and d["higher_is_better"] is True
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] >= 1
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["e2e"]["value"] == d["value"] > 0


def test_reference_arm_other_ranks_do_nothing():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                         capture_output=True, text=True, timeout=120, env=env)
    assert out.returncode == 0 and out.stdout.strip() == ""


def test_generators_are_deterministic_and_shaped():
    from paper_2605_10760_b200 import scenes
    a, b = scenes.replica_scene(seed=30, N=1000), scenes.replica_scene(seed=30, N=1000)
    for k in ("means", "scales", "quats", "opacities", "sh"):
        assert np.array_equal(getattr(a, k), getattr(b, k)) and getattr(a, k).dtype == np.float32
    assert a.sh.shape == (1000, 16, 3) and a.camera.width == 1200 and a.camera.cx == 599.5
    R = a.camera.T_cw[:, :3].astype(np.float64)
    assert np.allclose(R @ R.T, np.eye(3), atol=1e-6) and np.linalg.det(R) > 0
    sc, cams = scenes.fused_scene(seed=50, N_sub=500, views=3, width=64, height=48, f=32.0)
    assert sc.N == 2000 and len(cams) == 3
    xi = scenes.tracking_perturbation(40)
    assert abs(np.linalg.norm(xi[:3]) - 0.02) < 1e-12 and abs(np.linalg.norm(xi[3:]) - np.deg2rad(1)) < 1e-12
