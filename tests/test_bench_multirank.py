"""The N > 1 path of bench.py on CPU: world-size-2 gloo ranks aggregate time as max-over-ranks and units as the sum
(independent replicas, no data-path collective); the reference arm prints on rank 0 only."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench

    dist.init_process_group("gloo", rank=rank, world_size=world)
    t, u = bench.aggregate_over_ranks(1.0 + rank, 10.0 * (rank + 1), world, dist, torch.device("cpu"))
    out.put((rank, t, u))
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_over_two_gloo_ranks():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29731, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for _, t, u in got:
        assert t == 2.0 and u == 30.0  # max of (1, 2) seconds, sum of (10, 20) units


def test_single_rank_aggregate_is_identity():
    sys.path.insert(0, ROOT)
    import bench

    assert bench.aggregate_over_ranks(0.5, 7.0, 1) == (0.5, 7.0)
    assert [bench.trajectory_offsets(k) for k in (0, 1, 25, 26, 49, 50, 51)] == [0.0, 1.0, 25.0, 24.0, 1.0, 0.0, 1.0]


def test_reference_arm_two_ranks_prints_once():
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29733", WORLD_SIZE="2")
    outs = []
    for rank in (0, 1):
        e = dict(env, RANK=str(rank), LOCAL_RANK=str(rank))
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
                            "--warmup", "0"], env=e, capture_output=True, text=True, timeout=300)
        assert r.returncode == 0, r.stderr
        outs.append(r.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "pair interactions/s"
