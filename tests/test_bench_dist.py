"""bench.py's N > 1 host logic on CPU: world-size-2 gloo. Frames are sharded across ranks (no
data-path collective); the whole-job value divides all ranks' frames by the slowest rank's time."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import bench


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group(backend="gloo", rank=rank, world_size=world)

    def reduce_max(x):
        t = torch.tensor([x], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    local_ms = 100.0 * (rank + 1)  # rank 1 is the slow one
    fps, ms = bench.aggregate(local_ms, 36, world, reduce_max)
    order = bench.views_for_rank(rank, world, 36)
    out.put((rank, fps, ms, order[0], sorted(order) == list(range(36))))
    dist.barrier()
    dist.destroy_process_group()


def test_world_size_2_aggregate_and_view_sharding():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, fps, ms, first, full in res:
        assert ms == 200.0                       # max over ranks
        assert fps == pytest.approx(2 * 36 / 0.2)  # all ranks' frames over the slowest rank's time
        assert full                              # each rank still renders the whole cycle
    assert [r[3] for r in res] == [0, 18]        # ... from different view offsets


def test_single_rank_aggregate():
    fps, ms = bench.aggregate(50.0, 10, 1)
    assert ms == 50.0 and fps == pytest.approx(200.0)


def test_workloads_match_baseline_configs():
    for name, dims, brick, wh, step in (("c0", (64, 64, 64), 64, (256, 256), 0.5), ("c1", (512, 512, 512), 256, (1024, 1024), 0.5),
                                        ("c2", (1024, 1024, 1024), 256, (1920, 1080), 0.5),
                                        ("c3", (4096, 4096, 1536), 512, (1920, 1080), 1.0)):
        w = bench.workload(name)
        assert (w["nx"], w["ny"], w["nz"]) == dims and w["brick"] == brick and (w["width"], w["height"]) == wh
        assert w["step"] == step and len(w["views"]) == 36 and w["tau"] == 0.99 and w["ghost"] == 1


def test_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` (the oracle timed on the host cores, this tier's reference arm) on the
    smallest workload: one JSON line with the base contract's keys, no GPU involved."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--workload", "c0", "--steps", "2",
                        "--warmup", "1"], capture_output=True, text=True, timeout=600, cwd=root)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    j = json.loads(lines[0])
    for key in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "e2e", "cpu_baseline", "impl"):
        assert key in j, key
    assert j["impl"] == "reference" and j["unit"] == "frames/s" and j["value"] > 0 and j["steps"] == 2
    assert j["cpu_baseline"]["kind"] == "oracle" and j["cpu_baseline"]["cores"] >= 1
    assert j["e2e"]["h2d_bytes_per_step"] == 0 and j["e2e"]["d2h_bytes_per_step"] == 0 and j["vs_baseline"] is None


def test_product_arm_refuses_to_run_without_a_gpu():
    """No CPU fallback: without a CUDA device the product arm exits loudly instead of measuring something else."""
    import subprocess
    import sys
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--workload", "c0", "--steps", "1"], capture_output=True,
                       text=True, timeout=600, cwd=root)
    assert r.returncode != 0 and "no CUDA device" in (r.stderr + r.stdout)
