"""Host logic of bench.py's N > 1 path on CPU: two ranks over the gloo backend (no GPU needed).

The hot path does not shard in this build ("replicas only"): every rank solves its own replica and
the only cross-rank step is the aggregation of the timed region — MAX of the device times, SUM of the iterations and
launches — which is what this test drives; plus: under `--impl reference` only rank 0 works."""
import json
import os
import socket
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    import torch.distributed as dist

    sys.path.insert(0, ROOT)
    import bench

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r "measured" 10 + r ms, did 100 + r iterations with 4 launches each
    maxes, sums = bench.reduce_over_ranks(dist, [10.0 + rank], [100 + rank, 4 * (100 + rank)], torch.device("cpu"))
    dist.barrier()
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump({"maxes": maxes, "sums": sums}, f)
    dist.destroy_process_group()


def test_aggregation_over_two_gloo_ranks(tmp_path):
    import torch.multiprocessing as mp

    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    for r in range(world):
        d = json.load(open(tmp_path / f"r{r}.json"))
        assert d["maxes"] == [11.0]            # the slowest rank sets the time
        assert d["sums"] == [201.0, 804.0]     # work adds up: value = 201 iterations / 11 ms
    # single rank: identity
    sys.path.insert(0, ROOT)
    import bench

    assert bench.reduce_over_ranks(None, [3.5], [7, 28], None) == ([3.5], [7.0, 28.0])


def test_reference_arm_only_rank0_works():
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2")
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "c1",
                          "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    assert res.returncode == 0 and res.stdout.strip() == ""
    env["RANK"] = "0"
    res = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "c1",
                          "--steps", "1", "--warmup", "0"], env=env, capture_output=True, text=True, timeout=120)
    line = json.loads(res.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
