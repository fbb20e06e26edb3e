"""Host-side logic of bench.py for N > 1 (replicas only): per-rank replica seeds, MAX over
ranks of the timings, whole-job rate; and the reference arm under a multi-rank launch (rank 0 alone works).
world_size-2 `gloo` on CPU; no GPU, no compute through the C ABI."""
import json
import os
import socket
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench

    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r pretends its K steps took (10 + 5 r) ms on the device and (40 - 3 r) ms end to end
    ms, e2e = bench.max_over_ranks([10.0 + 5.0 * rank, 40.0 - 3.0 * rank], world)
    seed = bench.replica_seed(1005, rank)
    with open(os.path.join(out_dir, f"r{rank}.json"), "w") as f:
        json.dump({"ms": ms, "e2e": e2e, "seed": seed,
                   "value": bench.whole_job_rate(world, 1000, 4, ms)}, f)
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate_gloo(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    r = [json.load(open(tmp_path / f"r{k}.json")) for k in range(world)]
    for k in range(world):
        assert r[k]["ms"] == 15.0 and r[k]["e2e"] == 40.0  # the slowest rank decides, on every rank
        assert r[k]["value"] == pytest.approx(2 * 1000 * 4 / 15e-3)  # units of ALL ranks / max time
    assert r[0]["seed"] != r[1]["seed"] and r[0]["seed"] == 1005  # independent replicas


def test_single_rank_needs_no_process_group():
    import bench

    assert bench.max_over_ranks([3.0, 4.0], 1) == [3.0, 4.0]
    assert bench.whole_job_rate(1, 134217728, 10, 80.0) == pytest.approx(134217728 * 10 / 0.08)


def test_reference_arm_under_two_ranks_only_rank0_prints():
    """`bench.py --impl reference` under a 2-rank launch: rank 0 prints the JSON line, rank 1 exits 0 silently."""
    outs = []
    for rank in (0, 1):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT="29511")
        p = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                            "--steps", "1", "--warmup", "0", "--ref-np", "16"], env=env, capture_output=True,
                           text=True, timeout=300)
        assert p.returncode == 0, p.stderr
        outs.append(p.stdout.strip())
    assert outs[1] == ""
    line = json.loads(outs[0])
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle"
    assert line["value"] > 0 and line["e2e"]["h2d_bytes_per_step"] == 0 and line["unit"] == "particles/s"
