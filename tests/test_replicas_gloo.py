"""N>1 host logic on CPU: world_size 2, gloo.  Walker sharding, max-over-ranks timing, aggregate value."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2003_09468_b200 import replicas


def test_shard_walkers_partitions_exactly():
    for total in (0, 1, 7, 32, 33):
        for world in (1, 2, 3, 8):
            spans = [replicas.shard_walkers(total, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == total
            for a, b in zip(spans, spans[1:]):
                assert a[1] == b[0]
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        replicas.shard_walkers(4, 2, 2)


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    my_ms = 10.0 + 5.0 * rank                      # rank 1 is slower
    mx = replicas.max_over_ranks(my_ms)
    dist.barrier()
    out[rank] = (mx, replicas.aggregate_throughput(32, 10, world, mx), replicas.shard_walkers(33, rank, world))
    dist.destroy_process_group()


def test_two_rank_timing_is_max_over_ranks():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert out[0][0] == out[1][0] == 15.0
    assert out[0][1] == pytest.approx(32 * 2 * 10 / 15e-3)
    assert out[0][2] == (0, 17) and out[1][2] == (17, 33)


def test_single_process_identity():
    assert replicas.max_over_ranks(3.5) == 3.5


def test_launch_command_is_the_drivers_line():
    cmd = replicas.launch_command("bench.py", ["--gpus", "2"], 2, port=29511)
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"]
    assert cmd[cmd.index("--nproc-per-node") + 1] == "2"
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29511"
    assert cmd[-3:] == ["bench.py", "--gpus", "2"]
    assert replicas.rank_env() == (0, 0, 1) or "WORLD_SIZE" in os.environ


def test_needs_launch_only_without_a_rank_environment(monkeypatch):
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    assert not replicas.needs_launch(1)
    assert replicas.needs_launch(2)
    monkeypatch.setenv("WORLD_SIZE", "2")
    assert not replicas.needs_launch(2)


def test_bench_gpus_2_starts_two_ranks_and_rank0_prints_one_line():
    """`python bench.py --gpus 2` (no torchrun) must start the two ranks itself.  Driven here on CPU through the
    reference arm (the CPU oracle: rank 0 works, the other rank exits 0), smallest config."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--impl", "reference", "--config", "C1",
                        "--steps", "1", "--warmup", "0", "--cores", "2"], capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    rec = json.loads(lines[0])
    assert rec["impl"] == "reference" and rec["n_gpus"] == 2 and rec["cpu_baseline"]["cores"] == 2
    assert rec["value"] > 0 and rec["e2e"]["h2d_bytes_per_step"] == 0
