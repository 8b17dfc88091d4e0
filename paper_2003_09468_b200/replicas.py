"""Host-side logic of the N>1 path: independent replicas, one process per GPU, walkers sharded by rank, no data-path
collective.  The only communication is the timing reduction.  `bench.py --gpus N` uses every
function here; tests/test_replicas_gloo.py drives them with two CPU ranks (gloo)."""
from __future__ import annotations

import os
import socket
import subprocess
import sys


def shard_walkers(total_walkers: int, rank: int, world: int):
    """Contiguous, balanced [start, stop) walker range of `rank` (first `total % world` ranks get one more)."""
    if world < 1 or not (0 <= rank < world) or total_walkers < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(total_walkers, world)
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)


def max_over_ranks(value_ms: float, device=None) -> float:
    """MAX all-reduce of a timing (any backend); identity when torch.distributed is not initialised."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value_ms)
    t = torch.tensor([value_ms], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t[0])


def aggregate_throughput(walkers_per_rank: int, steps: int, world: int, max_ms: float) -> float:
    """Whole-job walker-steps/s: all ranks' walkers over the slowest rank's time."""
    return walkers_per_rank * world * steps / (max_ms * 1e-3)


def rank_env():
    """(rank, local_rank, world) from the torchrun environment; (0, 0, 1) for a plain `python` run."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")))


def free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def launch_command(script: str, argv, nproc: int, port: int | None = None):
    """The command that starts `nproc` ranks of `script` on this node, one per GPU (the same line the driver uses)."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(int(nproc)),
            "--master-addr", "127.0.0.1", "--master-port", str(port or free_port()), script] + list(argv)


def needs_launch(ngpus: int) -> bool:
    """True when `--gpus N` (N > 1) was given to a plain `python` process: the ranks do not exist yet."""
    return ngpus > 1 and "WORLD_SIZE" not in os.environ


def launch_ranks(script: str, argv, nproc: int, timeout=None) -> int:
    """Re-executes `script argv` as `nproc` ranks under torchrun and returns its exit code (stdout/stderr inherited)."""
    return subprocess.call(launch_command(script, argv, nproc), timeout=timeout)
