"""Host-side plumbing of the N > 1 bench (replicas only -- the path does not
shard below one frame, so there is no data-path collective).  One process per GPU; the only
communication is the barrier around the timed region and the max-over-ranks of the device time.
Backend "nccl" on GPUs, "gloo" in the CPU tests."""
from __future__ import annotations

import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist


def world_info():
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")),
            int(os.environ.get("LOCAL_RANK", "0")))


def needs_spawn(n_gpus: int) -> bool:
    """True when N > 1 ranks were asked for but this process was not started by torchrun."""
    return n_gpus > 1 and "WORLD_SIZE" not in os.environ


def spawn(script: str, argv: list, n: int, env: dict | None = None, timeout: float | None = None) -> int:
    """Start `script argv` as n ranks of one node (torchrun, rendezvous on 127.0.0.1, a free port):
    what `python bench.py --gpus N` does when it was started plainly.  Returns the exit code."""
    with socket.socket() as sock:
        sock.bind(("127.0.0.1", 0))
        port = sock.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), script, *map(str, argv)]
    return subprocess.run(cmd, env=env, timeout=timeout).returncode


def init(backend: str | None = None):
    """Join the process group if launched under torchrun; returns (world, rank, local_rank)."""
    world, rank, local_rank = world_info()
    if world > 1 and not dist.is_initialized():
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        kw = {}
        if backend == "nccl":
            kw["device_id"] = torch.device("cuda", local_rank)
        dist.init_process_group(backend, **kw)
    return world, rank, local_rank


def barrier():
    if torch.cuda.is_available():
        torch.cuda.synchronize()
    if dist.is_initialized():
        dist.barrier()
        if torch.cuda.is_available():
            torch.cuda.synchronize()


def max_over_ranks(value: float) -> float:
    """The slowest rank's time decides the job's throughput."""
    if not dist.is_initialized():
        return float(value)
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(value)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank: float, ms_this_rank: float) -> float:
    """Whole-job units/s: every rank processed `units_per_rank`; time = max over ranks."""
    world = dist.get_world_size() if dist.is_initialized() else 1
    ms = max_over_ranks(ms_this_rank)
    return world * units_per_rank / (ms * 1e-3)


def shutdown():
    if dist.is_initialized():
        dist.barrier()
        dist.destroy_process_group()
