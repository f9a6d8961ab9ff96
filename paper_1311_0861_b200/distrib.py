"""Multi-GPU plumbing for bench.py: replicas only.

The path is single-GPU by construction (BASELINE.json north_star: no sharding, no collectives),
so N ranks run N independent replicas of the same workload ("weak" scaling).  The only
communication is the measurement itself: a barrier on both sides of the timed region and the
max over ranks of the device-timed milliseconds.  Works with NCCL (GPU) and gloo (CPU tests).
"""
import os


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when absent."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def free_port():
    import socket
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def launch_replicas(n, argv, timeout=None):
    """Start `n` copies of the command `argv`, one per GPU, the way torchrun would (RANK = LOCAL_RANK = 0..n-1,
    WORLD_SIZE = n, MASTER_ADDR 127.0.0.1, a free MASTER_PORT), and wait for them.  Rank 0 inherits this process's
    stdout (it prints the one JSON line); the other ranks' stdout is dropped, every rank's stderr is inherited.
    Returns the largest exit code.  This is what `python bench.py --gpus N` does when it is not already running
    under torchrun; processes are started and stopped by handle, never by name."""
    import subprocess
    port = free_port()
    procs = []
    for rank in range(n):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(n),
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen(list(argv), env=env, stdout=None if rank == 0 else subprocess.DEVNULL))
    rc = 0
    try:
        for p in procs:
            rc = max(rc, abs(p.wait(timeout=timeout)))
    finally:
        for p in procs:
            if p.poll() is None:
                p.kill()
    return rc


def init(backend, device=None):
    import torch.distributed as dist
    rank, _, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        kw = {}
        if backend == "nccl" and device is not None:
            kw["device_id"] = device
        dist.init_process_group(backend=backend, rank=rank, world_size=world, **kw)
    return rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value, device="cpu"):
    """Max over ranks of a Python float (the per-rank device-timed milliseconds)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(cells_per_rank, steps, ms_max, world):
    """Whole-job cell-updates/s of `world` replicas that each advanced `cells_per_rank` cells
    `steps` times within `ms_max` milliseconds (max over ranks)."""
    return world * cells_per_rank * steps / (ms_max * 1e-3)


def shutdown():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
