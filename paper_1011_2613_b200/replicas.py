"""Multi-GPU plumbing: "replicas only" (multi-GPU section).

BASELINE.json's north_star fixes the path to one GPU (no sharding, no inter-GPU
collective), so N GPUs run N independent replicas of the workload, one process
per GPU.  The only communication is the bookkeeping below: a barrier around the
timed region, the MAX over ranks of the device time and the SUM over ranks of the
lattice updates done.  Works with the nccl backend (GPU tensors) and with gloo
(CPU tensors; used by the world_size-2 CPU tests).
"""
import os

import torch
import torch.distributed as dist


def init_from_env(backend=None):
    """Initialises torch.distributed from RANK/WORLD_SIZE/MASTER_* when launched by torchrun.
    Returns (rank, world_size, local_rank)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1 and not dist.is_initialized():
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, world, local


def _device():
    if dist.is_initialized() and dist.get_backend() == "nccl":
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def barrier():
    if dist.is_initialized():
        dist.barrier()


def aggregate(units_local, ms_local):
    """-> (sum over ranks of units, max over ranks of ms).  Identity without a process group."""
    if not dist.is_initialized():
        return float(units_local), float(ms_local)
    dev = _device()
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=dev)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=dev)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(u.item()), float(t.item())


def mlups(units_total, ms_max):
    """Whole-job throughput in million lattice updates per second."""
    return units_total / (ms_max * 1e-3) / 1e6


def shutdown():
    if dist.is_initialized():
        dist.destroy_process_group()
