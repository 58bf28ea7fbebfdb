"""Multi-GPU = replicas only: the path does not shard, so N GPUs run
N independent copies of the workload.  This module holds the only cross-rank logic there is:
the barrier and the reduction of per-rank timings into one whole-job figure."""
import os


def world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process = 1 GPU)."""
    return (int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)),
            int(os.environ.get("WORLD_SIZE", 1)))


def init(backend):
    import torch.distributed as dist
    rank, _, ws = world()
    if ws > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        dist.init_process_group(backend=backend, rank=rank, world_size=ws)
    return rank, ws


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def aggregate(units_local, ms_local, device="cpu"):
    """Whole-job throughput of independent replicas: sum of the units all ranks processed
    divided by the slowest rank's time.  Returns (units_total, ms_max, units_per_s)."""
    import torch
    import torch.distributed as dist
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized():
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    units, ms = float(u.item()), float(t.item())
    return units, ms, units / (ms * 1e-3) if ms > 0 else 0.0
