"""Multi-GPU plumbing of the bench: the path does not shard ("replicas only"), so N ranks
run N independent replicas; the only communication is the timing protocol -- a barrier on both sides
of the timed region and the MAX over ranks of the device-measured time.  Backend-agnostic
(`nccl` on GPUs, `gloo` in the CPU tests); holds none of the method's arithmetic."""
import os


def init(backend, device_id=None):
    """Initialise torch.distributed from the torchrun environment; returns (rank, world)."""
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        kw = {}
        if device_id is not None:
            kw["device_id"] = device_id
        dist.init_process_group(backend, **kw)
    return rank, world


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def max_over_ranks(value, device="cpu"):
    """MAX over ranks of a python float (the slowest rank defines the step time)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank, world, ms_max):
    """Whole-job throughput: every rank processed `units_per_rank` units in `ms_max` milliseconds
    (weak scaling: replicas)."""
    return world * units_per_rank / (ms_max * 1e-3)


def finalize():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()
        dist.destroy_process_group()
