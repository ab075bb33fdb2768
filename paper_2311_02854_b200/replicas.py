"""Multi-GPU plumbing: "replicas only".

BASELINE.json fixes the hot path to one GPU with no sharding and no collectives, so `bench.py --gpus N` runs N
independent replicas of the same bond, one process per GPU.  The only communication is the measurement
protocol: a barrier on both sides of the timed region and the MAX over ranks of the device time; the job
throughput is (units all ranks processed) / (slowest rank's time).  This module holds that logic so that it
can be exercised with the gloo backend on CPU.
"""
import os


def dist_env():
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0")))


def init(backend, device=None):
    import torch.distributed as dist
    _, world, _ = dist_env()
    if world > 1 and not dist.is_initialized():
        kw = {"device_id": device} if (device is not None and backend == "nccl") else {}
        dist.init_process_group(backend, **kw)
    return world


def barrier(sync=None):
    """sync(); barrier; sync()  -- sync is torch.cuda.synchronize on a GPU rank."""
    import torch.distributed as dist
    if sync:
        sync()
    if dist.is_available() and dist.is_initialized():
        dist.barrier()
        if sync:
            sync()


def max_over_ranks(x, device="cpu"):
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(units_per_rank_per_step, ms_per_step_local, world, device="cpu"):
    """Whole-job units/s: every rank does the same work; the step time is the slowest rank's."""
    ms = max_over_ranks(ms_per_step_local, device)
    return world * units_per_rank_per_step / (ms * 1e-3), ms
