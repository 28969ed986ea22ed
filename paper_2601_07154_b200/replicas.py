"""Multi-GPU plumbing for the "replicas only" scaling of this path.

Windows, heads and frames are independent and the only ordered step (the fold of <= 112 4x4 transforms) stays on
one device, so every rank runs one whole clip and no collective sits on the data path.  torch.distributed is used
for exactly two things: the barrier around the timed region and the max-over-ranks of the device time.
The same code runs on `nccl` (GPUs) and on `gloo` (the CPU tests, world_size 2)."""
import os

import torch
import torch.distributed as dist


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) outside it."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")))


def init(backend, device=None):
    """Joins the process group when WORLD_SIZE > 1 (rendezvous from MASTER_ADDR / MASTER_PORT).  Returns world size."""
    _, _, world = env_world()
    if world > 1 and not dist.is_initialized():
        kw = {"device_id": device} if (backend == "nccl" and device is not None) else {}
        dist.init_process_group(backend, **kw)
    return world


def barrier(device=None):
    if dist.is_initialized():
        dist.barrier()
    if device is not None and device.type == "cuda":
        torch.cuda.synchronize(device)


def max_over_ranks(x, device=None):
    """The slowest rank's time: every multi-GPU number is max over ranks of a device-side time."""
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank, ms_per_step_max, world):
    """Weak scaling: every rank processes `units_per_rank` per step; value = all ranks' units / slowest rank's time."""
    return world * units_per_rank / (ms_per_step_max * 1e-3)


def finish():
    if dist.is_initialized():
        dist.destroy_process_group()
