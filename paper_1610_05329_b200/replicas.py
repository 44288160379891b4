"""Multi-GPU plumbing for independent replicas (the step does not shard
without all-to-all transposes, which BASELINE.json rules out, so N GPUs run N independent
simulations -- "replicas only").  One process per GPU; torch.distributed carries only the barrier
and the max-over-ranks of the timing: there is no data-path collective."""
import os

import torch
import torch.distributed as dist


def env_world():
    """(rank, local_rank, world_size) from the torchrun environment; (0, 0, 1) when run directly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend=None):
    """Initialise the process group if WORLD_SIZE > 1. Returns (rank, local_rank, world_size)."""
    rank, local_rank, world = env_world()
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        if backend == "nccl":
            torch.cuda.set_device(local_rank)
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier():
    if dist.is_initialized():
        dist.barrier()


def _device():
    return torch.device("cuda", torch.cuda.current_device()) if dist.get_backend() == "nccl" else torch.device("cpu")


def max_over_ranks(x: float) -> float:
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=_device())
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float) -> float:
    if not dist.is_initialized():
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=_device())
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def replica_seed(base_seed: int, rank: int) -> int:
    """Each replica evolves its own seeded state (a parameter/seed scan): seed = base + 1000 rank."""
    return base_seed + 1000 * rank


def aggregate_throughput(units_local: float, seconds_local: float):
    """Whole-job throughput of independent replicas: all ranks' units / the slowest rank's time."""
    t = max_over_ranks(seconds_local)
    u = sum_over_ranks(units_local)
    return u / t, t


def shutdown():
    if dist.is_initialized():
        dist.destroy_process_group()
