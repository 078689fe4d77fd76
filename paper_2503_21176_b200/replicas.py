"""Multi-GPU host logic: replicas only.

The path does not shard (no data-path collective): under torchrun every rank runs the same
workload on its own GPU.  The only cross-rank operations are the barrier around the timed region
and the MAX over ranks of the device-timed milliseconds; the whole-job value is
world_size * units_per_rank / max_ms.  Backend-agnostic so that the N > 1 path is testable with
gloo on CPU.
"""
import torch
import torch.distributed as dist


def world():
    return dist.get_world_size() if dist.is_available() and dist.is_initialized() else 1


def barrier():
    if world() > 1:
        dist.barrier()


def max_over_ranks(ms: float, device="cpu") -> float:
    if world() == 1:
        return float(ms)
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank: float, ms: float, device="cpu") -> float:
    """Whole-job units/s: every rank did `units_per_rank`, the job took the slowest rank's time."""
    return world() * units_per_rank / (max_over_ranks(ms, device) * 1e-3)
