"""Host-side logic of the multi-GPU run (bench.py --gpus N under torchrun).

The path shards over INDEPENDENT problems only: the six load cases of one image (S: 8(e)); rank r takes load case
(base + r) mod 6 on its own GPU.  There is no data-path collective; the only communication is the barrier and the
max-over-ranks reduction of the device time.  No method arithmetic lives here.
"""
from __future__ import annotations


def load_case_of_rank(rank: int, world: int, base: int = 2) -> int:
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return (base + rank) % 6 if world > 1 else base % 6


def max_over_ranks(ms: float, dist=None, device="cpu") -> float:
    """device time of the job = slowest rank (all_reduce MAX); dist = torch.distributed or None for one process"""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(voxels_per_rank: int, steps: int, world: int, ms: float) -> float:
    """whole-job voxel-updates/s: all ranks' units over the max-over-ranks time (weak scaling)"""
    return world * voxels_per_rank * steps / (ms * 1e-3)
