"""Host-side logic of the N > 1 launch: replicas only.

``BASELINE.json:north_star`` fixes "one GPU, with no sharding and no collectives": a galaxy's cube
is one reduction over all its particles, so ``bench.py --gpus N`` runs N independent replicas,
rank r building its own galaxy.  The only communication is the barrier around the timed region and
the max-over-ranks reduction of the elapsed time; both work on any ``torch.distributed`` backend
(NCCL on the GPU box, gloo in the CPU tests).  No method arithmetic lives here.
"""
from __future__ import annotations

BASE_GALAXY_SEED = 1000          # synth: galaxy seed of config i is 1000 + i


def replica_seed(workload_index: int, rank: int) -> int:
    """Galaxy seed of rank ``rank`` for config ``workload_index``: rank 0 is the config's own
    galaxy (1000 + i); rank r > 0 draws the same recipe from seed 1000 + 10 r + i."""
    if rank < 0 or workload_index < 0 or workload_index >= 10:
        raise ValueError("rank >= 0 and 0 <= workload_index < 10 required")
    return BASE_GALAXY_SEED + 10 * rank + workload_index


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a host scalar (elapsed milliseconds); identity without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank: float, world: int, elapsed_ms_max: float, steps: int) -> float:
    """Weak-scaling aggregate: every rank processed ``units_per_rank`` units per step; the job took
    the slowest rank's time.  Returns units per second over all ranks."""
    if steps <= 0 or elapsed_ms_max <= 0.0 or world <= 0:
        raise ValueError("steps, world and elapsed time must be positive")
    return world * units_per_rank * steps / (elapsed_ms_max * 1e-3)
