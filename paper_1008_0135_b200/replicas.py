"""Replica plumbing for N > 1 (replicas only).

The path does not shard on one B200 (north_star: one GPU holds the whole cube, no data-path
collective), so N ranks are N independent replicas that render different views of the orbit.
The only communication is the barrier around the timed region and the max-over-ranks of the time.
No arithmetic of the method lives here.
"""
import torch


def view_of(step_idx: int, rank: int, world: int, n_views: int) -> int:
    """View index rendered by `rank` at step `step_idx`: ranks start at evenly spaced points of the orbit."""
    return (step_idx + rank * max(1, n_views // max(1, world))) % n_views


def max_over_ranks(value: float, dist=None, device="cpu") -> float:
    """Max of a per-rank scalar (a time in ms) over all ranks; identity when not distributed."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_ms_per_frame(total_ms_max: float, steps_per_rank: int, world: int) -> float:
    """Whole-job ms/frame: the ranks' K frames each finish inside the slowest rank's time."""
    return total_ms_max / float(steps_per_rank * world)
