"""Host-side logic of the N > 1 bench ("replicas only"): every rank runs the same
step on its own GPU with no data-path collective; the only communication is the barrier around the
timed region and the max-over-ranks reduction of the device time."""
from __future__ import annotations


def max_over_ranks(ms: float, dist=None, device=None) -> float:
    """Device time of the timed region as the MAX over ranks (identity when not distributed)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms)
    import torch
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_us_per_layer(ms_step: float, layers_per_step: int, world: int) -> float:
    """N replicas each finish `layers_per_step` layers in `ms_step`: whole-job time per layer."""
    return ms_step * 1e3 / (layers_per_step * world)
