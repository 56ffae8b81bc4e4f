"""Host-side logic of the N > 1 path ("replicas only").

BASELINE.json north_star: "one B200 holding the cube in HBM, with no sharding and no
collectives", so N GPUs are N independent replicas of the renderer, each holding its own copy of
the cube and taking its own frames of the camera orbit ("interactive frame
rates": the unit of work is a frame).  The only communication is the reduction of the timing and
of the work counters at the end of a run.  No method arithmetic lives here.
"""
from __future__ import annotations


def orbit_frame(step_index: int, n_steps: int, rank: int = 0, world: int = 1, n_frames: int = 360) -> int:
    """Frame of the n_frames-frame orbit that `rank` renders at its step `step_index`: the
    n_steps * world frames of a run are spread evenly over the orbit and interleaved over the
    ranks, so every rank sees every viewing direction and no frame is rendered twice as long as
    n_steps * world <= n_frames."""
    total = max(1, n_steps * world)
    return int(round((step_index * world + rank) * float(n_frames) / total)) % n_frames


def frames_of_rank(n_steps: int, rank: int, world: int, n_frames: int = 360) -> list:
    return [orbit_frame(i, n_steps, rank, world, n_frames) for i in range(n_steps)]


def reduce_run(dist, device, ms_total: float, sums) -> tuple:
    """Whole-job figures from per-rank ones: the run takes as long as its slowest rank (MAX of the
    device-timed milliseconds), work counters add up (SUM).  `dist` is torch.distributed (or None
    for one process); `device` is where the small reduction tensors live ("cuda" under NCCL, "cpu"
    under gloo).  Returns (ms_total, [sums...])."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms_total), [int(v) for v in sums]
    import torch
    t = torch.tensor([float(ms_total)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    s = torch.tensor([float(v) for v in sums], dtype=torch.float64, device=device)
    dist.all_reduce(s, op=dist.ReduceOp.SUM)
    return float(t.item()), [int(v) for v in s.tolist()]
