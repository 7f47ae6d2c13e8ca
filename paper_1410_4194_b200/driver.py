"""Time-loop driver shared by tests and bench.py.  Duck-typed over anything with the
`set_state / compute_dt / step / get_state` surface (the CUDA `Grid` or the oracle's `RefGrid`);
it holds none of the method's arithmetic and imports neither implementation.

The loop is the paper's main loop (Fig. 3) minus the per-step host<->device copies:
`dt = compute_dt(cfl)` (Eq. 22), `step(dt)` (steps 1-5), repeat.
"""
from __future__ import annotations

import math


def run(grid, wl, max_steps=None, dts=None, record_dts=None, set_state=True):
    """Advance `grid` through workload `wl`.  Returns (steps taken, final time).

    dts         — optional list of time steps to replay (lock-step mode: the oracle's dt fed to both).
    record_dts  — optional list that receives the dt of every step taken.
    """
    if set_state:
        grid.set_state(wl.u)
    t, n = 0.0, 0
    limit = wl.steps if wl.steps is not None else 10 ** 9
    if max_steps is not None:
        limit = min(limit, max_steps)
    while n < limit:
        if wl.t_end is not None and t >= wl.t_end * (1.0 - 1e-14):
            break
        if dts is not None:
            if n >= len(dts):
                break
            dt = dts[n]
        else:
            dt = grid.compute_dt(wl.cfl)
            if not math.isfinite(dt) or dt <= 0.0:
                raise FloatingPointError(f"compute_dt returned {dt} at step {n}")
            if wl.t_end is not None and t + dt > wl.t_end:
                dt = wl.t_end - t
        grid.step(dt)
        if record_dts is not None:
            record_dts.append(dt)
        t += dt
        n += 1
    return n, t


def max_over_ranks(seconds: float, dist=None, device="cpu") -> float:
    """Elapsed time of the slowest rank (bench.py: the whole job's time when every rank steps its own
    replica).  `dist` is torch.distributed once initialised (nccl on GPUs, gloo in the CPU tests), or
    None for a single process.  The only collective on the path: a MAX all-reduce of one double."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(seconds)
    import torch
    t = torch.tensor([seconds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_rate(units_per_rank: float, seconds: float, dist=None, device="cpu") -> float:
    """Whole-job throughput of N independent replicas: all ranks' units / the slowest rank's time."""
    world = 1 if dist is None or not dist.is_initialized() else dist.get_world_size()
    return world * units_per_rank / max_over_ranks(seconds, dist, device)
