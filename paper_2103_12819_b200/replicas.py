"""Host-side plumbing of multi-process runs (one process per GPU, ``torch.distributed``).

The timing protocol ``bench.py`` uses at N > 1, whatever the ranks run -- the z-slabs of one grid
(``slabs.py``, the default) or, when the slab set-up fails, N independent replicas (labelled as such,
no headline value): a barrier on both sides of the timed region, the MAX over ranks of the device
time, and the whole-job rate = all ranks' cell updates / that time.  These helpers work on any
backend (``nccl`` on GPUs, ``gloo`` in the CPU tests) and hold none of the method's arithmetic.
"""
from __future__ import annotations


def _dist():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() else None


def barrier() -> None:
    d = _dist()
    if d is not None:
        d.barrier()


def max_over_ranks(x: float, device=None) -> float:
    """MAX over all ranks of a host scalar (identity without a process group)."""
    d = _dist()
    if d is None:
        return float(x)
    import torch
    if d.get_backend() == "gloo":
        device = "cpu"
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    d.all_reduce(t, op=d.ReduceOp.MAX)
    return float(t[0])


def whole_job_rate(cells_per_rank: int, steps: int, seconds_max: float, world: int) -> float:
    """Cell updates per second of the whole job: every rank advanced ``cells_per_rank`` cells by
    ``steps`` steps within ``seconds_max`` (the slowest rank's time)."""
    return world * cells_per_rank * steps / seconds_max
