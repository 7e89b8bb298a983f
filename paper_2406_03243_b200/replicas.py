"""Multi-GPU plumbing for bench.py.  The migration path shards with NO data-path collective: every
(block, layer, K|V) tile is independent, and a source/destination instance pair lives on one device
in this build.  N ranks therefore run N independent replicas;
the only cross-rank traffic is the timing protocol below (barrier, max of times, sum of units)."""
from __future__ import annotations


def _dist():
    try:
        import torch.distributed as dist
        if dist.is_available() and dist.is_initialized():
            return dist
    except Exception:  # noqa: BLE001
        pass
    return None


def world_size() -> int:
    d = _dist()
    return d.get_world_size() if d else 1


def _device():
    import torch
    d = _dist()
    if d and d.get_backend() == "nccl":
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def barrier() -> None:
    d = _dist()
    if d:
        d.barrier()


def max_over_ranks(x: float) -> float:
    d = _dist()
    if not d:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=_device())
    d.all_reduce(t, op=d.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float) -> float:
    d = _dist()
    if not d:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=_device())
    d.all_reduce(t, op=d.ReduceOp.SUM)
    return float(t.item())


def aggregate_throughput(units_local: float, seconds_local: float) -> float:
    """Whole-job throughput of independent replicas: all units processed / slowest rank's time."""
    return sum_over_ranks(units_local) / max_over_ranks(seconds_local)
