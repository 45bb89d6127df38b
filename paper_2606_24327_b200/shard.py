"""Marker sharding for N ranks (one process per GPU).  The push has no exchange step: markers are independent
(PAPER.md L81, L91), mesh and field tables are replicated, so ranks share nothing on the data path and the
job is weak-scaled - every rank owns the same number of markers, a disjoint slice of one counter-based
population (synth.make_markers(cfg, n, start))."""
from __future__ import annotations


def marker_slice(n_per_rank: int, rank: int, world: int):
    """[start, stop) of rank's markers in the global population of n_per_rank * world markers."""
    if not (0 <= rank < world) or n_per_rank < 0:
        raise ValueError("bad rank/world")
    return rank * n_per_rank, (rank + 1) * n_per_rank


def job_rate(units_per_rank: int, world: int, max_seconds: float) -> float:
    """Whole-job throughput: all ranks' units divided by the slowest rank's time."""
    return units_per_rank * world / max_seconds


def reduce_max_seconds(seconds: float, dist=None) -> float:
    """MAX over ranks of a device-measured duration (torch.distributed all_reduce); identity without a group."""
    if dist is None or not dist.is_initialized():
        return seconds
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([seconds], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def broadcast_fields(backend, dist, src: int = 0):
    """The one collective of a multi-rank run: rank `src` has run fields_set; its coefficient table is
    exported into a byte buffer, broadcast (NCCL over NVLink for CUDA buffers) and imported by every other rank.
    `backend` needs fields_export() -> buffer and fields_import(buffer); returns the bytes moved."""
    rank = dist.get_rank()
    buf = backend.fields_export()
    dist.broadcast(buf, src=src)
    if rank != src:
        backend.fields_import(buf)
    return int(buf.numel() * buf.element_size())
