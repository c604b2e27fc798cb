"""Multi-GPU plumbing: banks = (stream, layer, KV head) are independent, so N GPUs
run N states over disjoint slices of one of those axes with NO collective on the data path.  This module holds the
host logic only: which slice a rank owns, how a rank cuts its slice out of the token-major ABI tensors, and the
max-over-ranks reduction of device timings that bench.py reports.  No ProtoKV arithmetic here.
"""
from __future__ import annotations

from typing import Dict, Sequence, Tuple

import torch

AXES = ("stream", "layer", "kv_head")


def shard_range(n: int, world: int, rank: int) -> Tuple[int, int]:
    """Contiguous [begin, end) of `n` units owned by `rank`: sizes differ by at most one, lower ranks get the extra."""
    if not (world >= 1 and 0 <= rank < world):
        raise ValueError(f"bad rank {rank} of world {world}")
    base, extra = divmod(n, world)
    begin = rank * base + min(rank, extra)
    return begin, begin + base + (1 if rank < extra else 0)


def shard_config(n_streams: int, n_layers: int, n_q_heads: int, n_kv_heads: int, world: int, rank: int,
                 axis: str = "stream") -> Dict[str, int]:
    """The rank-local (n_streams, n_layers, n_q_heads, n_kv_heads) and the offset of the slice on `axis`.
    Sharding KV heads keeps the GQA group intact: query head h belongs to KV head h // group."""
    if axis not in AXES:
        raise ValueError(f"axis must be one of {AXES}")
    group = n_q_heads // n_kv_heads
    n = dict(stream=n_streams, layer=n_layers, kv_head=n_kv_heads)[axis]
    if world > n:
        raise ValueError(f"cannot shard {n} {axis}s over {world} ranks")
    b, e = shard_range(n, world, rank)
    out = dict(n_streams=n_streams, n_layers=n_layers, n_q_heads=n_q_heads, n_kv_heads=n_kv_heads, begin=b, end=e, axis=axis)
    if axis == "stream":
        out["n_streams"] = e - b
    elif axis == "layer":
        out["n_layers"] = e - b
    else:
        out["n_kv_heads"] = e - b
        out["n_q_heads"] = (e - b) * group
    return out


def slice_kv(x: torch.Tensor, sh: Dict[str, int]) -> torch.Tensor:
    """K or V [stream][layer][T][H_kv][d] -> the rank's contiguous slice."""
    b, e = sh["begin"], sh["end"]
    if sh["axis"] == "stream":
        return x[b:e].contiguous()
    if sh["axis"] == "layer":
        return x[:, b:e].contiguous()
    return x[:, :, :, b:e].contiguous()


def slice_q(x: torch.Tensor, sh: Dict[str, int], group: int) -> torch.Tensor:
    """Q or out [stream][layer][N_q][H_q][d] -> the rank's contiguous slice (query heads of the rank's KV heads)."""
    b, e = sh["begin"], sh["end"]
    if sh["axis"] == "stream":
        return x[b:e].contiguous()
    if sh["axis"] == "layer":
        return x[:, b:e].contiguous()
    return x[:, :, :, b * group:e * group].contiguous()


def slice_grid_pos(s: torch.Tensor, sh: Dict[str, int]) -> torch.Tensor:
    """grid_pos [stream][T][2]: only a stream shard cuts it."""
    return s[sh["begin"]:sh["end"]].contiguous() if sh["axis"] == "stream" else s


def owned_banks(n_streams: int, n_layers: int, n_kv_heads: int, sh: Dict[str, int]) -> Sequence[int]:
    """Global bank indices ((stream * L + layer) * H_kv + head) of the rank, in the rank-local bank order."""
    rs = range(sh["begin"], sh["end"]) if sh["axis"] == "stream" else range(n_streams)
    rl = range(sh["begin"], sh["end"]) if sh["axis"] == "layer" else range(n_layers)
    rh = range(sh["begin"], sh["end"]) if sh["axis"] == "kv_head" else range(n_kv_heads)
    return [(st * n_layers + la) * n_kv_heads + hd for st in rs for la in rl for hd in rh]


def max_over_ranks(values: Sequence[float], device=None) -> Sequence[float]:
    """Element-wise MAX over the ranks of the default process group (identity without one): the rule for every
    multi-GPU timing (a step is as slow as its slowest rank)."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return list(values)
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def whole_job_rate(units_per_rank: float, max_seconds: float, world: int) -> float:
    """Weak scaling: every rank processes `units_per_rank`; whole-job rate = all units / slowest rank's time."""
    return world * units_per_rank / max_seconds
