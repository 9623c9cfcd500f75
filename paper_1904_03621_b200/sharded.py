"""Range sharding over ranks (the paper only speculates about several GPUs).

Configurations are independent, so the state space [0, 2^N) is cut into `world` contiguous aligned ranges, one per
rank (one process per GPU). Each rank runs `ising_lowest_range` on its own range and keeps its own S lowest; the
ONE exchange step of the path is an all-gather of those lists (S x 16 bytes per rank -- a few KB, so NVLink bandwidth
is irrelevant and NCCL's all_gather is the right tool), followed by `ising_merge_lists` on every rank
(the paper's low_en / low_st merge). Every rank ends with the same global list.

This module holds host logic only: the range arithmetic, the collective and the call order. The per-range solver and
the merge are the C-ABI calls of `binding`; they are parameters so that the host logic can be exercised on CPU
(`gloo`, world_size 2) in tests/test_sharded_gloo.py, where no CUDA device exists.
"""
from __future__ import annotations

from typing import Callable, List, Optional, Tuple

RANGE_UNIT_LOG2 = 20     # ising_lowest_range wants q_begin, q_end to be multiples of 2^min(N, 20)


def shard_ranges(N: int, world: int) -> List[Tuple[int, int]]:
    """`world` contiguous ranges covering [0, 2^N), each a multiple of the range unit; sizes differ by at most one
    unit; ranks beyond the number of units get an empty range (q_begin == q_end)."""
    if N < 1 or N > 63:
        raise ValueError("N out of range")
    if world < 1:
        raise ValueError("world must be >= 1")
    unit = 1 << min(N, RANGE_UNIT_LOG2)
    units = (1 << N) // unit
    base, extra = divmod(units, world)
    out, cur = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((cur * unit, (cur + n) * unit))
        cur += n
    assert cur == units
    return out


def local_quota(S: int, q_begin: int, q_end: int) -> int:
    """A rank cannot return more states than its range holds."""
    return max(0, min(S, q_end - q_begin))


def ising_lowest_sharded(J, h, S: int, group=None, solver: Optional[Callable] = None,
                         merger: Optional[Callable] = None, device=None, always_exchange: bool = False):
    """The S lowest (E, q) of the whole space, computed by all ranks of `group` together.

    J, h: the instance (identical on every rank). Returns (states, energies) tensors of length S on every rank.
    solver(J, h, S_local, q_begin, q_end) -> (states int64[S_local], energies float64[S_local]) tensors;
    merger(states int64[n], energies float64[n], S) -> (states[S], energies[S]).
    Defaults: the C-ABI calls `binding.ising_lowest_range` / `binding.ising_merge_lists` (CUDA; no CPU fallback).
    always_exchange: run the all-gather and the merge even with a single rank (exercises the collective path on a
    one-GPU box).
    """
    import torch
    import torch.distributed as dist

    if solver is None or merger is None:
        from . import binding
        solver = solver or binding.ising_lowest_range
        merger = merger or binding.ising_merge_lists
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    N = len(h)
    if S < 1 or S > (1 << N):
        raise ValueError("S out of range")
    ranges = shard_ranges(N, world)
    q_begin, q_end = ranges[rank]
    n_local = local_quota(S, q_begin, q_end)
    if n_local > 0:
        st, en = solver(J, h, n_local, q_begin, q_end)
        dev = st.device
    else:
        dev = torch.device(device) if device is not None else torch.device("cpu")
        st = torch.empty(0, dtype=torch.int64, device=dev)
        en = torch.empty(0, dtype=torch.float64, device=dev)
    if world == 1 and not (always_exchange and dist.is_initialized()):
        return st, en
    # fixed-size exchange: every rank sends S slots, the unused tail is cut off again by the known quotas
    send_q = torch.zeros(S, dtype=torch.int64, device=dev)
    send_e = torch.full((S,), float("inf"), dtype=torch.float64, device=dev)
    send_q[:n_local] = st
    send_e[:n_local] = en
    all_q = [torch.empty_like(send_q) for _ in range(world)]
    all_e = [torch.empty_like(send_e) for _ in range(world)]
    dist.all_gather(all_q, send_q, group=group)
    dist.all_gather(all_e, send_e, group=group)
    quotas = [local_quota(S, a, b) for a, b in ranges]
    cat_q = torch.cat([t[:n] for t, n in zip(all_q, quotas)])
    cat_e = torch.cat([t[:n] for t, n in zip(all_e, quotas)])
    return merger(cat_q, cat_e, S)
