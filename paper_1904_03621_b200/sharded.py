"""Range sharding over ranks (the paper only speculates about several GPUs).

Configurations are independent, so the state space [0, 2^N) is cut into `world` contiguous aligned ranges, one per
rank (one process per GPU). Each rank runs `ising_lowest_range` on its own range and keeps its own S lowest; the
ONE exchange step of the path is a single all-gather of those lists -- (q, E) packed into one int64 tensor of
2 S words per rank, a few KB, so NVLink bandwidth is irrelevant and NCCL's all_gather is the right tool -- followed by
`ising_merge_lists` on every rank (the paper's low_en / low_st merge). Every rank ends with the
same global list.

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


def _exchange_device(group, compute_device):
    """Where the all-gather buffers live: NCCL moves CUDA tensors; gloo (CPU tests, or several ranks sharing one GPU)
    moves host tensors, so the packed lists are staged through the host and the merge input goes back to the GPU."""
    import torch
    import torch.distributed as dist
    backend = dist.get_backend(group)
    if backend == "nccl":
        if compute_device is not None and compute_device.type == "cuda":
            return compute_device
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def ising_lowest_sharded(J, h, S: int, group=None, solver: Optional[Callable] = None,
                         merger: Optional[Callable] = None, device=None, always_exchange: bool = False):
    """The S lowest (E, q) of the whole space, computed by all ranks of `group` together.

    J, h: the instance (identical on every rank). Returns (states, energies) tensors of length S on every rank.
    solver(J, h, S_local, q_begin, q_end) -> (states int64[S_local], energies float64[S_local]) tensors;
    merger(states int64[n], energies float64[n], S) -> (states[S], energies[S]).
    Defaults: the C-ABI calls `binding.ising_lowest_range` / `binding.ising_merge_lists` (CUDA; no CPU fallback).
    A merge that must not allocate device memory inside the library: `merger=binding.ising_merge_lists_static`
    (world x S <= 131072 pairs; include/ising.h says which callers need it).
    device: where this rank computes (default: J's device if it is a tensor, else the current CUDA device when the
    default solver is used, else the CPU); a rank with an empty range builds its buffers there.
    always_exchange: run the all-gather and the merge even with a single rank (exercises the collective path on a
    one-GPU box).
    """
    import torch
    import torch.distributed as dist

    default_path = solver is None and merger is None
    if solver is None or merger is None:
        from . import binding
        solver = solver or binding.ising_lowest_range
        merger = merger or binding.ising_merge_lists
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    N = len(h)
    if S < 1 or S > (1 << N):
        raise ValueError("S out of range")
    if device is not None:
        compute_dev = torch.device(device)
    elif isinstance(J, torch.Tensor):
        compute_dev = J.device
    elif default_path:
        compute_dev = torch.device("cuda", torch.cuda.current_device())
    else:
        compute_dev = torch.device("cpu")
    ranges = shard_ranges(N, world)
    q_begin, q_end = ranges[rank]
    n_local = local_quota(S, q_begin, q_end)
    if n_local > 0:
        st, en = solver(J, h, n_local, q_begin, q_end)
        compute_dev = st.device
    else:
        st = torch.empty(0, dtype=torch.int64, device=compute_dev)
        en = torch.empty(0, dtype=torch.float64, device=compute_dev)
    if world == 1 and not (always_exchange and dist.is_initialized()):
        return st, en
    # ONE fixed-size all-gather: every rank sends 2 S int64 words (S state indices, then the S energies' bit
    # patterns); the unused tail is cut off again by the known quotas
    xdev = _exchange_device(group, compute_dev)
    send = torch.zeros(2 * S, dtype=torch.int64, device=xdev)
    send[:n_local] = st.to(xdev)
    send[S:S + n_local] = en.to(xdev).view(torch.int64)
    recv = torch.empty(world * 2 * S, dtype=torch.int64, device=xdev)
    dist.all_gather_into_tensor(recv, send, group=group)
    recv = recv.view(world, 2, S)
    quotas = [local_quota(S, a, b) for a, b in ranges]
    cat_q = torch.cat([recv[r, 0, :n] for r, n in enumerate(quotas)]).to(compute_dev)
    cat_e = torch.cat([recv[r, 1, :n] for r, n in enumerate(quotas)]).view(torch.float64).to(compute_dev)
    return merger(cat_q.contiguous(), cat_e.contiguous(), S)
