"""Host logic of the multi-rank path (paper_1904_03621_b200/sharded.py) on CPU: gloo backend, world_size 2 and 3.
No CUDA here: the per-range solver and the merge are stand-ins built on the CPU oracle (test infrastructure), so what
is under test is the range arithmetic, the exchange and the call order -- the code every GPU rank runs."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1904_03621_b200 import instances as I
from paper_1904_03621_b200 import sharded


def test_shard_ranges_cover_and_align():
    for N in (1, 5, 19, 20, 21, 24, 36, 48):
        for world in (1, 2, 3, 4, 7, 8):
            r = sharded.shard_ranges(N, world)
            assert len(r) == world and r[0][0] == 0 and r[-1][1] == 1 << N
            unit = 1 << min(N, sharded.RANGE_UNIT_LOG2)
            sizes = []
            for (a, b), (c, _) in zip(r, r[1:] + [(1 << N, None)]):
                assert b == c and a <= b and a % unit == 0 and b % unit == 0
                sizes.append(b - a)
            assert max(sizes) - min(sizes) <= unit
    with pytest.raises(ValueError):
        sharded.shard_ranges(0, 2)
    with pytest.raises(ValueError):
        sharded.shard_ranges(10, 0)


def test_local_quota():
    assert sharded.local_quota(100, 0, 16) == 16
    assert sharded.local_quota(100, 1 << 20, 2 << 20) == 100
    assert sharded.local_quota(5, 7, 7) == 0


def _oracle_solver(J, h, S, q_begin, q_end):
    from oracle import oracle
    q, e = oracle.lowest(np.asarray(J), np.asarray(h), S, q_begin, q_end, threads=1)
    return torch.from_numpy(q.astype(np.int64)), torch.from_numpy(e)


def _sort_merger(states, energies, S):
    order = np.lexsort((states.numpy().astype(np.uint64), energies.numpy()))[:S]
    return states[order], energies[order]


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, N, S, seed, integer, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        J, h = I.random_integer(N, seed, wmax=2, density=0.5) if integer else I.complete_gaussian(N, seed)
        q, e = sharded.ising_lowest_sharded(J, h, S, solver=_oracle_solver, merger=_sort_merger)
        np.save(os.path.join(out_dir, f"q{rank}.npy"), q.numpy())
        np.save(os.path.join(out_dir, f"e{rank}.npy"), e.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,N,S,integer", [(2, 21, 50, False), (2, 22, 300, True), (3, 21, 64, True),
                                               (2, 12, 3000, False)])
def test_sharded_matches_single_range(tmp_path, world, N, S, integer):
    """Every rank ends with the oracle's global list (ties by q across the rank seam included)."""
    from oracle import oracle
    seed = 900 + N
    mp.spawn(_worker, args=(world, _free_port(), N, S, seed, integer, str(tmp_path)), nprocs=world, join=True)
    J, h = I.random_integer(N, seed, wmax=2, density=0.5) if integer else I.complete_gaussian(N, seed)
    qo, eo = oracle.lowest(J, h, S)
    for r in range(world):
        q = np.load(tmp_path / f"q{r}.npy").astype(np.uint64)
        e = np.load(tmp_path / f"e{r}.npy")
        assert q.tolist() == qo.tolist()
        assert e.tolist() == eo.tolist()
