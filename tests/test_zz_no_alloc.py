"""ising_merge_lists_static: the list merge for callers that cannot allocate on the device.

Some users of this library run inside a process whose GPU memory is already spoken for -- a framework pool that
reserved the whole device at start-up -- or on a thread that must not trigger cudaMalloc's device-wide
synchronisation while other streams are busy. Every other compute entry point builds a ~130 MiB workspace with
cudaMalloc on a thread's first call; `ising_merge_lists_static` sorts in a fixed 2 MiB array that is part of the
library image instead (include/ising.h, csrc/merge_static.cu) and accepts at most 131072 input pairs.

What is checked: its output equals that of the allocating path `ising_merge_lists` bit for bit (the bar every merge
test in this suite uses: states and fp64 bit patterns) on calls made back to back -- the array is shared and keeps
the previous call's entries, so a large merge is followed by a small one that would pick up stale entries if the
padding were wrong -- plus the size limit's error, and that a call leaves the device's free memory where it was.

This file sorts last on purpose (pytest -x stops at the first failure: a problem here must not hide the parity
tests), and it passes alone in a fresh process -- where the static entry point is the first thing that touches the
GPU, before any workspace exists -- as well as after the rest of the suite."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_1904_03621_b200 import binding, build
    build.build()
    binding.load()
    return binding


def _lists(n, seed, levels):
    """n seeded (state, energy) pairs shaped like concatenated per-range results: distinct 48-bit states, energies
    drawn from `levels` distinct values (heavy ties, so the order among equal energies -- by state -- is exercised),
    both signs and a few zeros of either sign."""
    import torch
    rng = np.random.default_rng(seed)
    q = rng.choice(1 << 48, size=n, replace=False).astype(np.int64)
    vals = np.concatenate([rng.normal(size=levels - 2) * 37.0, [0.0, -0.0]])
    e = vals[rng.integers(0, levels, size=n)]
    return torch.from_numpy(q).cuda(), torch.from_numpy(e).cuda()


def _expected(q, e, S):
    """(energy, state) order written out with numpy: an independent statement of what both entry points return."""
    qn = q.cpu().numpy().view(np.uint64)
    en = e.cpu().numpy() + 0.0
    order = np.lexsort((qn, en))[:S]
    return qn[order], en[order]


def test_static_merge_equals_allocating_merge_on_consecutive_calls(B):
    import torch
    # (n, S): several sort tiles with a ragged tail; then a small single-tile merge into the same, now dirty, array;
    # then the largest size the entry point takes; then small again
    cases = [(100_000, 5_000, 11), (3_000, 3_000, 12), (B.MERGE_STATIC_MAX, 65_536, 13), (77, 5, 14)]
    inputs = [(_lists(n, seed, levels=max(3, n // 50)), S) for n, S, seed in cases]
    static = []
    for (q, e), S in inputs:                                   # the calls under test, back to back
        static.append(B.ising_merge_lists_static(q, e, S))
    for ((q, e), S), (qs, es) in zip(inputs, static):
        qa, ea = B.ising_merge_lists(q, e, S)                  # the existing path (allocates its workspace)
        assert torch.equal(qs, qa), "states differ from ising_merge_lists"
        assert torch.equal(es.view(torch.int64), ea.view(torch.int64)), "energies differ from ising_merge_lists (bit patterns)"
        qx, ex = _expected(q, e, S)
        assert B.states_to_numpy(qs).tolist() == qx.tolist()
        assert (es.cpu().numpy() + 0.0).tolist() == ex.tolist()


def test_static_merge_refuses_more_than_its_array_holds(B):
    import torch
    n = B.MERGE_STATIC_MAX + 1
    q = torch.arange(n, dtype=torch.int64, device="cuda")
    e = torch.zeros(n, dtype=torch.float64, device="cuda")
    with pytest.raises(B.IsingError) as info:
        B.ising_merge_lists_static(q, e, 10)
    assert info.value.status == B.ERR_BAD_S
    assert str(B.MERGE_STATIC_MAX) in str(info.value) and "ISING_MERGE_STATIC_MAX" in str(info.value)
    with pytest.raises(B.IsingError):
        B.ising_merge_lists_static(q[:10], e[:10], 11)        # S > n, as for ising_merge_lists


def test_static_merge_leaves_free_device_memory_alone(B):
    """With caller-owned outputs a call must not change the device's free memory (the allocating path's workspace is
    over 130 MiB; the allowance here is 1 MiB for anything the driver does on its own)."""
    import torch
    (q, e), S = _lists(50_000, 21, levels=500), 1_000
    out = (torch.empty(S, dtype=torch.int64, device="cuda"), torch.empty(S, dtype=torch.float64, device="cuda"))
    B.ising_merge_lists_static(q, e, S, out=out)               # first call on the device: set-up, kernels loaded
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    B.ising_merge_lists_static(q, e, S, out=out)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_before - free_after < (1 << 20), (free_before, free_after)
    qx, ex = _expected(q, e, S)
    assert B.states_to_numpy(out[0]).tolist() == qx.tolist() and (out[1].cpu().numpy() + 0.0).tolist() == ex.tolist()
