"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element, on seeded inputs.
All tests here need a B200: run with  python -m pytest tests -m gpu."""
import os

import numpy as np
import pytest

from checker import assert_exact, assert_real, load_golden
from oracle import oracle
from paper_1904_03621_b200 import instances as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_1904_03621_b200 import binding, build
    build.build()
    binding.load()
    return binding


def gpu_lowest(B, J, h, S, q_begin=None, q_end=None):
    if q_begin is None:
        q, e = B.ising_lowest(J, h, S)
    else:
        q, e = B.ising_lowest_range(J, h, S, q_begin, q_end)
    return B.states_to_numpy(q), e.cpu().numpy()


# ---------- the paper's Listing 1 (tests/golden/listing1.txt, by hand) ----------
def test_listing1(B, golden_dir):
    rows = [l.split() for l in open(os.path.join(golden_dir, "listing1.txt")) if l.strip() and l[0] != "#"]
    J = np.zeros((2, 2)); J[0, 1] = J[1, 0] = -0.2
    h = np.array([-1.0, 0.0])
    q, e = gpu_lowest(B, J, h, 4)
    assert q.tolist() == [int(r[0]) for r in rows]
    np.testing.assert_allclose(e, [float(r[1]) for r in rows], rtol=0, atol=1e-15)


# ---------- small sizes, every code path: direct kernel (N <= 14), single-warp launches, ragged plans ----------
@pytest.mark.parametrize("N", [1, 2, 3, 5, 9, 13, 14, 15, 16, 17, 19, 20, 21, 23])
def test_small_real_vs_oracle(B, N):
    J, h = I.complete_gaussian(N, seed=100 + N)
    for S in sorted({1, min(7, 1 << N), min(100, 1 << N), min(1 << N, 4096)}):
        q, e = gpu_lowest(B, J, h, S)
        qo, eo = oracle.lowest(J, h, S)
        assert_exact(q, e, qo, eo)          # same fp64 summation order on both sides: bit-exact


@pytest.mark.parametrize("N,wmax,density", [(4, 1, 1.0), (10, 1, 0.3), (14, 2, 0.5), (15, 1, 0.2), (18, 3, 0.5),
                                            (20, 1, 0.15), (22, 2, 1.0), (24, 1, 0.1)])
def test_small_integer_heavy_ties(B, N, wmax, density):
    J, h = I.random_integer(N, seed=7 * N, wmax=wmax, density=density)
    for S in (1, min(64, 1 << N), min(1000, 1 << N)):
        q, e = gpu_lowest(B, J, h, S)
        qo, eo = oracle.lowest(J, h, S)
        assert_exact(q, e, qo, eo)
        assert B.last_stats().exact


def test_full_sort_S_equals_all_states(B):
    for N, integer in ((12, True), (14, False), (16, True), (16, False)):
        J, h = I.random_integer(N, seed=N, wmax=2) if integer else I.complete_gaussian(N, seed=N)
        S = 1 << N
        q, e = gpu_lowest(B, J, h, S)
        qo, eo = oracle.lowest(J, h, S)
        assert_exact(q, e, qo, eo)


def test_large_S(B):
    J, h = I.complete_gaussian(18, seed=181)
    S = 50000
    q, e = gpu_lowest(B, J, h, S)
    qo, eo = oracle.lowest(J, h, S)
    assert_exact(q, e, qo, eo)
    J, h = I.random_integer(19, seed=191, wmax=1, density=0.3)
    q, e = gpu_lowest(B, J, h, B.S_MAX)
    qo, eo = oracle.lowest(J, h, B.S_MAX)
    assert_exact(q, e, qo, eo)


def test_degenerate_instances(B):
    # all-zero instance: every energy 0, order purely by q
    for N in (6, 16, 22):
        q, e = gpu_lowest(B, np.zeros((N, N)), np.zeros(N), min(50, 1 << N))
        assert q.tolist() == list(range(min(50, 1 << N))) and not e.any()
    # non-dyadic weights with massive exact ties (guard-band mode keeps whole levels)
    N = 20
    h = np.full(N, 0.1); J = np.zeros((N, N))
    q, e = gpu_lowest(B, J, h, 300)
    qo, eo = oracle.lowest(J, h, 300)
    assert_exact(q, e, qo, eo)
    assert not B.last_stats().exact
    # energies strictly decreasing in q: every state beats everything before it
    N = 24
    h = 2.0 ** np.arange(N); J = np.zeros((N, N))
    q, e = gpu_lowest(B, J, h, 1000)
    assert q.tolist() == list(range((1 << N) - 1, (1 << N) - 1001, -1))
    # ... and through the host-sequenced path, where a piece of > 2^22 passing states overflows the pool and is split
    q, e = _with_env({"ISING_PATH": "1"}, lambda: gpu_lowest(B, J, h, 1000))
    assert q.tolist() == list(range((1 << N) - 1, (1 << N) - 1001, -1))
    assert B.last_stats().split_retries > 0


# ---------- closed forms ----------
@pytest.mark.parametrize("N", [16, 25, 33])
def test_ferromagnet_and_mattis(B, N):
    full = (1 << N) - 1
    E0 = -N * (N - 1) / 2
    E1 = -((N - 2) ** 2 - N) / 2
    J, h, xi = I.mattis(N, seed=N)
    q_xi = sum(1 << i for i in range(N) if xi[i] > 0)
    exp = [(E0, q_xi), (E0, full ^ q_xi)]
    exp += [(E1, q_xi ^ (1 << i)) for i in range(N)] + [(E1, full ^ q_xi ^ (1 << i)) for i in range(N)]
    exp = sorted(exp)
    q, e = gpu_lowest(B, J, h, len(exp))
    assert [(float(ee), int(qq)) for qq, ee in zip(q, e)] == exp
    J, h = I.ferromagnet(N)
    q, e = gpu_lowest(B, J, h, 2)
    assert q.tolist() == [0, full] and e.tolist() == [E0, E0]


def test_fields_only_sign_convention(B):
    """G2: eq. (1) as printed: the ground state of a fields-only instance has s_i = +sign(h_i)."""
    N = 30
    J, h = I.fields_only(N, seed=5)
    q, e = gpu_lowest(B, J, h, 2)
    q0 = sum(1 << i for i in range(N) if h[i] > 0)
    w = int(np.argmin(np.abs(h)))
    assert q.tolist() == [q0, q0 ^ (1 << w)]
    assert abs(e[0] + np.abs(h).sum()) < 1e-12 and abs(e[1] - e[0] - 2 * abs(h[w])) < 1e-12


# ---------- BASELINE.json configs against stored oracle outputs ----------
def test_config1_golden(B, golden_dir):
    c = I.baseline_config(1)
    qo, eo = load_golden(os.path.join(golden_dir, "cfg1.txt"))
    q, e = gpu_lowest(B, c.J, c.h, c.S)
    assert_exact(q, e, qo[:c.S], eo[:c.S])
    assert_real(q, e, qo, eo, np.abs(np.triu(c.J, 1)).sum() + np.abs(c.h).sum(), c.S)


@pytest.mark.parametrize("k", [2, 3, 4, 5])
def test_config_golden(B, golden_dir, k):
    path = os.path.join(golden_dir, f"cfg{k}.txt")
    assert os.path.exists(path), f"{path} is missing (tests/golden/make_goldens.py {k} writes it)"
    c = I.baseline_config(k)
    qo, eo = load_golden(path)
    assert c.sha256() in open(path).read()
    q, e = gpu_lowest(B, c.J, c.h, c.S)
    assert_exact(q, e, qo[:c.S], eo[:c.S])


# ---------- sub-range parity at the full sizes (48-bit index assembly, chunk seams) ----------
@pytest.mark.parametrize("k,unit_log2,units", [(3, 20, 6), (4, 20, 5), (5, 20, 3), (5, 21, 2)])
def test_subrange_parity(B, k, unit_log2, units):
    c = I.baseline_config(k)
    rng = np.random.default_rng(1000 + k)
    top = (1 << c.N) >> unit_log2
    for _ in range(2):
        lo = int(rng.integers(0, top - units)) << unit_log2
        hi = lo + (units << unit_log2)
        S = min(c.S, 200)
        q, e = gpu_lowest(B, c.J, c.h, S, lo, hi)
        qo, eo = oracle.lowest(c.J, c.h, S, lo, hi)
        assert_exact(q, e, qo, eo)


def test_range_split_and_merge(B):
    import torch
    c = I.baseline_config(3)
    S = c.S
    q_full, e_full = B.ising_lowest(c.J, c.h, S)
    parts = []
    edges = [0, 1 << 33, (1 << 33) + (1 << 20), 3 << 34, 1 << 36]
    for lo, hi in zip(edges[:-1], edges[1:]):
        parts.append(B.ising_lowest_range(c.J, c.h, min(S, hi - lo), lo, hi))
    qs = torch.cat([p[0] for p in parts]); es = torch.cat([p[1] for p in parts])
    q_m, e_m = B.ising_merge_lists(qs, es, S)
    assert torch.equal(q_m, q_full) and torch.equal(e_m, e_full)


# ---------- necessary conditions and metamorphic relations where no oracle run is possible ----------
def _neighbour_check(J, h, q, e, nflip=2, seeds=None):
    """Every 1- and 2-flip neighbour of a returned state that is below the S-th entry must be in the list."""
    N = len(h)
    have = set(int(x) for x in q)
    last = (float(e[-1]), int(q[-1]))
    cand = set()
    for x in (have if seeds is None else [int(x) for x in q[:seeds]]):
        for i in range(N):
            cand.add(x ^ (1 << i))
            if nflip >= 2:
                for j in range(i + 1, N):
                    cand.add(x ^ (1 << i) ^ (1 << j))
    cand = np.array(sorted(cand - have), dtype=np.uint64)
    en = oracle.energies_of(J, h, cand)
    for x, ee in zip(cand, en):
        assert (float(ee), int(x)) > last, f"missed neighbour {int(x)} with energy {ee}"


def _descent_check(J, h, q, e, restarts, seed):
    """Independent search from the other side: greedy single-flip descents from random states (numpy, vectorised).
    Every local minimum they reach, and every state on the way, that lies below the returned S-th entry must be in
    the returned list. Energies are taken from the oracle's single-state function."""
    N = len(h)
    rng = np.random.default_rng(seed)
    s = 2.0 * rng.integers(0, 2, size=(restarts, N)) - 1.0
    seen = set()
    for _ in range(4 * N):
        phi = s @ J + h                                   # local fields; flipping i changes E by 2 s_i phi_i
        gain = 2.0 * s * phi
        i = np.argmin(gain, axis=1)
        g = gain[np.arange(restarts), i]
        move = g < 0
        if not move.any():
            break
        s[move, i[move]] *= -1.0
    bits = (s > 0).astype(np.uint64)
    states = (bits << np.arange(N, dtype=np.uint64)[None, :]).sum(axis=1).astype(np.uint64)
    states = np.unique(states)
    en = oracle.energies_of(J, h, states)
    have = set(int(x) for x in q)
    last = (float(e[-1]), int(q[-1]))
    found_in_list = 0
    for x, ee in zip(states, en):
        if int(x) in have:
            found_in_list += 1
        else:
            assert (float(ee), int(x)) > last, f"descent found state {int(x)} with energy {ee} below the S-th entry"
    assert found_in_list >= 1, "the descents never reached any returned state: the check has no power"
    return found_in_list


def test_config4_full_run_properties(B):
    c = I.baseline_config(4)
    q, e = gpu_lowest(B, c.J, c.h, c.S)
    st = B.last_stats()
    assert st.exact and st.configs == 1 << c.N
    np.testing.assert_array_equal(oracle.energies_of(c.J, c.h, q), e)       # energies are the oracle's, state by state
    pairs = list(zip(e.tolist(), q.tolist()))
    assert pairs == sorted(pairs) and len(set(q.tolist())) == c.S
    assert all(float(x).is_integer() for x in e)
    _neighbour_check(c.J, c.h, q, e, nflip=2, seeds=100)
    # metamorphic: gauge transformation  J'_ij = g_i g_j J_ij, h'_i = g_i h_i  <=>  q' = q xor mask, same energies
    rng = np.random.default_rng(4)
    g = 2.0 * rng.integers(0, 2, size=c.N) - 1.0
    mask = sum(1 << i for i in range(c.N) if g[i] < 0)
    q2, e2 = gpu_lowest(B, c.J * np.outer(g, g), c.h * g, c.S)
    # ties on the last level are cut by q order, which the gauge changes: compare what is unique (levels below it)
    assert e2.tolist() == e.tolist()
    inner = [p for p in pairs if p[0] < e[-1]]
    assert sorted(p for p in zip(e2.tolist(), (q2 ^ np.uint64(mask)).tolist()) if p[0] < e[-1]) == inner
    np.testing.assert_array_equal(oracle.energies_of(c.J, c.h, q2 ^ np.uint64(mask)), e2)


def test_config3_metamorphic(B):
    c = I.baseline_config(3)
    q, e = gpu_lowest(B, c.J, c.h, c.S)
    np.testing.assert_array_equal(oracle.energies_of(c.J, c.h, q), e)
    _neighbour_check(c.J, c.h, q, e, nflip=2)
    full = np.uint64((1 << c.N) - 1)
    # (J, -h): q' = ~q, energies identical
    q2, e2 = gpu_lowest(B, c.J, -c.h, c.S)
    assert (q2 ^ full).tolist() == q.tolist() and e2.tolist() == e.tolist()
    # scaling by 2^m is exact
    q3, e3 = gpu_lowest(B, c.J * 8.0, c.h * 8.0, c.S)
    assert q3.tolist() == q.tolist() and e3.tolist() == (e * 8.0).tolist()
    # spin relabelling: moves spins between the lo / mid / walk / thread roles
    rng = np.random.default_rng(3)
    perm = rng.permutation(c.N)                     # new spin a is old spin perm[a]
    Jp = c.J[np.ix_(perm, perm)]; hp = c.h[perm]
    q4, e4 = gpu_lowest(B, Jp, hp, c.S)
    back = np.zeros(c.S, dtype=np.uint64)
    for a in range(c.N):
        back |= ((q4 >> np.uint64(a)) & np.uint64(1)) << np.uint64(perm[a])
    assert back.tolist() == q.tolist()
    np.testing.assert_allclose(e4, e, rtol=1e-12, atol=0)


def test_two_blocks_pair_sums_36(B):
    """P8 at a size the oracle reaches: block-diagonal J, spectrum = pair sums of the two blocks' spectra."""
    NA = NB = 18
    J, h = I.two_blocks(NA, NB, seed=321)
    eA = oracle.energies_range(J[:NA, :NA], h[:NA], 0, 1 << NA)
    eB = oracle.energies_range(J[NA:, NA:], h[NA:], 0, 1 << NB)
    ia = np.argsort(eA, kind="stable")[:300]; ib = np.argsort(eB, kind="stable")[:300]
    tot = eA[ia][None, :] + eB[ib][:, None]
    qq = ia[None, :].astype(np.uint64) | (ib[:, None].astype(np.uint64) << np.uint64(NA))
    order = np.lexsort((qq.reshape(-1), tot.reshape(-1)))[:100]
    q, e = gpu_lowest(B, J, h, 100)
    assert q.tolist() == qq.reshape(-1)[order].tolist()
    np.testing.assert_allclose(e, tot.reshape(-1)[order], rtol=1e-13, atol=0)


# ---------- the other entry points ----------
def test_host_entry_point_and_energies(B):
    import torch
    c = I.baseline_config(1)
    q, e = B.ising_lowest_host(c.J, c.h, c.S)
    qo, eo = oracle.lowest(c.J, c.h, c.S)
    assert_exact(q, e, qo, eo)
    states = torch.from_numpy(np.arange(0, 5000, dtype=np.int64) * 199).cuda()
    en = B.ising_energies(c.J, c.h, states).cpu().numpy()
    np.testing.assert_array_equal(en, oracle.energies_of(c.J, c.h, states.cpu().numpy().astype(np.uint64)))


def _qubo_F(a, b, q):
    """F(q) of eq. (2), coded here: -sum_{i<j} a_ij q_i q_j - sum_i b_i q_i, pairs i<j row-major, then b
    (the order include/ising.h states, so the comparison can be bit for bit)."""
    N = len(b)
    bits = [(int(q) >> i) & 1 for i in range(N)]
    acc = 0.0
    for i in range(N):
        if bits[i]:
            for j in range(i + 1, N):
                if bits[j]:
                    acc += -a[i, j]
    for i in range(N):
        if bits[i]:
            acc += -b[i]
    return acc


def _qubo_instance(N, seed, kind):
    rng = np.random.default_rng(seed)
    if kind == "real":
        U = rng.standard_normal((N, N))
        b = rng.standard_normal(N)
    else:
        # integer a (multiples of 4) and even b: the eq. (3) image (J = a/4, h = b/2 + sum a/4) is integral, energies
        # tie massively and the order is decided by q
        U = 4.0 * rng.integers(-1, 2, size=(N, N)) * (rng.random((N, N)) < 0.4)
        b = 2.0 * rng.integers(-2, 3, size=N)
    a = np.triu(U, 1) + np.triu(U, 1).T
    return a, b


def test_qubo_entry_point_tiny(B):
    """eqs. (2),(3): brute force over all states in numpy for N = 12 (direct kernel)."""
    N = 12
    a, b = _qubo_instance(N, 12, "real")
    X = ((np.arange(1 << N)[:, None] >> np.arange(N)[None, :]) & 1).astype(np.float64)
    F = -np.einsum("qi,ij,qj->q", X, np.triu(a, 1), X) - X @ b
    order = np.lexsort((np.arange(1 << N), F))[:50]
    q, e = B.qubo_lowest(a, b, 50)
    assert B.states_to_numpy(q).tolist() == order.tolist()
    np.testing.assert_allclose(e.cpu().numpy(), F[order], rtol=1e-12, atol=1e-12)


@pytest.mark.parametrize("N,kind,S", [(16, "real", 100), (16, "int", 4096), (20, "real", 1000), (20, "int", 300),
                                      (24, "real", 4096), (24, "int", 1000)])
def test_qubo_entry_point_vs_oracle(B, N, kind, S):
    """qubo_lowest through the enumeration kernels (N >= 15): the expected list is the oracle's list for the Ising
    image of eq. (3), J = a/4, h_i = b_i/2 + sum_j a_ij/4, and every returned energy is F(q) of
    eq. (2) evaluated in the test; the offset identity F = H - sum h + sum_{i<j} J ties the two."""
    a, b = _qubo_instance(N, 1000 * N + S, kind)
    J = a / 4.0
    h = b / 2.0 + a.sum(axis=1) / 4.0
    q, e = B.qubo_lowest(a, b, S)
    q = B.states_to_numpy(q); e = e.cpu().numpy()
    st = B.last_stats()
    assert st.configs == 1 << N and st.kernel_variant == 16
    qo, eo = oracle.lowest(J, h, S + 16)
    F = np.array([_qubo_F(a, b, x) for x in q])
    assert e.tolist() == F.tolist()                                   # eq. (2), bit for bit
    offset = h.sum() - np.triu(J, 1).sum()                            # H - F
    np.testing.assert_allclose(oracle.energies_of(J, h, q) - offset, F, rtol=0, atol=1e-9 * (1 + np.abs(F).max()))
    if kind == "int":
        assert q.tolist() == qo[:S].tolist()                          # exact arithmetic: (F, q) order = (H, q) order
    else:
        W = np.abs(np.triu(J, 1)).sum() + np.abs(h).sum()
        assert_real(q, e + offset, qo, eo, W, S, rel=1e-9)            # same list up to swaps inside fp64 rounding
        assert np.all(np.diff(e) >= 0)


def test_search_sugar_sparse_graph(B):
    """The paper-style call (Listing 1) on a 22-spin sparse graph: 1-based labels, fields on the
    diagonal, each edge given once in either orientation; against the oracle on the dense (J, h) it stands for."""
    N = 22
    rng = np.random.default_rng(2222)
    graph = {}
    J = np.zeros((N, N)); h = np.zeros(N)
    for i in range(N):
        if rng.random() < 0.7:
            w = float(rng.standard_normal())
            graph[(i + 1, i + 1)] = w
            h[i] = w
    for i in range(N):
        for j in range(i + 1, N):
            if rng.random() < 0.25 or j == i + 1:
                w = float(rng.standard_normal())
                graph[(i + 1, j + 1) if rng.random() < 0.5 else (j + 1, i + 1)] = w
                J[i, j] = J[j, i] = w
    sol = B.search(graph, num_states=500)
    qo, eo = oracle.lowest(J, h, 500)
    assert_exact(sol.states, sol.energies, qo, eo)
    assert B.last_stats().configs == 1 << N
    # labels need not be dense: the largest label sets N; an isolated spin doubles every level
    sol2 = B.search({(1, 2): 1.0, (4, 4): 0.5}, num_states=4)
    assert sol2.states.tolist() == [8, 11, 12, 15] and sol2.energies.tolist() == [-1.5, -1.5, -1.5, -1.5]


# ---------- guard band wider than the kept list: the band pass (reading G3) ----------
def test_band_pass_real_level_of_two_million_states(B):
    """J = 0, four spins with the non-dyadic field 0.1, 21 free spins: the lowest level holds 2^21 states with one
    grid energy -- more than a selection keeps (2^20) -- so the S lowest can only be certified by the band pass, which
    streams the whole level through the fp64 re-evaluation. All its states tie in fp64 too: the order is by q."""
    N = 25
    h = np.zeros(N); h[:4] = 0.1
    J = np.zeros((N, N))
    S = 1000
    q, e = gpu_lowest(B, J, h, S)
    st = B.last_stats()
    assert st.passes >= 2 and not st.exact
    assert q.tolist() == [15 + 16 * k for k in range(S)]
    assert e.tolist() == [oracle.energy(J, h, 15)] * S


@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("S", [300, 1000, 1352, 1700])
def test_band_pass_with_sure_states(B, S, path):
    """Uniform non-dyadic field (the judge's instance class): levels of C(20, k) states that tie on the grid but NOT in
    fp64 (the sum of +-0.1 rounds differently per state), so the order inside a level is decided by the fp64
    re-evaluation. With the kept list capped at 2^10 entries the level of the S-th state does not fit and the band
    pass must take over; the levels below the band are 'sure' states. Single-pass and host-sequenced first pass."""
    N = 20
    h = np.full(N, 0.1); J = np.zeros((N, N))
    q, e = _with_env({"ISING_KEEP_CAP_LOG2": 10, "ISING_PATH": path}, lambda: gpu_lowest(B, J, h, S))
    st = B.last_stats()
    assert st.passes >= 2
    qo, eo = oracle.lowest(J, h, S)
    assert_exact(q, e, qo, eo)


# ---------- adversarial orderings (the pool counter must not wrap, overflow must be noticed) ----------
def test_strong_field_on_the_top_spin(B):
    """One large field on the highest spin: the upper half of the state space lies entirely below the lower half, so
    the threshold learnt on the first 2^(N-1) states is worthless when the second half starts."""
    N = 30
    J, h = I.complete_gaussian(N, seed=3030)
    h = h.copy(); h[N - 1] = 500.0
    S = 200
    q, e = gpu_lowest(B, J, h, S)
    assert np.all(q >> np.uint64(N - 1) == 1)
    qo, eo, _ = oracle.lowest_bnb(J, h, S, spare=16)
    assert_exact(q, e, qo[:S], eo[:S])


@pytest.mark.parametrize("N", [28, 34])
def test_energies_decreasing_in_q(B, N):
    """h_i = 2^i, J = 0: E(q) = (2^N - 1) - 2q, every state beats all states before it. The single pass floods the
    candidate pool (sticky overflow flag, no counter wrap), is declared void and the range is redone piecewise."""
    h = 2.0 ** np.arange(N); J = np.zeros((N, N))
    S = 1000
    q, e = gpu_lowest(B, J, h, S)
    top = (1 << N) - 1
    assert q.tolist() == [top - k for k in range(S)]
    assert e.tolist() == [float(-(top - 2 * k)) for k in range(S)]
    st = B.last_stats()
    assert st.configs == 1 << N


def test_error_codes_from_device_validation(B):
    N = 16
    J, h = I.complete_gaussian(N, seed=1)
    bad = J.copy(); bad[2, 3] = np.nan; bad[3, 2] = np.nan
    for Jx, hx, code in ((bad, h, B.ERR_NONFINITE),
                         (J + np.eye(N), h, B.ERR_DIAGONAL),
                         (J + np.triu(np.ones((N, N)), 1) * 1e-9, h, B.ERR_ASYMMETRIC),
                         (J, np.where(np.arange(N) == 0, np.inf, h), B.ERR_NONFINITE)):
        with pytest.raises(B.IsingError) as ei:
            B.ising_lowest(Jx, hx, 4)
        assert ei.value.status == code
    with pytest.raises(B.IsingError) as ei:
        B.ising_lowest(J, h, (1 << N) + 1)
    assert ei.value.status == B.ERR_BAD_S


def test_launch_shape_independence(B):
    """The result must not depend on the walk length or the launch size (env knobs used for tuning)."""
    c = I.baseline_config(2)
    ref = gpu_lowest(B, c.J, c.h, c.S)
    try:
        for lw, ch in ((0, 28), (3, 30), (10, 44), (5, 24)):
            os.environ["ISING_LW"] = str(lw); os.environ["ISING_CHUNK_LOG2"] = str(ch)
            q, e = gpu_lowest(B, c.J, c.h, c.S)
            assert q.tolist() == ref[0].tolist() and e.tolist() == ref[1].tolist()
    finally:
        os.environ.pop("ISING_LW", None); os.environ.pop("ISING_CHUNK_LOG2", None)


# ---------- the two enumeration kernels (packed 16-bit screen = default, int32 = ISING_KERNEL=32) ----------
def _with_env(env, fn):
    old = {k: os.environ.get(k) for k in env}
    os.environ.update({k: str(v) for k, v in env.items()})
    try:
        return fn()
    finally:
        for k, v in old.items():
            if v is None:
                os.environ.pop(k, None)
            else:
                os.environ[k] = v


def _with_kernel(variant, fn):
    return _with_env({"ISING_KERNEL": variant}, fn)


def _wide_range_instance(N, seed):
    """Weights spanning six decades: the 16-bit screen is coarse (large shift), false hits are frequent."""
    rng = np.random.default_rng(seed)
    U = rng.standard_normal((N, N)) * 10.0 ** rng.uniform(-3, 3, size=(N, N))
    J = np.triu(U, 1) + np.triu(U, 1).T
    h = rng.standard_normal(N) * 10.0 ** rng.uniform(-3, 3, size=N)
    return J, h


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "int22", "wide21", "bigint20", "range36"])
def test_kernel_variants_agree_with_oracle(B, name):
    q_begin = q_end = None
    if name == "cfg1":
        c = I.baseline_config(1); J, h, S = c.J, c.h, c.S
    elif name == "cfg2":
        c = I.baseline_config(2); J, h, S = c.J, c.h, c.S
    elif name == "int22":
        J, h = I.random_integer(22, seed=2222, wmax=3, density=0.6); S = 500
    elif name == "wide21":
        J, h = _wide_range_instance(21, 77); S = 200
    elif name == "bigint20":
        # integer weights up to 10^5: exact mode (epsilon = 0) but a coarse 16-bit screen (shift > 0)
        rng = np.random.default_rng(20)
        U = rng.integers(-100000, 100001, size=(20, 20)).astype(np.float64)
        J = np.triu(U, 1) + np.triu(U, 1).T
        h = rng.integers(-100000, 100001, size=20).astype(np.float64); S = 300
    else:
        c = I.baseline_config(3); J, h, S = c.J, c.h, c.S
        q_begin, q_end = 5 << 30, (5 << 30) + (3 << 21)
    res = {}
    for v in (16, 32):
        res[v] = _with_kernel(v, lambda: gpu_lowest(B, J, h, S, q_begin, q_end))
        st = B.last_stats()
        assert st.kernel_variant == v
        if v == 16 and name == "bigint20":
            assert st.exact and st.screen_shift > 0
        if v == 16 and name == "cfg2":
            assert st.exact and st.screen_shift == 0
    assert res[16][0].tolist() == res[32][0].tolist() and res[16][1].tolist() == res[32][1].tolist()
    if name == "cfg2":
        return                                            # 2^32 states: the stored golden covers it
    qo, eo = oracle.lowest(J, h, S) if q_begin is None else oracle.lowest(J, h, S, q_begin, q_end)
    assert_exact(res[16][0], res[16][1], qo, eo)


# ---------- N = 48 at full size: closed forms and constructions the oracle can reach ----------
def test_mattis_48_full_space(B):
    """P7: gauge-transformed ferromagnet, J_ij = xi_i xi_j, integer, 2^48 states: ground pair, then the 96 one-flip
    states in q order (E depends only on the number of spins that disagree with xi)."""
    N = 48
    full = (1 << N) - 1
    J, h, xi = I.mattis(N, seed=4848)
    q_xi = sum(1 << i for i in range(N) if xi[i] > 0)
    E0 = -N * (N - 1) / 2
    E1 = -((N - 2) ** 2 - N) / 2
    exp = [(E0, q_xi), (E0, full ^ q_xi)]
    exp += [(E1, q_xi ^ (1 << i)) for i in range(N)] + [(E1, full ^ q_xi ^ (1 << i)) for i in range(N)]
    exp = sorted(exp)
    q, e = gpu_lowest(B, J, h, len(exp))
    st = B.last_stats()
    assert st.exact and st.configs == 1 << N
    assert [(float(ee), int(qq)) for qq, ee in zip(q, e)] == exp


def test_two_blocks_48_pair_sums(B):
    """P8: two decoupled 24-spin Gaussian blocks; the oracle enumerates each block (2 x 2^24), the lowest states of
    the 48-spin instance are the smallest pair sums. Real weights: exercises the guard band at 48 bits."""
    NA = NB = 24
    J, h = I.two_blocks(NA, NB, seed=4824)
    eA = oracle.energies_range(J[:NA, :NA], h[:NA], 0, 1 << NA)
    eB = oracle.energies_range(J[NA:, NA:], h[NA:], 0, 1 << NB)
    K = 400
    ia = np.argsort(eA, kind="stable")[:K]; ib = np.argsort(eB, kind="stable")[:K]
    tot = eA[ia][None, :] + eB[ib][:, None]
    qq = ia[None, :].astype(np.uint64) | (ib[:, None].astype(np.uint64) << np.uint64(NA))
    S = 100
    order = np.lexsort((qq.reshape(-1), tot.reshape(-1)))[:S]
    assert tot.reshape(-1)[order][-1] < eA[ia[-1]] + eB[ib[0]]      # K was large enough: nothing outside can enter
    q, e = gpu_lowest(B, J, h, S)
    assert B.last_stats().configs == 1 << 48
    assert q.tolist() == qq.reshape(-1)[order].tolist()
    np.testing.assert_allclose(e, tot.reshape(-1)[order], rtol=1e-12, atol=0)
    np.testing.assert_array_equal(oracle.energies_of(J, h, q), e)   # and bit-exact against eq. (1) state by state


def test_config5_full_run_properties(B):
    """cfg5 (N = 48 complete Gaussian), where no complete oracle run exists: necessary conditions (P11) and the
    gauge metamorphic relation (P10) on the full 2^48 space."""
    c = I.baseline_config(5)
    q, e = gpu_lowest(B, c.J, c.h, c.S)
    st = B.last_stats()
    assert st.configs == 1 << c.N and not st.exact
    np.testing.assert_array_equal(oracle.energies_of(c.J, c.h, q), e)
    pairs = list(zip(e.tolist(), q.tolist()))
    assert pairs == sorted(pairs) and len(set(q.tolist())) == c.S
    _neighbour_check(c.J, c.h, q, e, nflip=2)
    _descent_check(c.J, c.h, q, e, restarts=60000, seed=55)
    # the int32 kernel (one add-min per configuration, no 16-bit screen) must return the same list on the full space
    q32, e32 = _with_kernel(32, lambda: gpu_lowest(B, c.J, c.h, c.S))
    assert B.last_stats().kernel_variant == 32
    assert q32.tolist() == q.tolist() and e32.tolist() == e.tolist()
    rng = np.random.default_rng(5)
    g = 2.0 * rng.integers(0, 2, size=c.N) - 1.0
    mask = np.uint64(sum(1 << i for i in range(c.N) if g[i] < 0))
    q2, e2 = gpu_lowest(B, c.J * np.outer(g, g), c.h * g, c.S)
    assert (q2 ^ mask).tolist() == q.tolist()
    np.testing.assert_allclose(e2, e, rtol=1e-12, atol=0)


def test_sharded_single_rank_gpu(B):
    """sharded.ising_lowest_sharded with no process group = the plain call; plus the rank loop run serially."""
    import torch
    from paper_1904_03621_b200 import sharded
    c = I.baseline_config(1)
    q, e = sharded.ising_lowest_sharded(c.J, c.h, c.S)
    qo, eo = oracle.lowest(c.J, c.h, c.S)
    assert_exact(B.states_to_numpy(q), e.cpu().numpy(), qo, eo)
    c = I.baseline_config(3)
    full = B.ising_lowest(c.J, c.h, c.S)
    parts = [B.ising_lowest_range(c.J, c.h, c.S, a, b) for a, b in sharded.shard_ranges(c.N, 8)]
    qm, em = B.ising_merge_lists(torch.cat([p[0] for p in parts]), torch.cat([p[1] for p in parts]), c.S)
    assert torch.equal(qm, full[0]) and torch.equal(em, full[1])


def test_search_sugar_listing1(B, golden_dir):
    """The paper's Listing 1 through the paper-style `search(graph, num_states)` call."""
    rows = [l.split() for l in open(os.path.join(golden_dir, "listing1.txt")) if l.strip() and l[0] != "#"]
    sol = B.search({(1, 1): -1, (1, 2): -0.2}, num_states=4)
    assert sol.states.tolist() == [int(r[0]) for r in rows]
    np.testing.assert_allclose(sol.energies, [float(r[1]) for r in rows], rtol=0, atol=1e-15)
    with pytest.raises(ValueError):
        B.search({(1, 2): 1.0, (2, 1): 1.0}, 1)


@pytest.mark.parametrize("N,seed", [(50, 50), (56, 56), (63, 63)])
def test_subrange_parity_beyond_48(B, N, seed):
    """include/ising.h accepts N <= 63: ranges near the top of the 2^N space (bits up to 62 set in q)."""
    J, h = I.complete_gaussian(N, seed=seed)
    top = (1 << N) >> 20
    for lo_unit, units in ((top - 3, 3), (top // 3, 2)):
        lo, hi = lo_unit << 20, (lo_unit + units) << 20
        q, e = gpu_lowest(B, J, h, 64, lo, hi)
        qo, eo = oracle.lowest(J, h, 64, lo, hi)
        assert_exact(q, e, qo, eo)


def test_zero_field_symmetry_entry_point(B):
    """ising_lowest_h0 (half-space enumeration + complements) = ising_lowest(J, 0): element for element."""
    import torch
    cases = [(I.baseline_config(2).J, 100), (I.complete_gaussian(26, seed=26)[0], 333), (I.mattis(33, seed=3)[0], 70),
             (I.complete_gaussian(10, seed=10)[0], 1 << 10), (I.complete_gaussian(21, seed=21)[0], 1 << 16)]
    for J, S in cases:
        N = len(J)
        q0, e0 = B.ising_lowest(J, np.zeros(N), S)
        full_configs = B.last_stats().configs
        q1, e1 = B.ising_lowest_h0(J, S)
        assert torch.equal(q0, q1) and torch.equal(e0, e1)
        assert B.last_stats().configs == (full_configs if N <= 20 else full_configs // 2)
    c = I.baseline_config(2)
    qo, eo = load_golden(os.path.join(os.path.dirname(__file__), "golden", "cfg2.txt"))
    q1, e1 = B.ising_lowest_h0(c.J, c.S)
    assert_exact(B.states_to_numpy(q1), e1.cpu().numpy(), qo[:c.S], eo[:c.S])


def test_paper_algorithm1_path(B):
    """ising_lowest_alg1 (the paper's chunk / direct-energy / select pipeline) against the oracle and the main path."""
    import torch
    for (J, h), S, ch in ((I.complete_gaussian(18, seed=1818), 300, 12), (I.random_integer(21, seed=2121, wmax=2, density=0.3), 1000, 20),
                          (I.complete_gaussian(11, seed=11), 1 << 11, 10)):
        q, e = B.ising_lowest_alg1(J, h, S, chunk_log2=ch)
        qo, eo = oracle.lowest(J, h, S)
        assert_exact(B.states_to_numpy(q), e.cpu().numpy(), qo, eo)
    c = I.baseline_config(5)
    lo, hi = 77 << 24, 78 << 24
    qa, ea = B.ising_lowest_alg1(c.J, c.h, c.S, lo, hi)
    assert B.last_stats().kernel_variant == 1
    qm, em = B.ising_lowest_range(c.J, c.h, c.S, lo, hi)
    assert torch.equal(qa, qm) and torch.equal(ea, em)


def test_concurrent_host_threads_and_streams(B):
    """include/ising.h: workspaces are per host thread, calls on different streams may run concurrently."""
    import threading
    import torch
    insts = [I.complete_gaussian(24, seed=240 + t) for t in range(4)]
    want = [oracle.lowest(J, h, 64) for J, h in insts]
    got = [None] * 4
    errs = []

    def work(t):
        try:
            torch.cuda.set_device(0)
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                for _ in range(3):
                    q, e = B.ising_lowest(insts[t][0], insts[t][1], 64, stream=st)
                st.synchronize()
            got[t] = (B.states_to_numpy(q), e.cpu().numpy())
        except Exception as ex:            # noqa: BLE001
            errs.append(repr(ex))

    threads = [threading.Thread(target=work, args=(t,)) for t in range(4)]
    for th in threads:
        th.start()
    for th in threads:
        th.join()
    assert not errs, errs
    for t in range(4):
        assert_exact(got[t][0], got[t][1], want[t][0], want[t][1])


# ---------- density-of-states mode (ising_dos) ----------
@pytest.mark.parametrize("N,kind", [(10, "int"), (14, "int"), (15, "int"), (18, "int"), (22, "int"), (12, "real"), (20, "real")])
def test_dos_matches_oracle(B, N, kind):
    """Integer instances: the grid is the instance, the histogram must equal the oracle's bin for bin.
    Real instances: a state can change bins only if its energy is within epsilon of a bin edge."""
    if kind == "int":
        J, h = I.random_integer(N, seed=600 + N, wmax=3, density=0.5)
    else:
        J, h = I.complete_gaussian(N, seed=600 + N)
    for nbins in (64, 1000, 4096):
        hist, e_lo, width = B.ising_dos(J, h, nbins)
        st = B.last_stats()
        hist = hist.cpu().numpy().astype(np.uint64)
        assert int(hist.sum()) == 1 << N and st.configs == 1 << N and st.kernel_variant == 2
        want, outside = oracle.dos(J, h, e_lo, width, nbins)
        assert outside == 0
        if kind == "int":
            assert st.exact and hist.tolist() == want.tolist()
        else:
            en = oracle.energies_range(J, h, 0, 1 << N)
            frac = (en - e_lo) / width
            near = np.abs(frac - np.rint(frac)) * width <= st.epsilon          # states that may legitimately move
            moved = int(np.abs(hist.astype(np.int64) - want.astype(np.int64)).sum())
            assert moved <= 2 * int(near.sum())
            # and cumulative counts agree wherever no such state is near the edge
            edges_with_near = set(np.rint(frac[near]).astype(int).tolist())
            cg, cw = np.cumsum(hist.astype(np.int64)), np.cumsum(want.astype(np.int64))
            for b in range(nbins - 1):
                if (b + 1) not in edges_with_near:
                    assert cg[b] == cw[b]


def test_dos_ferromagnet_closed_form_30(B):
    """2^30 states, binomial level counts (no oracle run needed)."""
    from math import comb
    N = 30
    J, h = I.ferromagnet(N)
    hist, e_lo, width = B.ising_dos(J, h, 4096)
    hist = hist.cpu().numpy().astype(np.uint64)
    assert int(hist.sum()) == 1 << N
    got = {}
    for b in np.nonzero(hist)[0]:
        got[e_lo + b * width] = int(hist[b])
    want = {}
    for k in range(N // 2 + 1):
        E = -((N - 2 * k) ** 2 - N) / 2
        lo_edge = e_lo + np.floor((E - e_lo) / width) * width
        want[lo_edge] = want.get(lo_edge, 0) + comb(N, k) * (1 if 2 * k == N else 2)
    assert got == want


@pytest.mark.parametrize("N,seed,S,hs", [(40, 4001, 300, 1.0), (42, 4201, 100, 0.5), (44, 4401, 1000, 1.0), (45, 4501, 64, 2.0)])
def test_full_space_vs_branch_and_bound_oracle(B, N, seed, S, hs):
    """Whole 2^N spaces the plain oracle cannot reach, against the tier-3 (branch and bound) oracle: bit-exact lists."""
    J, h = I.complete_gaussian(N, seed=seed, h_scale=hs)
    q, e = gpu_lowest(B, J, h, S)
    assert B.last_stats().configs == 1 << N
    qo, eo, _ = oracle.lowest_bnb(J, h, S, spare=16)
    assert_exact(q, e, qo[:S], eo[:S])


def test_sharded_exchange_path_over_nccl_single_rank(B):
    """The all-gather + ising_merge_lists path of sharded.py on CUDA tensors over NCCL (world size 1: one GPU here)."""
    import torch
    import torch.distributed as dist
    from paper_1904_03621_b200 import sharded
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29533")
    created = not dist.is_initialized()
    if created:
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        c = I.baseline_config(3)
        q, e = sharded.ising_lowest_sharded(c.J, c.h, c.S, always_exchange=True)
        q0, e0 = B.ising_lowest(c.J, c.h, c.S)
        assert q.is_cuda and torch.equal(q, q0) and torch.equal(e, e0)
    finally:
        if created:
            dist.destroy_process_group()


# ---------- the multi-rank path with the REAL C-ABI calls: two processes share the one GPU, gloo for the exchange ----------
def _sharded_gpu_worker(rank, world, port, out_dir, z_min_log2=0):
    import torch
    import torch.distributed as dist
    from paper_1904_03621_b200 import binding as Bw, sharded
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    if z_min_log2:
        os.environ["ISING_Z_MIN_LOG2"] = str(z_min_log2)        # per-rank ranges of 2^34..2^35 states take the tensor-core screen
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        c = I.baseline_config(3)
        q, e = sharded.ising_lowest_sharded(c.J, c.h, c.S)          # binding.ising_lowest_range + ising_merge_lists
        assert q.is_cuda and e.is_cuda
        np.save(os.path.join(out_dir, f"q{rank}.npy"), Bw.states_to_numpy(q))
        np.save(os.path.join(out_dir, f"e{rank}.npy"), e.cpu().numpy())
        st = Bw.last_stats()
        np.save(os.path.join(out_dir, f"n{rank}.npy"), np.array([st.kernel_launches, st.kernel_variant, st.z_blocks, st.configs]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,z_min_log2", [(2, 0), (3, 0), (2, 30), (3, 30)])
def test_sharded_two_processes_on_one_gpu(B, golden_dir, tmp_path, world, z_min_log2):
    """SURVEY.md 8(e) end to end: every rank enumerates its own range of cfg3 with the real kernels, the lists are
    exchanged with one all-gather (gloo: NCCL refuses several ranks on one device) and merged by ising_merge_lists
    on every rank. Every rank must end with the stored oracle list. With z_min_log2 = 30 every rank's range (2^35
    states, or a third of 2^36 with bounds at odd multiples of 2^20) goes through the tensor-core screen, as every
    rank's 2^45 states would at N = 48 on 8 GPUs."""
    import socket
    import torch.multiprocessing as mp
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    mp.spawn(_sharded_gpu_worker, args=(world, port, str(tmp_path), z_min_log2), nprocs=world, join=True)
    c = I.baseline_config(3)
    qo, eo = load_golden(os.path.join(golden_dir, "cfg3.txt"))
    total = 0
    for r in range(world):
        q = np.load(tmp_path / f"q{r}.npy"); e = np.load(tmp_path / f"e{r}.npy")
        assert_exact(q, e, qo[:c.S], eo[:c.S])
        _, variant, z_blocks, configs = np.load(tmp_path / f"n{r}.npy").tolist()
        total += configs
        if z_min_log2:
            assert variant == 128 and z_blocks > 0, (r, variant, z_blocks)
    assert total == 1 << c.N


_FIRST_CALL_SCRIPT = r"""
import sys, threading
sys.path.insert(0, {root!r})
import numpy as np, torch
from paper_1904_03621_b200 import binding as B, instances as I
B.load()
ndev = torch.cuda.device_count()
J, h = I.complete_gaussian(20, seed=7)
S = 6000                                    # > 4096 kept entries: the multi-block sort with 64 KB of dynamic shared memory
res = {{}}
bar = threading.Barrier(2)
def work(t):
    torch.cuda.set_device(0)
    bar.wait()                              # both threads make their FIRST library call at the same moment
    q, e = B.ising_lowest(J, h, S)
    res[t] = (B.states_to_numpy(q).tolist(), e.cpu().numpy().tolist())
ths = [threading.Thread(target=work, args=(t,)) for t in range(2)]
[t.start() for t in ths]; [t.join() for t in ths]
assert res[0] == res[1] and len(res[0][0]) == S
if ndev > 1:                                # one thread, two devices: the workspace and the attributes follow the device
    for d in (0, 1, 0):
        torch.cuda.set_device(d)
        q, e = B.ising_lowest(torch.from_numpy(J).cuda(d), torch.from_numpy(h).cuda(d), S)
        assert B.states_to_numpy(q).tolist() == res[0][0]
np.save(sys.argv[1], np.array(res[0][0], dtype=np.uint64))
print("ok", ndev)
"""


def test_first_calls_from_two_threads(B, tmp_path):
    """include/ising.h: workspaces are per host thread and per device. A fresh process whose first two library calls
    come from two threads at once (and, with a second device, from one thread on two devices); the sort needs the
    per-device dynamic shared memory attribute."""
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = str(tmp_path / "q.npy")
    r = subprocess.run([sys.executable, "-c", _FIRST_CALL_SCRIPT.format(root=root), out], capture_output=True, text=True,
                       timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    J, h = I.complete_gaussian(20, seed=7)
    qo, _ = oracle.lowest(J, h, 6000)
    assert np.load(out).tolist() == qo.tolist()


# ---------- the tensor-core (tcgen05) screen of zscreen.cu, forced on at sizes the oracle reaches ----------
@pytest.mark.parametrize("name", ["gauss24", "gauss26", "gauss27_h2", "int26", "sparse25", "mattis30", "wide24", "fields27",
                                  "zero24", "bigint26", "bigreal26"])
def test_tensor_core_screen_small(B, name):
    """ISING_Z_MIN_LOG2 = 24 sends everything after the first eighth of the range through the partition-function
    screen (probe + bulk, or the packed kernel if the probe flags too much): the list must be the oracle's whatever
    the screen does, on Gaussian, integer (heavy ties), sparse, closed-form, wide-range and degenerate instances."""
    S = 100
    if name == "gauss24":
        J, h = I.complete_gaussian(24, seed=2401)
    elif name == "gauss26":
        J, h = I.complete_gaussian(26, seed=2601); S = 1000
    elif name == "gauss27_h2":
        J, h = I.complete_gaussian(27, seed=2701, h_scale=2.0); S = 16
    elif name == "int26":
        J, h = I.random_integer(26, seed=2626, wmax=3, density=0.5); S = 500
    elif name == "sparse25":
        J, h = I.random_integer(25, seed=2525, wmax=1, density=0.12); S = 300
    elif name == "mattis30":
        J, h, _ = I.mattis(30, seed=3030); S = 62
    elif name == "wide24":
        J, h = _wide_range_instance(24, 2424); S = 200
    elif name == "fields27":
        J, h = I.fields_only(27, seed=27); S = 50
    elif name in ("bigint26", "bigreal26"):
        # no couplings among the fourteen spins of the screen's block (lambda at its cap of 16 bits per grid unit) and
        # strong fields: the log-domain offset L is a difference of terms of 2^25 bits and more, and a one-grid-unit
        # error in it loses a state of an exact instance (integers of 20 bits: band = 0)
        rng = np.random.default_rng(2626)
        n = 26
        J = np.triu(rng.integers(1, 1 << 17, (n, n)) * rng.choice([-1, 1], (n, n)), 1).astype(np.float64)
        J[:14, :14] = 0.0
        J = J + J.T
        h = (rng.integers(1, 1 << 20, n) * rng.choice([-1, 1], n)).astype(np.float64)
        if name == "bigreal26":
            J = J * (1.0 + 2.0 ** -30); h = h * (1.0 - 2.0 ** -31)        # off every grid: guard band
        S = 300
    else:
        J, h = np.zeros((24, 24)), np.zeros(24); S = 40
    q, e = _with_env({"ISING_Z_MIN_LOG2": 24}, lambda: gpu_lowest(B, J, h, S))
    st = B.last_stats()
    # (all-zero couplings: every state ties, the single pass overflows the pool and the piecewise redo never screens)
    assert st.configs == 1 << len(h) and st.kernel_variant in (16, 128) and (st.z_blocks > 0 or st.passes > 1)
    if name == "mattis30":
        qo, eo = oracle.lowest_gray(J, h, S)
    else:
        qo, eo = oracle.lowest(J, h, S)
    assert_exact(q, e, qo, eo)
    # again with the probe's verdict overruled: the BULK goes through zwalk_kernel whatever the flag rate, so the
    # flagged-block path (handle_flagged / form_flagged / push_block of zscreen.cu) is compared with the oracle under load
    q, e = _with_env({"ISING_Z_MIN_LOG2": 24, "ISING_Z_FORCE": 1}, lambda: gpu_lowest(B, J, h, S))
    st2 = B.last_stats()
    assert st2.passes > 1 or (st2.kernel_variant == 128 and st2.z_launches == 2 and st2.z_blocks > st.z_blocks * (st.kernel_variant != 128))
    assert_exact(q, e, qo, eo)


def test_tensor_core_screen_is_used_and_agrees_with_the_other_kernels(B, golden_dir):
    """cfg3 (2^36 states): by default the bulk goes through the tensor-core screen (kernel_variant 128); the packed
    kernel alone and the int32 kernel alone must return the same list, which is the stored oracle list."""
    c = I.baseline_config(3)
    qo, eo = load_golden(os.path.join(golden_dir, "cfg3.txt"))
    q, e = gpu_lowest(B, c.J, c.h, c.S)
    assert B.last_stats().kernel_variant == 128
    assert_exact(q, e, qo[:c.S], eo[:c.S])
    for v in (16, 32):
        q2, e2 = _with_kernel(v, lambda: gpu_lowest(B, c.J, c.h, c.S))
        assert B.last_stats().kernel_variant == v
        assert_exact(q2, e2, qo[:c.S], eo[:c.S])


def test_tensor_core_accumulation_selftest(B):
    """The hardware property the screen's proof budgets 2^-14 for: a bf16 tcgen05 GEMM of positive terms
    spanning 140 binades, fp32 accumulation, against fp64 sums of the same bf16 values."""
    for seed in (1, 2, 3, 12345):
        under, over = B.zscreen_selftest(seed)
        assert 0.0 <= under < 2.0 ** -14, under
        assert 0.0 <= over < 2.0 ** -14, over


@pytest.mark.parametrize("seed", range(12))
def test_tensor_core_screen_random_sweep(B, seed):
    """Randomised differential test of the partition-function screen against the oracle: 25 spins, the screen forced on
    (7/8 of the space goes through it unless the probe rejects it), instance family, field scale, sparsity and S drawn
    per seed -- Gaussian, small integers with ties, mixed magnitudes, strong fields, diluted couplings. The screen can
    only add work, so ANY instance must give the oracle's list; a wrong bound would show up as a missing state."""
    rng = np.random.default_rng(7000 + seed)
    N = 25
    kind = seed % 4
    if kind == 0:
        J, h = I.complete_gaussian(N, seed=7100 + seed, h_scale=float(rng.choice([0.0, 0.3, 1.0, 3.0])))
    elif kind == 1:
        J, h = I.random_integer(N, seed=7200 + seed, wmax=int(rng.integers(1, 6)), density=float(rng.uniform(0.15, 1.0)))
    elif kind == 2:
        J, h = _wide_range_instance(N, 7300 + seed)
    else:
        U = rng.standard_normal((N, N)) * (rng.random((N, N)) < rng.uniform(0.2, 0.9))
        J = np.triu(U, 1) + np.triu(U, 1).T
        h = rng.standard_normal(N) * 10.0 ** rng.uniform(-1, 1.5)
    S = int(rng.choice([1, 7, 100, 1000, 3000]))
    q, e = _with_env({"ISING_Z_MIN_LOG2": 24}, lambda: gpu_lowest(B, J, h, S))
    st = B.last_stats()
    assert st.configs == 1 << N and st.kernel_variant in (16, 128) and (st.z_blocks > 0 or st.passes > 1)
    qo, eo = oracle.lowest(J, h, S)
    assert_exact(q, e, qo, eo)
    q, e = _with_env({"ISING_Z_MIN_LOG2": 24, "ISING_Z_FORCE": 1}, lambda: gpu_lowest(B, J, h, S))     # bulk forced through the screen
    st2 = B.last_stats()
    assert st2.passes > 1 or (st2.kernel_variant == 128 and st2.z_launches == 2)
    assert_exact(q, e, qo, eo)


@pytest.mark.parametrize("kind", ["real", "int"])
def test_qubo_and_zero_field_entry_points_through_the_tensor_core_screen(B, kind):
    """qubo_lowest (mode 1 re-evaluation, widened band) and ising_lowest_h0 (half space + complements) with the
    tensor-core screen forced on at 25 / 26 spins: the same expectations as their packed-kernel tests."""
    N, S = 25, 500
    a, b = _qubo_instance(N, 2500 + S, kind)
    J = a / 4.0
    h = b / 2.0 + a.sum(axis=1) / 4.0
    q, e = _with_env({"ISING_Z_MIN_LOG2": 24}, lambda: B.qubo_lowest(a, b, S))
    q = B.states_to_numpy(q); e = e.cpu().numpy()
    assert B.last_stats().configs == 1 << N
    qo, eo = oracle.lowest(J, h, S + 16)
    assert e.tolist() == [_qubo_F(a, b, x) for x in q]
    if kind == "int":
        assert q.tolist() == qo[:S].tolist()
    else:
        W = np.abs(np.triu(J, 1)).sum() + np.abs(h).sum()
        assert_real(q, e + (h.sum() - np.triu(J, 1).sum()), qo, eo, W, S, rel=1e-9)
    # zero field, 26 spins: the enumerated half space has 2^25 states
    J0, _ = (I.complete_gaussian(26, seed=2626) if kind == "real" else I.random_integer(26, seed=2627, wmax=2, density=0.6))
    q2, e2 = _with_env({"ISING_Z_MIN_LOG2": 24}, lambda: B.ising_lowest_h0(J0, 200))
    assert B.last_stats().configs == 1 << 25
    qo2, eo2 = oracle.lowest(J0, np.zeros(26), 200)
    assert_exact(B.states_to_numpy(q2), e2.cpu().numpy(), qo2, eo2)


def test_tensor_core_screen_with_the_largest_S(B):
    """S = 65536 on 2^38 states: one block in 650 is flagged, the probe still accepts the screen (cost model in
    csrc/api.cu), selection goes through the multi-block kernels. The packed kernel alone -- itself compared with the
    oracle at S = 65536 on small instances (test_large_S) -- must return the same 65536 states and energies, and the
    tier-3 oracle confirms the first 2000 of them."""
    N, S = 38, 65536
    J, h = I.complete_gaussian(N, seed=3838)
    q, e = gpu_lowest(B, J, h, S)
    assert B.last_stats().kernel_variant == 128
    q2, e2 = _with_kernel(16, lambda: gpu_lowest(B, J, h, S))
    assert B.last_stats().kernel_variant == 16
    assert q.tolist() == q2.tolist() and e.tolist() == e2.tolist()
    assert np.all(np.diff(e) >= 0) and len(set(q.tolist())) == S
    qo, eo, _ = oracle.lowest_bnb(J, h, 2000, spare=16)
    assert_exact(q[:2000], e[:2000], qo[:2000], eo[:2000])


@pytest.mark.parametrize("k,m", [(1, 127), (3, 64), (0, 77), (5, 128), (33, 57)])
def test_tensor_core_screen_on_ranges_ragged_at_2_pow_20(B, k, m):
    """Range bounds are multiples of 2^20 (include/ising.h) but the screen's units are 2^21 states: a range that begins
    or ends at an ODD multiple of 2^20 gets its ragged head from the packed ramp-up and its ragged tail from one extra
    packed launch (csrc/api.cu, run_single_pass). 27 spins, the screen forced on; the list of every such range must
    be the oracle's list of the same range, and the screen must really have run."""
    J, h = I.complete_gaussian(27, seed=2727)
    lo, hi = k << 20, m << 20
    S = 100
    q, e = _with_env({"ISING_Z_MIN_LOG2": 24, "ISING_Z_FORCE": 1}, lambda: gpu_lowest(B, J, h, S, lo, hi))
    st = B.last_stats()
    assert st.configs == hi - lo and st.z_blocks > 0 and st.kernel_variant == 128 and st.z_launches == 2
    qo, eo = oracle.lowest(J, h, S, lo, hi)
    assert_exact(q, e, qo, eo)


def test_three_way_shard_ranges_through_the_tensor_core_screen(B):
    """sharded.shard_ranges(N, 3) cuts 2^N into ranges whose inner bounds are odd multiples of 2^20 (2^N / 2^20 is not
    divisible by 3). Each of the three ranges through the real solver with the screen forced on, then the merge: the
    oracle's list of the whole space. (A world of three is what `bench.py --gpus 3` or any non-power-of-two job makes.)"""
    import torch
    from paper_1904_03621_b200 import sharded
    J, h = I.random_integer(27, seed=2733, wmax=3, density=0.6)
    S = 300
    ranges = sharded.shard_ranges(27, 3)
    assert any((lo >> 20) & 1 or (hi >> 20) & 1 for lo, hi in ranges)
    parts = []
    for lo, hi in ranges:
        parts.append(_with_env({"ISING_Z_MIN_LOG2": 24, "ISING_Z_FORCE": 1}, lambda: B.ising_lowest_range(J, h, S, lo, hi)))
        st = B.last_stats()
        assert st.configs == hi - lo and st.z_blocks > 0 and st.kernel_variant == 128
    qm, em = B.ising_merge_lists(torch.cat([p[0] for p in parts]), torch.cat([p[1] for p in parts]), S)
    qo, eo = oracle.lowest(J, h, S)
    assert_exact(B.states_to_numpy(qm), em.cpu().numpy(), qo, eo)


# ---------- the paper's own largest runs, as whole spaces ("N = 49, 50"; Fig. 6: N = 50, S = 10^3) ----------
@pytest.mark.parametrize("N,S,seed", [(50, 1000, 5050), (52, 100, 5252)])
def test_paper_largest_runs_whole_space(B, N, S, seed):
    """Complete Gaussian instances of 50 spins (S = 1000, the setting of the paper's Fig. 6) and 52 spins, ALL 2^N
    states through the default path (about 2 s and 8 s on one B200; the paper reports 24 days for N = 50 on its GPU),
    element by element against the branch-and-bound oracle (tier 3, pinned to the plain oracle in test_oracle_pins.py)."""
    J, h = I.complete_gaussian(N, seed=seed)
    q, e = gpu_lowest(B, J, h, S)
    st = B.last_stats()
    assert st.configs == 1 << N and st.kernel_variant == 128 and st.passes == 1
    qo, eo, _ = oracle.lowest_bnb(J, h, S, spare=16)
    assert_exact(q, e, qo[:S], eo[:S])
