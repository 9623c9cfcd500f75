"""Pins for the CPU oracle (oracle/oracle.c) against what the paper and the mathematics fix.

None of these retypes the oracle's own double loop: each expected value comes from a worked example
(Listing 1, by hand), a closed form (ferromagnet / Mattis levels, fields-only, open chain), the
paper's second formulation (QUBO, eqs. (2),(3)), a symmetry, or an independent construction
(pair sums of decoupled blocks, numpy sort of a full spectrum for the selection logic).
"""
import itertools
import os

import numpy as np
import pytest

from oracle import oracle
from paper_1904_03621_b200 import instances as I


def _popcount(x: int) -> int:
    return bin(x).count("1")


# ---------- P1: Listing 1 of the paper, evaluated by hand (tests/golden/listing1.txt) ----------
def test_listing1_by_hand(golden_dir):
    rows = [l.split() for l in open(os.path.join(golden_dir, "listing1.txt")) if l.strip() and l[0] != "#"]
    q_exp = np.array([int(r[0]) for r in rows], dtype=np.uint64)
    e_exp = np.array([float(r[1]) for r in rows])
    J = np.zeros((2, 2)); J[0, 1] = J[1, 0] = -0.2     # (1,2): -0.2
    h = np.array([-1.0, 0.0])                          # (1,1): -1
    q, e = oracle.lowest(J, h, 4)
    assert q.tolist() == q_exp.tolist()
    np.testing.assert_allclose(e, e_exp, rtol=0, atol=1e-15)
    for qq, ee in zip(q_exp, e_exp):
        assert abs(oracle.energy(J, h, int(qq)) - ee) < 1e-15


# ---------- P4: uniform ferromagnet: E = -((N-2k)^2 - N)/2, k = number of up spins ----------
@pytest.mark.parametrize("N", [3, 6, 11, 16])
def test_ferromagnet_closed_form(N):
    J, h = I.ferromagnet(N)
    full = (1 << N) - 1
    assert oracle.energy(J, h, 0) == -N * (N - 1) / 2          # ground energy -N(N-1)/2 (BASELINE.json)
    assert oracle.energy(J, h, full) == -N * (N - 1) / 2       # degeneracy 2
    # every state's energy from its magnetisation
    rng = np.random.default_rng(N)
    for q in rng.integers(0, 1 << N, size=50):
        k = _popcount(int(q))
        assert oracle.energy(J, h, int(q)) == -((N - 2 * k) ** 2 - N) / 2
    # lowest list: the two ground states, then the 2N one-flip states in q order
    S = 2 + 2 * N
    cand = [0, full] + [1 << i for i in range(N)] + [full ^ (1 << i) for i in range(N)]
    E1 = -((N - 2) ** 2 - N) / 2
    exp = sorted(set((-N * (N - 1) / 2 if c in (0, full) else E1, c) for c in cand))
    if N > 3:  # for N=3 one-flip of 000 and of 111 coincide in level with each other only
        q, e = oracle.lowest(J, h, S)
        assert [(ee, int(qq)) for qq, ee in zip(q, e)] == exp[:S]


# ---------- P7: Mattis (gauge-transformed ferromagnet): same levels around q_xi ----------
@pytest.mark.parametrize("N,seed", [(8, 1), (13, 2), (18, 3)])
def test_mattis_closed_form(N, seed):
    J, h, xi = I.mattis(N, seed)
    q_xi = sum(1 << i for i in range(N) if xi[i] > 0)
    full = (1 << N) - 1
    E0 = -N * (N - 1) / 2
    E1 = -((N - 2) ** 2 - N) / 2
    exp = [(E0, q_xi), (E0, full ^ q_xi)]
    exp += [(E1, q_xi ^ (1 << i)) for i in range(N)] + [(E1, full ^ q_xi ^ (1 << i)) for i in range(N)]
    exp = sorted(exp)
    q, e = oracle.lowest(J, h, len(exp))
    assert [(ee, int(qq)) for qq, ee in zip(q, e)] == exp
    # with a field along xi the degeneracy is lifted: E = -((N-2k)^2-N)/2 - c(N-2k)
    c = 0.5
    J, h, xi = I.mattis(N, seed, field=c)
    q, e = oracle.lowest(J, h, 1)
    assert int(q[0]) == q_xi and e[0] == E0 - c * N


# ---------- P5: fields only (G2: eq. (1) literally => s_i = +sign(h_i)) ----------
def test_fields_only_ground_state_and_subset_sums():
    N = 12
    J, h = I.fields_only(N, seed=5, integer=True)
    q0 = sum(1 << i for i in range(N) if h[i] > 0)
    S = 200
    q, e = oracle.lowest(J, h, S)
    assert int(q[0]) == q0 and e[0] == -np.abs(h).sum()
    # excitations: E0 + 2 * (sum of |h_i| over flipped spins); brute force over subsets in python ints
    a = [int(abs(x)) for x in h]
    E0 = -sum(a)
    allp = sorted((E0 + 2 * sum(a[i] for i in range(N) if m >> i & 1), q0 ^ m) for m in range(1 << N))
    assert [(int(ee), int(qq)) for qq, ee in zip(q, e)] == allp[:S]
    # real-valued: ground state and first excitation (flip the weakest field)
    J, h = I.fields_only(48, seed=6)
    q0 = sum(1 << i for i in range(48) if h[i] > 0)
    assert abs(oracle.energy(J, h, q0) + np.abs(h).sum()) < 1e-12
    w = int(np.argmin(np.abs(h)))
    assert abs(oracle.energy(J, h, q0 ^ (1 << w)) - (-np.abs(h).sum() + 2 * abs(h[w]))) < 1e-12
    # the other sign convention would put the ground state at the complement
    assert oracle.energy(J, h, q0) < oracle.energy(J, h, ((1 << 48) - 1) ^ q0)


# ---------- P9: open chain: E0 = -sum|w|, s_{i+1} = s_i sign(w_i) ----------
def test_open_chain():
    N = 14
    J, h, w = I.open_chain(N, seed=9)
    s = [-1]
    for i in range(N - 1):
        s.append(s[-1] * (1 if w[i] > 0 else -1))
    qa = sum(1 << i for i in range(N) if s[i] > 0)
    qb = ((1 << N) - 1) ^ qa
    q, e = oracle.lowest(J, h, 4)
    assert sorted([int(q[0]), int(q[1])]) == sorted([qa, qb]) and int(q[0]) < int(q[1])
    np.testing.assert_allclose(e[:2], -np.abs(w).sum(), rtol=1e-14)
    np.testing.assert_allclose(e[2:4], -np.abs(w).sum() + 2 * np.abs(w).min(), rtol=1e-14)


# ---------- P2: QUBO formulation, eqs. (2),(3), coded separately ----------
def _qubo_F(J, h, q, N):
    a = 4.0 * J
    b = 2.0 * h - 2.0 * J.sum(axis=1)
    x = np.array([(q >> i) & 1 for i in range(N)], dtype=np.float64)
    return -sum(a[i, j] * x[i] * x[j] for i in range(N) for j in range(i + 1, N)) - float(b @ x)


@pytest.mark.parametrize("N", [5, 9])
def test_qubo_offset_identity_all_states(N):
    J, h = I.complete_gaussian(N, seed=40 + N)
    off = h.sum() - np.triu(J, 1).sum()          # H(s) - F(q)
    for q in range(1 << N):
        assert abs(oracle.energy(J, h, q) - _qubo_F(J, h, q, N) - off) < 1e-11


def test_qubo_offset_identity_n48_samples():
    c = I.baseline_config(5)
    off = c.h.sum() - np.triu(c.J, 1).sum()
    rng = np.random.default_rng(0)
    for q in rng.integers(0, 1 << 48, size=20):
        assert abs(oracle.energy(c.J, c.h, int(q)) - _qubo_F(c.J, c.h, int(q), 48) - off) < 1e-9


# ---------- P6: h = 0  =>  E(q) = E(~q) ----------
def test_global_flip_symmetry():
    c = I.baseline_config(2)
    full = (1 << c.N) - 1
    rng = np.random.default_rng(1)
    for q in rng.integers(0, 1 << c.N, size=100):
        assert oracle.energy(c.J, c.h, int(q)) == oracle.energy(c.J, c.h, full ^ int(q))
    J, h = I.random_integer(12, seed=3)
    h[:] = 0
    q, e = oracle.lowest(J, h, 64)
    got = set(int(x) for x in q)
    full = (1 << 12) - 1
    # complement pairs appear together unless cut by the S boundary level
    inner = [int(x) for x, ee in zip(q, e) if ee < e[-1]]
    assert all((full ^ x) in got for x in inner)


# ---------- P3: selection / tie logic against a numpy sort of the full spectrum ----------
@pytest.mark.parametrize("N,integer", [(10, False), (12, True), (14, False), (16, True)])
def test_selection_matches_full_sort(N, integer):
    if integer:
        J, h = I.random_integer(N, seed=N, wmax=2, density=0.5)   # heavy ties
    else:
        J, h = I.complete_gaussian(N, seed=N)
    en = oracle.energies_range(J, h, 0, 1 << N)
    order = np.lexsort((np.arange(1 << N), en))       # by energy, then q
    for S in (1, 7, 100, 1 << N if N <= 12 else 1000):
        q, e = oracle.lowest(J, h, S)
        assert q.tolist() == order[:S].tolist()
        assert e.tolist() == en[order[:S]].tolist()
    # thread count must not matter
    q1, e1 = oracle.lowest(J, h, 50, threads=1)
    q3, e3 = oracle.lowest(J, h, 50, threads=3)
    assert q1.tolist() == q3.tolist() and e1.tolist() == e3.tolist()


def test_range_split_merges_to_full():
    J, h = I.complete_gaussian(14, seed=77)
    S = 40
    q, e = oracle.lowest(J, h, S)
    parts = [oracle.lowest(J, h, S, lo, lo + (1 << 12)) for lo in range(0, 1 << 14, 1 << 12)]
    allq = np.concatenate([p[0] for p in parts]); alle = np.concatenate([p[1] for p in parts])
    order = np.lexsort((allq, alle))[:S]
    assert allq[order].tolist() == q.tolist() and alle[order].tolist() == e.tolist()


# ---------- P8: two decoupled blocks: spectrum = pair sums of the blocks' spectra ----------
def test_two_decoupled_blocks_pair_sums():
    NA, NB = 9, 8
    J, h = I.two_blocks(NA, NB, seed=123)
    eA = oracle.energies_range(J[:NA, :NA], h[:NA], 0, 1 << NA)
    eB = oracle.energies_range(J[NA:, NA:], h[NA:], 0, 1 << NB)
    tot = eA[None, :] + eB[:, None]                    # [qB, qA]; q = qA | qB << NA
    flat = tot.reshape(-1)
    order = np.lexsort((np.arange(flat.size), flat))[:100]
    q, e = oracle.lowest(J, h, 100)
    assert q.tolist() == order.tolist()
    np.testing.assert_allclose(e, flat[order], rtol=0, atol=1e-12)


def test_bad_arguments():
    J, h = I.ferromagnet(4)
    with pytest.raises(ValueError):
        oracle.lowest(J, h, 0)
    with pytest.raises(ValueError):
        oracle.lowest(J, h, 4, 0, 1 << 5)


# ---------- tier-2 oracle (oracle_gray.c, integer instances only) pinned to the plain oracle ----------
@pytest.mark.parametrize("N,wmax,density,S", [(3, 1, 1.0, 8), (8, 3, 1.0, 256), (13, 2, 0.4, 500), (17, 1, 0.2, 1000),
                                              (20, 3, 0.3, 2000), (22, 5, 0.15, 300)])
def test_gray_oracle_equals_plain_oracle(N, wmax, density, S):
    J, h = I.random_integer(N, seed=31 * N + wmax, wmax=wmax, density=density)
    qo, eo = oracle.lowest(J, h, S)
    for slab in sorted({0, 1, min(N, 5), min(N, 11), N}):
        qg, eg = oracle.lowest_gray(J, h, S, slab_bits=slab)
        assert qg.tolist() == qo.tolist() and eg.tolist() == eo.tolist()


def test_gray_oracle_ranges_threads_and_closed_form():
    J, h = I.random_integer(18, seed=99, wmax=2, density=0.5)
    lo, hi = 3 << 14, 11 << 14
    qo, eo = oracle.lowest(J, h, 700, lo, hi)
    for threads in (1, 3):
        qg, eg = oracle.lowest_gray(J, h, 700, lo, hi, slab_bits=12, threads=threads)
        assert qg.tolist() == qo.tolist() and eg.tolist() == eo.tolist()
    # Mattis closed form at a size the plain oracle does not reach quickly (N = 30): ground pair + 2N one-flip states
    N = 30
    J, h, xi = I.mattis(N, seed=7)
    q_xi = sum(1 << i for i in range(N) if xi[i] > 0)
    full = (1 << N) - 1
    E0 = -N * (N - 1) / 2
    E1 = -((N - 2) ** 2 - N) / 2
    exp = sorted([(E0, q_xi), (E0, full ^ q_xi)] + [(E1, q_xi ^ (1 << i)) for i in range(N)]
                 + [(E1, full ^ q_xi ^ (1 << i)) for i in range(N)])
    qg, eg = oracle.lowest_gray(J, h, len(exp))
    assert [(float(e), int(q)) for q, e in zip(qg, eg)] == exp
    with pytest.raises(ValueError):
        oracle.lowest_gray(J + 0.5 * (1 - np.eye(N)), h, 4)          # non-integer weights are refused


def test_gray_oracle_reproduces_config2_golden(golden_dir):
    """Config 2's stored list was written by the PLAIN oracle (358 s); the tier-2 oracle must reproduce it exactly."""
    from checker import load_golden
    c = I.baseline_config(2)
    qo, eo = load_golden(os.path.join(golden_dir, "cfg2.txt"))
    qg, eg = oracle.lowest_gray(c.J, c.h, len(qo), threads=2)
    assert qg.tolist() == qo.tolist() and eg.tolist() == eo.tolist()


# ---------- density of states: closed-form level counts ----------
def test_dos_binomial_levels():
    from math import comb
    N = 14
    # uniform field h_i = 1, no couplings: E = -(N - 2k) for k spins down, C(N, k) states
    hist, outside = oracle.dos(np.zeros((N, N)), np.ones(N), -N - 0.5, 1.0, 2 * N + 1)
    assert outside == 0 and int(hist.sum()) == 1 << N
    for k in range(N + 1):
        assert int(hist[2 * k]) == comb(N, k)              # E = -N + 2k sits in bin 2k
    assert not hist[1::2].any()
    # uniform ferromagnet: E(k) = -((N-2k)^2 - N)/2 shared by k and N-k flipped spins
    J, h = I.ferromagnet(N)
    lo = -N * (N - 1) / 2
    hist, outside = oracle.dos(J, h, lo - 0.5, 1.0, N * (N - 1) // 2 + N // 2 + 2)
    assert outside == 0
    for k in range(N // 2 + 1):
        E = -((N - 2 * k) ** 2 - N) / 2
        want = comb(N, k) * (1 if 2 * k == N else 2)
        assert int(hist[int(E - lo)]) == want
    assert int(hist.sum()) == 1 << N
    # states below the first bin are reported, not counted
    hist, outside = oracle.dos(J, h, lo + 0.5, 1.0, 4096)
    assert outside == 2 and int(hist.sum()) == (1 << N) - 2


# ---------- tier-3 oracle (oracle_bnb.c, exact branch and bound) pinned to the plain oracle ----------
@pytest.mark.parametrize("N,S,kind", [(1, 2, "real"), (4, 16, "real"), (9, 100, "real"), (14, 300, "real"), (18, 64, "real"),
                                      (21, 1000, "real"), (24, 100, "real"), (12, 500, "int"), (20, 200, "int"),
                                      (22, 300, "sparse"), (16, 65536, "real")])
def test_bnb_oracle_equals_plain_oracle(N, S, kind):
    if kind == "real":
        J, h = I.complete_gaussian(N, seed=41 * N + S)
    elif kind == "int":
        J, h = I.random_integer(N, seed=43 * N, wmax=2, density=0.6)          # heavy ties: order decided by q
    else:
        J, h = I.random_integer(N, seed=47 * N, wmax=3, density=0.15)
    qo, eo = oracle.lowest(J, h, S)
    spare = min(16, (1 << N) - S)
    for threads in (1, 4):
        qb, eb, nodes = oracle.lowest_bnb(J, h, S, spare=spare, threads=threads)
        assert len(qb) == S + spare and nodes > 0
        assert qb[:S].tolist() == qo.tolist() and eb[:S].tolist() == eo.tolist()


def test_bnb_oracle_closed_forms_and_goldens(golden_dir):
    from checker import load_golden
    # fields only, N = 40 (2^40 states: out of reach of the plain oracle): ground state and first excitation
    N = 40
    J, h = I.fields_only(N, seed=9)
    qb, eb, _ = oracle.lowest_bnb(J, h, 2, spare=0)
    q0 = sum(1 << i for i in range(N) if h[i] > 0)
    w = int(np.argmin(np.abs(h)))
    assert qb.tolist() == [q0, q0 ^ (1 << w)]
    assert abs(eb[0] + np.abs(h).sum()) < 1e-12 and abs(eb[1] - eb[0] - 2 * abs(h[w])) < 1e-12
    # Mattis N = 34: ground pair + the 2N one-flip states, ties by q
    N = 34
    J, h, xi = I.mattis(N, seed=11)
    q_xi = sum(1 << i for i in range(N) if xi[i] > 0)
    full = (1 << N) - 1
    E0, E1 = -N * (N - 1) / 2, -((N - 2) ** 2 - N) / 2
    exp = sorted([(E0, q_xi), (E0, full ^ q_xi)] + [(E1, q_xi ^ (1 << i)) for i in range(N)]
                 + [(E1, full ^ q_xi ^ (1 << i)) for i in range(N)])
    qb, eb, _ = oracle.lowest_bnb(J, h, len(exp), spare=0)
    assert [(float(e), int(q)) for q, e in zip(qb, eb)] == exp
    # the stored lists written by the plain oracle (configs 1, 3) and by the tier-2 oracle (config 4): S + 16 entries each
    for k in (1, 3, 4):
        c = I.baseline_config(k)
        qo, eo = load_golden(os.path.join(golden_dir, f"cfg{k}.txt"))
        qb, eb, _ = oracle.lowest_bnb(c.J, c.h, c.S, spare=16)
        assert qb.tolist() == qo.tolist() and eb.tolist() == eo.tolist(), f"config {k}"
