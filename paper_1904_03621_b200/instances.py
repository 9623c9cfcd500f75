"""Seeded synthetic Ising instances (inputs only -- none of the method's arithmetic lives here).

This module serves BOTH the CPU oracle's tests and the CUDA path (tests, bench.py, smoke()).
It only draws numbers and lays out graphs; it never evaluates an energy.

The paper's own benchmark instances ("fully connected, K = 100 randomly generated (cf. Ref. [53, 54])",
PAPER.md:187) are not available; the five BASELINE.json configs below stand in for them
(recipe: SURVEY.md section 8(d), restated in DESIGN.md "Input recipe").

Conventions: dense symmetric J (N x N, float64, zero diagonal), separate
field vector h (N, float64); node labels are 0-based; bit i of a state index q is spin i.
"""
from __future__ import annotations

import hashlib
from dataclasses import dataclass

import numpy as np

SEED_BASE = 1904036200


@dataclass(frozen=True)
class Instance:
    name: str
    N: int
    S: int
    J: np.ndarray  # (N, N) float64, symmetric, zero diagonal
    h: np.ndarray  # (N,) float64
    integer: bool  # all weights integral

    def sha256(self) -> str:
        m = hashlib.sha256()
        m.update(np.ascontiguousarray(self.J, dtype="<f8").tobytes())
        m.update(np.ascontiguousarray(self.h, dtype="<f8").tobytes())
        return m.hexdigest()

    @property
    def n_edges(self) -> int:
        return int(np.count_nonzero(np.triu(self.J, 1)))


def _sym_from_edges(N: int, edges, weights) -> np.ndarray:
    J = np.zeros((N, N), dtype=np.float64)
    for (i, j), w in zip(edges, weights):
        assert i != j and J[i, j] == 0.0
        J[i, j] = w
        J[j, i] = w
    return J


def complete_gaussian(N: int, seed: int, h_scale: float = 1.0):
    """Complete graph, J_ij = J_ji ~ N(0,1) for i<j, h_i ~ N(0, h_scale^2)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    U = rng.standard_normal((N, N))
    T = np.triu(U, 1)
    J = T + T.T
    h = h_scale * rng.standard_normal(N)
    return J, h


def chimera_edges(rows: int = 2, cols: int = 2):
    """Chimera graph of rows x cols K_{4,4} unit cells.

    node = 8*(cols*r + c) + 4*side + k, k < 4. Intra-cell: every side-0 node to every side-1 node.
    Vertical couplers join side-0,k of (r,c) with side-0,k of (r+1,c); horizontal couplers join
    side-1,k of (r,c) with side-1,k of (r,c+1).
    """
    def node(r, c, side, k):
        return 8 * (cols * r + c) + 4 * side + k

    edges = set()
    for r in range(rows):
        for c in range(cols):
            for a in range(4):
                for b in range(4):
                    edges.add(tuple(sorted((node(r, c, 0, a), node(r, c, 1, b)))))
            if r + 1 < rows:
                for k in range(4):
                    edges.add(tuple(sorted((node(r, c, 0, k), node(r + 1, c, 0, k)))))
            if c + 1 < cols:
                for k in range(4):
                    edges.add(tuple(sorted((node(r, c, 1, k), node(r, c + 1, 1, k)))))
    return sorted(edges)


def lattice_edges(rows: int, cols: int):
    """Open-boundary square lattice, node = cols*r + c."""
    edges = []
    for r in range(rows):
        for c in range(cols):
            if c + 1 < cols:
                edges.append((cols * r + c, cols * r + c + 1))
            if r + 1 < rows:
                edges.append((cols * r + c, cols * (r + 1) + c))
    return sorted(edges)


def baseline_config(k: int) -> Instance:
    """The k-th (1-based) BASELINE.json config, seed = SEED_BASE + k."""
    seed = SEED_BASE + k
    if k == 1:
        J, h = complete_gaussian(20, seed)
        return Instance("cfg1_N20_complete_gauss", 20, 16, J, h, False)
    if k == 2:
        rng = np.random.Generator(np.random.PCG64(seed))
        edges = chimera_edges(2, 2)
        assert len(edges) == 80
        w = 2.0 * rng.integers(0, 2, size=len(edges)) - 1.0
        J = _sym_from_edges(32, edges, w)
        return Instance("cfg2_N32_chimera_pm1", 32, 100, J, np.zeros(32), True)
    if k == 3:
        J, h = complete_gaussian(36, seed, h_scale=0.5)
        return Instance("cfg3_N36_complete_gauss", 36, 100, J, h, False)
    if k == 4:
        rng = np.random.Generator(np.random.PCG64(seed))
        N = 40
        edges = lattice_edges(5, 8)
        assert len(edges) == 67
        have = set(edges)
        extra = []
        while len(extra) < 40:
            i, j = (int(x) for x in rng.integers(0, N, size=2))
            if i == j:
                continue
            e = (min(i, j), max(i, j))
            if e in have:
                continue
            have.add(e)
            extra.append(e)
        all_edges = edges + extra
        w = rng.choice(np.array([-3.0, -2.0, -1.0, 1.0, 2.0, 3.0]), size=len(all_edges))
        J = _sym_from_edges(N, all_edges, w)
        h = rng.integers(-1, 2, size=N).astype(np.float64)
        return Instance("cfg4_N40_lattice_plus40_int", N, 1000, J, h, True)
    if k == 5:
        J, h = complete_gaussian(48, seed)
        return Instance("cfg5_N48_complete_gauss", 48, 100, J, h, False)
    raise ValueError("BASELINE.json has configs 1..5")


# ---- constructed instances with closed-form spectra (used as pins and as full-size GPU checks) ----

def ferromagnet(N: int, coupling: float = 1.0):
    """Uniform ferromagnet on the complete graph, no field."""
    J = coupling * (np.ones((N, N)) - np.eye(N))
    return J, np.zeros(N)


def mattis(N: int, seed: int, field: float = 0.0):
    """Gauge-transformed ferromagnet J_ij = xi_i xi_j, h_i = field * xi_i, xi in {+-1}^N random."""
    rng = np.random.Generator(np.random.PCG64(seed))
    xi = 2.0 * rng.integers(0, 2, size=N) - 1.0
    J = np.outer(xi, xi)
    np.fill_diagonal(J, 0.0)
    return J, field * xi, xi


def fields_only(N: int, seed: int, integer: bool = False):
    rng = np.random.Generator(np.random.PCG64(seed))
    if integer:
        h = rng.integers(1, 50, size=N).astype(np.float64) * (2.0 * rng.integers(0, 2, size=N) - 1.0)
    else:
        h = rng.standard_normal(N)
    return np.zeros((N, N)), h


def open_chain(N: int, seed: int):
    """Open chain 0-1-2-...-(N-1) with Gaussian couplings, no field."""
    rng = np.random.Generator(np.random.PCG64(seed))
    w = rng.standard_normal(N - 1)
    J = _sym_from_edges(N, [(i, i + 1) for i in range(N - 1)], w)
    return J, np.zeros(N), w


def two_blocks(NA: int, NB: int, seed: int, h_scale: float = 1.0):
    """Block-diagonal J: spins 0..NA-1 and NA..NA+NB-1 are two decoupled complete Gaussian graphs."""
    JA, hA = complete_gaussian(NA, seed)
    JB, hB = complete_gaussian(NB, seed + 7919)
    N = NA + NB
    J = np.zeros((N, N))
    J[:NA, :NA] = JA
    J[NA:, NA:] = JB
    return J, np.concatenate([h_scale * hA, h_scale * hB])


def random_integer(N: int, seed: int, wmax: int = 3, density: float = 1.0):
    """Random integer couplings in [-wmax, wmax] on a random graph of the given edge density."""
    rng = np.random.Generator(np.random.PCG64(seed))
    U = rng.integers(-wmax, wmax + 1, size=(N, N)).astype(np.float64)
    M = rng.random((N, N)) < density
    T = np.triu(U * M, 1)
    J = T + T.T
    h = rng.integers(-wmax, wmax + 1, size=N).astype(np.float64)
    return J, h
