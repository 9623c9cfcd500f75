"""ctypes wrapper over oracle/oracle.c -- TEST INFRASTRUCTURE, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
import this. It imports nothing from paper_1904_03621_b200 (the CUDA path).
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile oracle.c with gcc (-O2 -fopenmp, no fp contraction)."""
    src = os.path.join(_HERE, "oracle.c")
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(src):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", "-o", _SO, src, "-lm"]
        )
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        dp = ctypes.POINTER(ctypes.c_double)
        up = ctypes.POINTER(ctypes.c_uint64)
        lib.oracle_energy.restype = ctypes.c_double
        lib.oracle_energy.argtypes = [dp, dp, ctypes.c_int, ctypes.c_uint64]
        lib.oracle_energies.restype = None
        lib.oracle_energies.argtypes = [dp, dp, ctypes.c_int, ctypes.c_uint64, ctypes.c_uint64, dp]
        lib.oracle_energies_of.restype = None
        lib.oracle_energies_of.argtypes = [dp, dp, ctypes.c_int, up, ctypes.c_uint64, dp]
        lib.oracle_lowest.restype = ctypes.c_int64
        lib.oracle_lowest.argtypes = [dp, dp, ctypes.c_int, ctypes.c_int64, ctypes.c_uint64,
                                      ctypes.c_uint64, up, dp, ctypes.c_int]
        lib.oracle_max_threads.restype = ctypes.c_int
        lib.oracle_dos.restype = ctypes.c_int64
        lib.oracle_dos.argtypes = [dp, dp, ctypes.c_int, ctypes.c_double, ctypes.c_double, ctypes.c_int, up]
        _lib = lib
    return _lib


def _prep(J, h):
    J = np.ascontiguousarray(J, dtype=np.float64)
    h = np.ascontiguousarray(h, dtype=np.float64)
    N = h.shape[0]
    assert J.shape == (N, N)
    dp = ctypes.POINTER(ctypes.c_double)
    return J, h, N, J.ctypes.data_as(dp), h.ctypes.data_as(dp)


def energy(J, h, q: int) -> float:
    """Eq. (1) energy of the single state q."""
    J, h, N, Jp, hp = _prep(J, h)
    return float(_load().oracle_energy(Jp, hp, N, int(q)))


def energies_range(J, h, q_begin: int, count: int) -> np.ndarray:
    J, h, N, Jp, hp = _prep(J, h)
    out = np.empty(count, dtype=np.float64)
    _load().oracle_energies(Jp, hp, N, int(q_begin), int(count),
                            out.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    return out


def energies_of(J, h, states) -> np.ndarray:
    J, h, N, Jp, hp = _prep(J, h)
    q = np.ascontiguousarray(states, dtype=np.uint64)
    out = np.empty(q.shape[0], dtype=np.float64)
    _load().oracle_energies_of(Jp, hp, N, q.ctypes.data_as(ctypes.POINTER(ctypes.c_uint64)),
                               q.shape[0], out.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
    return out


def lowest(J, h, S: int, q_begin: int = 0, q_end: int | None = None, threads: int = 0):
    """The S lowest (E, q) pairs of [q_begin, q_end), ascending under (E, q). Returns (states, energies)."""
    J, h, N, Jp, hp = _prep(J, h)
    if q_end is None:
        q_end = 1 << N
    states = np.empty(S, dtype=np.uint64)
    en = np.empty(S, dtype=np.float64)
    n = _load().oracle_lowest(Jp, hp, N, int(S), int(q_begin), int(q_end),
                              states.ctypes.data_as(ctypes.POINTER(ctypes.c_uint64)),
                              en.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), int(threads))
    if n < 0:
        raise ValueError("oracle_lowest: bad arguments")
    return states[:n].copy(), en[:n].copy()


def dos(J, h, e_lo: float, width: float, nbins: int):
    """Histogram of all 2^N energies of eq. (1): (hist uint64[nbins], number of states outside the bins)."""
    J, h, N, Jp, hp = _prep(J, h)
    hist = np.zeros(nbins, dtype=np.uint64)
    out = _load().oracle_dos(Jp, hp, N, float(e_lo), float(width), int(nbins),
                             hist.ctypes.data_as(ctypes.POINTER(ctypes.c_uint64)))
    if out < 0:
        raise ValueError("oracle_dos: bad arguments")
    return hist, int(out)


_SO_GRAY = os.path.join(_HERE, "liboracle_gray.so")
_lib_gray = None


def build_gray(force: bool = False) -> str:
    """Compile oracle_gray.c (tier-2 oracle for integer instances; see its header)."""
    src = os.path.join(_HERE, "oracle_gray.c")
    if force or not os.path.exists(_SO_GRAY) or os.path.getmtime(_SO_GRAY) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _SO_GRAY, src, "-lm"])
    return _SO_GRAY


def lowest_gray(J, h, S: int, q_begin: int = 0, q_end: int | None = None, slab_bits: int | None = None,
                threads: int = 0):
    """Tier-2 oracle (single-spin-flip recurrence in exact int64), INTEGER-weight instances only.
    Pinned to `lowest` by tests/test_oracle_pins.py; used to write tests/golden/cfg4.txt."""
    global _lib_gray
    if _lib_gray is None:
        build_gray()
        lib = ctypes.CDLL(_SO_GRAY)
        dp = ctypes.POINTER(ctypes.c_double)
        up = ctypes.POINTER(ctypes.c_uint64)
        lib.oracle_gray_lowest.restype = ctypes.c_int64
        lib.oracle_gray_lowest.argtypes = [dp, dp, ctypes.c_int, ctypes.c_int64, ctypes.c_uint64, ctypes.c_uint64,
                                           ctypes.c_int, up, dp, ctypes.c_int]
        _lib_gray = lib
    J, h, N, Jp, hp = _prep(J, h)
    if q_end is None:
        q_end = 1 << N
    if slab_bits is None:
        slab_bits = min(N, 22)
        while (q_begin | q_end) & ((1 << slab_bits) - 1):
            slab_bits -= 1
    states = np.empty(S, dtype=np.uint64)
    en = np.empty(S, dtype=np.float64)
    n = _lib_gray.oracle_gray_lowest(Jp, hp, N, int(S), int(q_begin), int(q_end), int(slab_bits),
                                     states.ctypes.data_as(ctypes.POINTER(ctypes.c_uint64)),
                                     en.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), int(threads))
    if n == -2:
        raise ValueError("oracle_gray_lowest: integer weights only")
    if n < 0:
        raise ValueError("oracle_gray_lowest: bad arguments")
    return states[:n].copy(), en[:n].copy()


_SO_BNB = os.path.join(_HERE, "liboracle_bnb.so")
_lib_bnb = None


def build_bnb(force: bool = False) -> str:
    """Compile oracle_bnb.c (tier-3 oracle: exact branch and bound; see its header)."""
    src = os.path.join(_HERE, "oracle_bnb.c")
    if force or not os.path.exists(_SO_BNB) or os.path.getmtime(_SO_BNB) < os.path.getmtime(src):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off", "-o", _SO_BNB, src, "-lm"])
    return _SO_BNB


def lowest_bnb(J, h, S: int, spare: int = 48, threads: int = 0):
    """Tier-3 oracle: the S + spare lowest (E, q) of the whole space by exact branch and bound (fp64).
    Pinned to `lowest` by tests/test_oracle_pins.py; used to write tests/golden/cfg5.txt.
    Returns (states, energies, nodes_visited); the first S entries are the answer, the rest are spare."""
    global _lib_bnb
    if _lib_bnb is None:
        build_bnb()
        lib = ctypes.CDLL(_SO_BNB)
        dp = ctypes.POINTER(ctypes.c_double)
        up = ctypes.POINTER(ctypes.c_uint64)
        lib.oracle_bnb_lowest.restype = ctypes.c_int64
        lib.oracle_bnb_lowest.argtypes = [dp, dp, ctypes.c_int, ctypes.c_int64, ctypes.c_int64, up, dp, ctypes.c_int, up]
        _lib_bnb = lib
    J, h, N, Jp, hp = _prep(J, h)
    K = S + spare
    states = np.empty(K, dtype=np.uint64)
    en = np.empty(K, dtype=np.float64)
    nodes = ctypes.c_uint64(0)
    n = _lib_bnb.oracle_bnb_lowest(Jp, hp, N, int(S), int(spare),
                                   states.ctypes.data_as(ctypes.POINTER(ctypes.c_uint64)),
                                   en.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), int(threads), ctypes.byref(nodes))
    if n < 0:
        raise ValueError("oracle_bnb_lowest: bad arguments")
    return states[:n].copy(), en[:n].copy(), int(nodes.value)


def max_threads() -> int:
    return int(_load().oracle_max_threads())
