"""Thin ctypes binding over the C-ABI library (include/ising.h). Argument marshalling only: every step of the
path runs in the CUDA kernels of csrc/. PyTorch supplies device buffers and the current stream, nothing else.

The library is loaded on first use and the load fails loudly if it is missing or cannot run: there is no CPU
fallback and nothing here imports the oracle.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libising_b200.so")

OK = 0
ERR_NULL, ERR_BAD_N, ERR_BAD_S, ERR_NONFINITE, ERR_ASYMMETRIC, ERR_DIAGONAL = -1, -2, -3, -4, -5, -6
ERR_BAD_RANGE, ERR_CUDA, ERR_BAND, ERR_INTERNAL, ERR_RANGE_W = -7, -8, -9, -10, -11
N_MAX = 63
S_MAX = 65536

# every symbol include/ising.h declares (tests/test_abi.py checks the header against this list and the .so)
EXPORTS = ["ising_lowest", "ising_lowest_range", "ising_lowest_host", "ising_lowest_h0", "ising_lowest_alg1", "ising_dos", "ising_merge_lists", "ising_merge_lists_static", "qubo_lowest",
           "ising_energies", "ising_get_last_stats", "ising_strerror", "ising_last_error", "ising_version",
           "ising_fma_peak", "ising_addmin_peak", "ising_addmin16x2_peak", "ising_addmin_mix_peak",
           "ising_zscreen_selftest", "ising_release_workspace"]


class IsingError(RuntimeError):
    def __init__(self, status: int, what: str, detail: str):
        super().__init__(f"{what} failed with status {status}: {detail}")
        self.status = status


class _Stats(ctypes.Structure):
    _fields_ = [("configs", ctypes.c_uint64), ("candidates", ctypes.c_uint64),
                ("kernel_launches", ctypes.c_uint32), ("enum_launches", ctypes.c_uint32),
                ("passes", ctypes.c_uint32), ("split_retries", ctypes.c_uint32),
                ("grid_exponent", ctypes.c_int32), ("exact", ctypes.c_int32),
                ("epsilon", ctypes.c_double), ("enum_ms", ctypes.c_double), ("total_ms", ctypes.c_double),
                ("keep", ctypes.c_int32), ("inner_bits", ctypes.c_int32),
                ("kernel_variant", ctypes.c_int32), ("screen_shift", ctypes.c_int32),
                ("hit_blocks", ctypes.c_uint64), ("false_hit_blocks", ctypes.c_uint64),
                ("z_ms", ctypes.c_double), ("z_configs", ctypes.c_uint64), ("z_blocks", ctypes.c_uint64),
                ("z_flagged_blocks", ctypes.c_uint64), ("z_launches", ctypes.c_uint32), ("reserved0", ctypes.c_uint32)]


@dataclass
class Stats:
    configs: int
    candidates: int
    kernel_launches: int
    enum_launches: int
    passes: int
    split_retries: int
    grid_exponent: int
    exact: bool
    epsilon: float
    enum_ms: float
    total_ms: float
    keep: int
    inner_bits: int
    kernel_variant: int
    screen_shift: int
    hit_blocks: int = 0
    false_hit_blocks: int = 0
    z_ms: float = 0.0
    z_configs: int = 0
    z_blocks: int = 0
    z_flagged_blocks: int = 0
    z_launches: int = 0


_lib = None


def load():
    """Load libising_b200.so (once). Raises if it has not been built -- the product path never falls back."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_1904_03621_b200.build` "
                           "(there is no CPU fallback)")
    try:
        import torch  # noqa: F401  (loads the CUDA runtime the library links against)
    except Exception:  # pragma: no cover
        pass
    lib = ctypes.CDLL(LIB_PATH)
    dp, up, vp = ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p
    i32, i64, u64 = ctypes.c_int, ctypes.c_int64, ctypes.c_uint64
    lib.ising_lowest.argtypes = [dp, dp, i32, i32, up, dp, vp]
    lib.ising_lowest_range.argtypes = [dp, dp, i32, i32, u64, u64, up, dp, vp]
    lib.ising_lowest_host.argtypes = [dp, dp, i32, i32, u64, u64, up, dp, vp]
    lib.ising_merge_lists.argtypes = [up, dp, i64, i32, up, dp, vp]
    lib.ising_merge_lists_static.argtypes = [up, dp, i64, i32, up, dp, vp]
    lib.ising_merge_lists_static.restype = ctypes.c_int
    lib.ising_lowest_h0.argtypes = [dp, i32, i32, up, dp, vp]
    lib.ising_lowest_alg1.argtypes = [dp, dp, i32, i32, u64, u64, i32, up, dp, vp]
    lib.ising_lowest_alg1.restype = ctypes.c_int
    lib.ising_dos.argtypes = [dp, dp, i32, i32, up, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double), vp]
    lib.ising_dos.restype = ctypes.c_int
    lib.ising_lowest_h0.restype = ctypes.c_int
    lib.qubo_lowest.argtypes = [dp, dp, i32, i32, up, dp, vp]
    lib.ising_energies.argtypes = [dp, dp, i32, up, i64, dp, vp]
    lib.ising_get_last_stats.argtypes = [ctypes.POINTER(_Stats)]
    lib.ising_fma_peak.argtypes = [ctypes.c_double, ctypes.POINTER(ctypes.c_double), vp]
    lib.ising_addmin_peak.argtypes = [ctypes.c_double, ctypes.POINTER(ctypes.c_double), vp]
    lib.ising_addmin16x2_peak.argtypes = [ctypes.c_double, ctypes.POINTER(ctypes.c_double), vp]
    lib.ising_addmin_mix_peak.argtypes = [ctypes.c_double, ctypes.POINTER(ctypes.c_double), vp]
    lib.ising_addmin_mix_peak.restype = ctypes.c_int
    lib.ising_zscreen_selftest.argtypes = [ctypes.c_uint32, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double), vp]
    lib.ising_zscreen_selftest.restype = ctypes.c_int
    for name in ("ising_lowest", "ising_lowest_range", "ising_lowest_host", "ising_merge_lists", "qubo_lowest",
                 "ising_energies", "ising_get_last_stats", "ising_fma_peak", "ising_addmin_peak", "ising_addmin16x2_peak",
                 "ising_version"):
        getattr(lib, name).restype = ctypes.c_int
    lib.ising_strerror.argtypes = [ctypes.c_int]
    lib.ising_strerror.restype = ctypes.c_char_p
    lib.ising_last_error.argtypes = []
    lib.ising_last_error.restype = ctypes.c_char_p
    lib.ising_release_workspace.argtypes = []
    lib.ising_release_workspace.restype = None
    _lib = lib
    return lib


def _check(rc: int, what: str):
    if rc != OK:
        lib = load()
        detail = (lib.ising_last_error() or b"").decode() or (lib.ising_strerror(rc) or b"").decode()
        raise IsingError(rc, what, detail)


def _stream(stream) -> int:
    import torch
    if stream is None:
        return int(torch.cuda.current_stream().cuda_stream)
    return int(getattr(stream, "cuda_stream", stream))


def _dev_f64(x, shape):
    import torch
    t = torch.as_tensor(x, dtype=torch.float64)
    if not t.is_cuda:
        t = t.cuda()
    t = t.contiguous()
    assert tuple(t.shape) == tuple(shape), f"expected shape {shape}, got {tuple(t.shape)}"
    return t


def strerror(status: int) -> str:
    return load().ising_strerror(int(status)).decode()


def version() -> int:
    return int(load().ising_version())


def last_stats() -> Stats:
    s = _Stats()
    _check(load().ising_get_last_stats(ctypes.byref(s)), "ising_get_last_stats")
    return Stats(s.configs, s.candidates, s.kernel_launches, s.enum_launches, s.passes, s.split_retries,
                 s.grid_exponent, bool(s.exact), s.epsilon, s.enum_ms, s.total_ms, s.keep, s.inner_bits, s.kernel_variant, s.screen_shift,
                 s.hit_blocks, s.false_hit_blocks, s.z_ms, s.z_configs, s.z_blocks, s.z_flagged_blocks, s.z_launches)


def ising_lowest_range(J, h, S: int, q_begin: int, q_end: int, stream=None, out=None):
    """Device tensors in, device tensors out: (states int64-viewed-as-uint64 [S], energies float64 [S])."""
    import torch
    h = _dev_f64(h, (len(h),))
    N = h.shape[0]
    J = _dev_f64(J, (N, N))
    if out is None:
        states = torch.empty(S, dtype=torch.int64, device=J.device)   # bit pattern of uint64 q
        energies = torch.empty(S, dtype=torch.float64, device=J.device)
    else:
        states, energies = out
    with torch.cuda.device(J.device):
        rc = load().ising_lowest_range(J.data_ptr(), h.data_ptr(), N, int(S), int(q_begin), int(q_end),
                                       states.data_ptr(), energies.data_ptr(), _stream(stream))
    _check(rc, "ising_lowest_range")
    return states, energies


def ising_lowest(J, h, S: int, stream=None, out=None):
    import torch
    h = _dev_f64(h, (len(h),))
    N = h.shape[0]
    J = _dev_f64(J, (N, N))
    if out is None:
        states = torch.empty(S, dtype=torch.int64, device=J.device)
        energies = torch.empty(S, dtype=torch.float64, device=J.device)
    else:
        states, energies = out
    with torch.cuda.device(J.device):
        rc = load().ising_lowest(J.data_ptr(), h.data_ptr(), N, int(S), states.data_ptr(), energies.data_ptr(),
                                 _stream(stream))
    _check(rc, "ising_lowest")
    return states, energies


def ising_lowest_alg1(J, h, S: int, q_begin: int = 0, q_end: int | None = None, chunk_log2: int = 20, stream=None):
    """The paper's Algorithm 1 written plainly (include/ising.h): direct fp64 energies per chunk + full-sort selection."""
    import torch
    h = _dev_f64(h, (len(h),))
    N = h.shape[0]
    J = _dev_f64(J, (N, N))
    if q_end is None:
        q_end = 1 << N
    states = torch.empty(S, dtype=torch.int64, device=J.device)
    energies = torch.empty(S, dtype=torch.float64, device=J.device)
    with torch.cuda.device(J.device):
        rc = load().ising_lowest_alg1(J.data_ptr(), h.data_ptr(), N, int(S), int(q_begin), int(q_end), int(chunk_log2),
                                      states.data_ptr(), energies.data_ptr(), _stream(stream))
    _check(rc, "ising_lowest_alg1")
    return states, energies


def ising_dos(J, h, nbins: int = 1024, stream=None):
    """Density of states (include/ising.h): returns (hist int64 [nbins] device tensor, e_lo, bin_width)."""
    import torch
    h = _dev_f64(h, (len(h),))
    N = h.shape[0]
    J = _dev_f64(J, (N, N))
    hist = torch.empty(nbins, dtype=torch.int64, device=J.device)
    e_lo, width = ctypes.c_double(0.0), ctypes.c_double(0.0)
    with torch.cuda.device(J.device):
        rc = load().ising_dos(J.data_ptr(), h.data_ptr(), N, int(nbins), hist.data_ptr(), ctypes.byref(e_lo),
                              ctypes.byref(width), _stream(stream))
    _check(rc, "ising_dos")
    return hist, e_lo.value, width.value


def ising_lowest_h0(J, S: int, stream=None):
    """Zero-field instance: half-space enumeration + complements (include/ising.h)."""
    import torch
    N = len(J)
    J = _dev_f64(J, (N, N))
    states = torch.empty(S, dtype=torch.int64, device=J.device)
    energies = torch.empty(S, dtype=torch.float64, device=J.device)
    with torch.cuda.device(J.device):
        rc = load().ising_lowest_h0(J.data_ptr(), N, int(S), states.data_ptr(), energies.data_ptr(), _stream(stream))
    _check(rc, "ising_lowest_h0")
    return states, energies


def ising_lowest_host(J, h, S: int, q_begin: int = 0, q_end: int | None = None, stream=None, out=None):
    """HOST numpy arrays (or pinned CPU tensors) in and out; host<->device copies happen inside the call."""
    import numpy as np
    J = np.ascontiguousarray(J, dtype=np.float64)
    h = np.ascontiguousarray(h, dtype=np.float64)
    N = h.shape[0]
    assert J.shape == (N, N)
    if q_end is None:
        q_end = 1 << N
    if out is None:
        states = np.empty(S, dtype=np.uint64)
        energies = np.empty(S, dtype=np.float64)
    else:
        states, energies = out
    rc = load().ising_lowest_host(J.ctypes.data, h.ctypes.data, N, int(S), int(q_begin), int(q_end),
                                  states.ctypes.data, energies.ctypes.data, _stream(stream))
    _check(rc, "ising_lowest_host")
    return states, energies


def qubo_lowest(a, b, S: int, stream=None):
    import torch
    b = _dev_f64(b, (len(b),))
    N = b.shape[0]
    a = _dev_f64(a, (N, N))
    states = torch.empty(S, dtype=torch.int64, device=a.device)
    energies = torch.empty(S, dtype=torch.float64, device=a.device)
    with torch.cuda.device(a.device):
        rc = load().qubo_lowest(a.data_ptr(), b.data_ptr(), N, int(S), states.data_ptr(), energies.data_ptr(),
                                _stream(stream))
    _check(rc, "qubo_lowest")
    return states, energies


def ising_merge_lists(states_in, energies_in, S: int, stream=None):
    import torch
    assert states_in.is_cuda and energies_in.is_cuda and states_in.dtype == torch.int64
    states_in = states_in.contiguous()
    energies_in = energies_in.to(torch.float64).contiguous()
    n = states_in.numel()
    states = torch.empty(S, dtype=torch.int64, device=states_in.device)
    energies = torch.empty(S, dtype=torch.float64, device=states_in.device)
    with torch.cuda.device(states_in.device):
        rc = load().ising_merge_lists(states_in.data_ptr(), energies_in.data_ptr(), n, int(S),
                                      states.data_ptr(), energies.data_ptr(), _stream(stream))
    _check(rc, "ising_merge_lists")
    return states, energies


MERGE_STATIC_MAX = 131072


def ising_merge_lists_static(states_in, energies_in, S: int, stream=None, out=None):
    """`ising_merge_lists` without any device allocation inside the library (include/ising.h): for callers whose GPU
    memory is already owned by another pool, or who cannot afford cudaMalloc's device-wide synchronisation. At most
    MERGE_STATIC_MAX input pairs; the library's 2 MiB static scratch is shared, so do not overlap two calls on one
    device. Pass `out=(states, energies)` (int64 [S], float64 [S] device tensors) and this wrapper allocates nothing
    either; inputs must then already be contiguous int64 / float64."""
    import torch
    assert states_in.is_cuda and energies_in.is_cuda and states_in.dtype == torch.int64
    states_in = states_in.contiguous()
    energies_in = energies_in.to(torch.float64).contiguous()
    n = states_in.numel()
    if out is None:
        states = torch.empty(S, dtype=torch.int64, device=states_in.device)
        energies = torch.empty(S, dtype=torch.float64, device=states_in.device)
    else:
        states, energies = out
        assert states.dtype == torch.int64 and energies.dtype == torch.float64
        assert states.numel() >= S and energies.numel() >= S and states.is_contiguous() and energies.is_contiguous()
    with torch.cuda.device(states_in.device):
        rc = load().ising_merge_lists_static(states_in.data_ptr(), energies_in.data_ptr(), n, int(S),
                                             states.data_ptr(), energies.data_ptr(), _stream(stream))
    _check(rc, "ising_merge_lists_static")
    return states, energies


def ising_energies(J, h, states, stream=None):
    import torch
    h = _dev_f64(h, (len(h),))
    N = h.shape[0]
    J = _dev_f64(J, (N, N))
    states = states.contiguous()
    assert states.is_cuda and states.dtype == torch.int64
    out = torch.empty(states.numel(), dtype=torch.float64, device=J.device)
    with torch.cuda.device(J.device):
        rc = load().ising_energies(J.data_ptr(), h.data_ptr(), N, states.data_ptr(), states.numel(), out.data_ptr(),
                                   _stream(stream))
    _check(rc, "ising_energies")
    return out


@dataclass
class Solution:
    """What the paper's `search` returns (Listing 1): energies and states, lowest first."""
    energies: "object"      # numpy float64 [num_states]
    states: "object"        # numpy uint64 [num_states]; bit i-1 of a state <-> the paper's 1-based spin i


def search(graph: dict, num_states: int = 1, stream=None) -> Solution:
    """The paper's one-call interface (Listing 1): `graph` maps 1-based index pairs to weights,
    (i, j) with i != j is the coupling J_ij of eq. (1) and (i, i) is the field h_i. Marshalling only:
    the dict is laid out as dense (J, h) and handed to `ising_lowest`; (i, j) and (j, i) must not both be given."""
    import numpy as np
    if not graph:
        raise ValueError("empty graph")
    N = max(max(i, j) for i, j in graph)
    if min(min(i, j) for i, j in graph) < 1:
        raise ValueError("spin indices are 1-based (PAPER.md:137)")
    J = np.zeros((N, N), dtype=np.float64)
    h = np.zeros(N, dtype=np.float64)
    for (i, j), w in graph.items():
        if i == j:
            h[i - 1] = w
        else:
            if (j, i) in graph:
                raise ValueError(f"both ({i},{j}) and ({j},{i}) given")
            J[i - 1, j - 1] = J[j - 1, i - 1] = w
    q, e = ising_lowest(J, h, int(num_states), stream=stream)
    return Solution(energies=e.cpu().numpy(), states=states_to_numpy(q))


def fma_peak(ms_target: float = 50.0, stream=None) -> float:
    v = ctypes.c_double(0.0)
    _check(load().ising_fma_peak(float(ms_target), ctypes.byref(v), _stream(stream)), "ising_fma_peak")
    return v.value


def addmin_peak(ms_target: float = 50.0, stream=None) -> float:
    v = ctypes.c_double(0.0)
    _check(load().ising_addmin_peak(float(ms_target), ctypes.byref(v), _stream(stream)), "ising_addmin_peak")
    return v.value


def addmin16x2_peak(ms_target: float = 50.0, stream=None) -> float:
    """VIADDMNMX.U16x2 lane instructions per second (two 16-bit add-mins each)."""
    v = ctypes.c_double(0.0)
    _check(load().ising_addmin16x2_peak(float(ms_target), ctypes.byref(v), _stream(stream)), "ising_addmin16x2_peak")
    return v.value


def addmin_mix_peak(ms_target: float = 50.0, stream=None) -> float:
    """Lane add-mins per second of the fused + split instruction mix (include/ising.h)."""
    v = ctypes.c_double(0.0)
    _check(load().ising_addmin_mix_peak(float(ms_target), ctypes.byref(v), _stream(stream)), "ising_addmin_mix_peak")
    return v.value


def zscreen_selftest(seed: int = 1, stream=None):
    """(largest relative under-estimate, largest relative over-estimate) of a positive-term tcgen05 bf16 GEMM against
    fp64 (include/ising.h)."""
    u, o = ctypes.c_double(0.0), ctypes.c_double(0.0)
    _check(load().ising_zscreen_selftest(int(seed), ctypes.byref(u), ctypes.byref(o), _stream(stream)), "ising_zscreen_selftest")
    return u.value, o.value


def release_workspace() -> None:
    load().ising_release_workspace()


def states_to_numpy(states):
    """int64 device/CPU tensor holding uint64 bit patterns -> numpy uint64."""
    import numpy as np
    return states.detach().cpu().numpy().view(np.uint64)
