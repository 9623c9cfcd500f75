"""How "identical to the oracle" is decided (BASELINE.json north_star; SURVEY.md section 8(c) "Checker")."""
import numpy as np


def assert_exact(q_gpu, e_gpu, q_orc, e_orc):
    """Integer-weight instances (and any case where both sides sum in the same fp64 order): element for element."""
    assert np.asarray(q_gpu, dtype=np.uint64).tolist() == np.asarray(q_orc, dtype=np.uint64).tolist()
    assert np.asarray(e_gpu, dtype=np.float64).tolist() == np.asarray(e_orc, dtype=np.float64).tolist()


def assert_real(q_gpu, e_gpu, q_orc, e_orc, W, S, rel=1e-12):
    """Real-weight instances. q_orc/e_orc hold the oracle's S (+ spare) lowest pairs.
    (i) energies agree rank by rank within rel; (ii) state lists identical except for swaps between states whose
    oracle energies differ by less than rel*W (also across the S / S+1 boundary)."""
    q_gpu = np.asarray(q_gpu, dtype=np.uint64); e_gpu = np.asarray(e_gpu, dtype=np.float64)
    q_orc = np.asarray(q_orc, dtype=np.uint64); e_orc = np.asarray(e_orc, dtype=np.float64)
    assert len(q_gpu) == S and len(q_orc) >= S
    tol = rel * W
    assert np.all(np.abs(e_gpu - e_orc[:S]) <= rel * np.abs(e_orc[:S]) + 1e-300)
    assert np.all(np.diff(e_gpu) >= 0)
    assert len(set(q_gpu.tolist())) == S
    orc_e = {int(q): float(e) for q, e in zip(q_orc, e_orc)}
    for r in range(S):
        if q_gpu[r] == q_orc[r]:
            continue
        # a swap: the GPU's state must be an oracle state of (nearly) the same energy
        assert int(q_gpu[r]) in orc_e, f"rank {r}: state {int(q_gpu[r])} not among the oracle's lowest"
        assert abs(orc_e[int(q_gpu[r])] - e_orc[r]) < tol, f"rank {r}: swap across a gap larger than {tol}"


def load_golden(path):
    q, e = [], []
    for line in open(path):
        if not line.strip() or line[0] == "#":
            continue
        a, b = line.split()
        q.append(int(a)); e.append(float.fromhex(b))
    return np.array(q, dtype=np.uint64), np.array(e, dtype=np.float64)
