"""Write the stored expected outputs under tests/golden/ by calling ONLY the CPU oracle.

Usage:  python tests/golden/make_goldens.py [config numbers ...]     (default: 1 2)

Each file cfg<k>.txt holds the oracle's S+16 lowest (q, E) pairs of BASELINE.json config k
(energy as a C99 hex float, so the file is bit-exact), plus the instance SHA-256. Config 1 takes
under a second, config 2 minutes, config 3 about two hours on 8 cores; configs 4 and 5 are out of
reach of the plain oracle.
Nothing here imports or runs the CUDA path.
"""
import os
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

from oracle import oracle  # noqa: E402
from paper_1904_03621_b200 import instances as I  # noqa: E402

EXTRA = 16  # spare entries past S so that boundary swaps can be adjudicated


def main(argv):
    ks = [int(a) for a in argv] or [1, 2]
    for k in ks:
        c = I.baseline_config(k)
        t0 = time.time()
        q, e = oracle.lowest(c.J, c.h, c.S + EXTRA)
        dt = time.time() - t0
        path = os.path.join(HERE, f"cfg{k}.txt")
        with open(path, "w") as f:
            f.write(f"# BASELINE.json config {k}: {c.name}, N={c.N}, S={c.S} (+{EXTRA} spare)\n")
            f.write(f"# written by tests/golden/make_goldens.py from oracle/oracle.c only; oracle wall time {dt:.1f} s, "
                    f"{oracle.max_threads()} threads\n")
            f.write(f"# instance sha256 {c.sha256()}\n")
            for qq, ee in zip(q, e):
                f.write(f"{int(qq)} {float(ee).hex()}\n")
        print(f"cfg{k}: {len(q)} pairs in {dt:.1f} s -> {path}", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:])
