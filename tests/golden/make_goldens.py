"""Write the stored expected outputs under tests/golden/ by calling ONLY the CPU oracle.

Usage:  python tests/golden/make_goldens.py [config numbers ...]     (default: 1 2)
        python tests/golden/make_goldens.py --chunks 64 3       (resumable: see below)

Each file cfg<k>.txt holds the oracle's S+16 lowest (q, E) pairs of BASELINE.json config k
(energy as a C99 hex float, so the file is bit-exact), plus the instance SHA-256. Config 1 takes
under a second, config 2 minutes, config 3 about 2.6 hours on 8 cores with the plain oracle (oracle.c).
Config 4 (2^40 states, integer weights) is out of reach of the plain oracle (about 40 hours) and is written
by the tier-2 oracle oracle_gray.c (exact int64 single-spin-flip recurrence, pinned to oracle.c by
tests/test_oracle_pins.py) in about an hour; its file says so. Config 5 (2^48 states, real weights) is out of
reach of both and is written by the tier-3 oracle oracle_bnb.c (exact branch and bound in fp64, pinned to oracle.c
by the same tests, including the stored lists of configs 1, 3 and 4) in seconds; its file says so.
With --chunks C the state space is cut into C equal ranges of q; the oracle's S+16 lowest of each range
(oracle_lowest on [q_begin, q_end)) are appended to tests/golden/.cfg<k>.partial as they finish, so an
interrupted run resumes where it stopped; the union of the per-range lists is then ordered by (E, q) and cut
at S+16 -- the lowest S+16 of the whole space are among the lowest S+16 of their own range.
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


def lowest_chunked(c, k, chunks):
    """oracle.lowest range by range, checkpointed to .cfg<k>.partial (lines: chunk q E.hex; 'done chunk seconds')."""
    part = os.path.join(HERE, f".cfg{k}.partial")
    done, pairs, spent = set(), [], 0.0
    if os.path.exists(part):
        rows = [l.split() for l in open(part) if l.strip()]
        if rows and rows[0] == ["sha", c.sha256(), str(chunks)]:
            done = {int(r[1]) for r in rows if r[0] == "done"}
            spent = sum(float(r[2]) for r in rows if r[0] == "done")
            pairs = [(float.fromhex(r[2]), int(r[1])) for r in rows if r[0] != "done" and r[0] != "sha" and int(r[0]) in done]
        else:
            os.remove(part)
    if not os.path.exists(part):
        with open(part, "w") as f:
            f.write(f"sha {c.sha256()} {chunks}\n")
    total = 1 << c.N
    assert total % chunks == 0
    step = total // chunks
    for i in range(chunks):
        if i in done:
            continue
        t0 = time.time()
        solve = oracle.lowest_gray if k == 4 else oracle.lowest
        q, e = solve(c.J, c.h, min(c.S + EXTRA, step), i * step, (i + 1) * step)
        dt = time.time() - t0
        with open(part, "a") as f:
            for qq, ee in zip(q, e):
                f.write(f"{i} {int(qq)} {float(ee).hex()}\n")
            f.write(f"done {i} {dt:.1f}\n")
        pairs += [(float(ee), int(qq)) for qq, ee in zip(q, e)]
        spent += dt
        print(f"cfg{k}: chunk {i + 1}/{chunks} in {dt:.1f} s", flush=True)
    pairs.sort()
    pairs = pairs[:c.S + EXTRA]
    return [p[1] for p in pairs], [p[0] for p in pairs], spent


def main(argv):
    chunks = 0
    if argv and argv[0] == "--chunks":
        chunks = int(argv[1]); argv = argv[2:]
    ks = [int(a) for a in argv] or [1, 2]
    for k in ks:
        c = I.baseline_config(k)
        t0 = time.time()
        if chunks:
            q, e, dt = lowest_chunked(c, k, chunks)
        else:
            if k == 5:
                q, e, _nodes = oracle.lowest_bnb(c.J, c.h, c.S, spare=EXTRA)
            else:
                q, e = (oracle.lowest_gray if k == 4 else oracle.lowest)(c.J, c.h, c.S + EXTRA)
            dt = time.time() - t0
        path = os.path.join(HERE, f"cfg{k}.txt")
        with open(path, "w") as f:
            f.write(f"# BASELINE.json config {k}: {c.name}, N={c.N}, S={c.S} (+{EXTRA} spare)\n")
            src = ("oracle/oracle_gray.c (tier-2 oracle, integer instances)" if k == 4 else
                   "oracle/oracle_bnb.c (tier-3 oracle, exact branch and bound)" if k == 5 else "oracle/oracle.c")
            f.write(f"# written by tests/golden/make_goldens.py from {src} only; oracle wall time {dt:.1f} s, "
                    f"{oracle.max_threads()} threads\n")
            f.write(f"# instance sha256 {c.sha256()}\n")
            for qq, ee in zip(q, e):
                f.write(f"{int(qq)} {float(ee).hex()}\n")
        print(f"cfg{k}: {len(q)} pairs in {dt:.1f} s -> {path}", flush=True)


if __name__ == "__main__":
    main(sys.argv[1:])
