"""Writes the stored expected values under tests/golden/ by calling ONLY gen/ and oracle/.

    python tests/golden/make_golden.py [8 16 32 48 64]

For each listed N^4 BASELINE.json config (and the two extra seeds +1000, +2000 at 8^4 and
16^4) it runs the oracle's Algorithm 1 (orc_fix, alpha = 0.08, eps = 1e-15) and writes
fix_<N>_<seed>.txt: iteration count, final F and theta, and the (F, theta) history.
48^4 (about 15 s per oracle iteration) and 64^4 (about 50 s per iteration, 25 GB) are run on request only;
the FP32 configuration (BASELINE config 4, eps = 1e-12) reads its iteration count off the same FP64
trajectory: the first row with theta <= 1e-12.
These are ORACLE values (the paper prints none): "parity unpinned" as values,
pinned through tests/test_oracle_pins.py.  The CUDA path is never called here.
"""
import os
import sys
import time

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))

import gen  # noqa: E402
import oracle  # noqa: E402

HERE = os.path.dirname(os.path.abspath(__file__))
SIGMA = {8: 0.3, 16: 0.5, 32: 0.5, 48: 0.5, 64: 0.6}


def run(n, seed):
    U = gen.gen_links(n, SIGMA[n], seed)
    t = time.time()
    it, F, th, hist = oracle.fix(n, U, 0.08, 1e-15)
    path = os.path.join(HERE, f"fix_{n}_{seed}.txt")
    with open(path, "w") as f:
        f.write(f"# oracle.fix on gen.gen_links({n}, {SIGMA[n]}, {seed}), alpha=0.08, eps=1e-15\n")
        f.write("# written by tests/golden/make_golden.py (oracle only); Algorithm 1, PAPER.md:75-111\n")
        f.write(f"iterations {it}\nF {F!r}\ntheta {th!r}\n# history: iteration F theta\n")
        for i, (a, b) in enumerate(hist):
            f.write(f"{i} {float(a)!r} {float(b)!r}\n")
    print(f"{n}^4 seed {seed}: {it} iterations, F = {F!r}, theta = {th:.3e}, {time.time() - t:.1f} s", flush=True)


if __name__ == "__main__":
    sizes = [int(a) for a in sys.argv[1:]] or [8, 16, 32]
    for n in sizes:
        seeds = [gen.BASE_SEED + n] + ([gen.BASE_SEED + n + 1000, gen.BASE_SEED + n + 2000] if n <= 16 else [])
        for s in seeds:
            run(n, s)
