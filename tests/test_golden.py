"""tests/golden/fix_*.txt are what the oracle gives today (they are oracle values, written by
tests/golden/make_golden.py; the paper prints none).  CPU only; re-runs the 8^4 cases and a
prefix of one 16^4 trajectory, and checks every stored trajectory for the invariants."""
import glob
import os

import numpy as np
import pytest

import gen
import oracle

HERE = os.path.dirname(os.path.abspath(__file__))


def read_golden(path):
    it = F = th = None
    hist = []
    for line in open(path):
        if line.startswith("#"):
            continue
        p = line.split()
        if p[0] == "iterations":
            it = int(p[1])
        elif p[0] == "F":
            F = float(p[1])
        elif p[0] == "theta":
            th = float(p[1])
        else:
            hist.append((float(p[1]), float(p[2])))
    return it, F, th, np.array(hist)


def golden_path(n, seed):
    return os.path.join(HERE, "golden", f"fix_{n}_{seed}.txt")


@pytest.mark.parametrize("seed", [gen.BASE_SEED + 8, gen.BASE_SEED + 1008, gen.BASE_SEED + 2008])
def test_golden_8(seed):
    it, F, th, hist = read_golden(golden_path(8, seed))
    U = gen.gen_links(8, 0.3, seed)
    it2, F2, th2, hist2 = oracle.fix(8, U, 0.08, 1e-15)
    assert it2 == it and F2 == F and th2 == th
    assert np.array_equal(hist, hist2)


def test_golden_16_prefix():
    seed = gen.BASE_SEED + 16
    it, F, th, hist = read_golden(golden_path(16, seed))
    U = gen.gen_links(16, 0.5, seed)
    h = oracle.iterate(16, U, 0.08, 3)
    assert np.array_equal(h, hist[:4])


def test_all_golden_trajectories_satisfy_the_invariants():
    files = sorted(glob.glob(os.path.join(HERE, "golden", "fix_*.txt")))
    assert len(files) >= 6
    for f in files:
        it, F, th, hist = read_golden(f)
        assert hist.shape[0] == it + 1
        assert th <= 1e-15 < hist[-2, 1]                       # stopped at the first theta <= eps
        # F never decreases (P12), up to the rounding of the stored double once the increments fall below one
        # unit in the last place at convergence (1.1e-16 for F in [0.5, 1): the 48^4 trajectory ends ...703, ...702)
        assert np.all(np.diff(hist[:, 0]) >= -2.3e-16)
        assert np.all(np.diff(hist[: it - 5, 0]) > 0)
        assert hist[-1, 0] == F and hist[-1, 1] == th
        tail = hist[-1, 1] / hist[-2, 1]
        assert 0.1 < tail < 0.5                                # tail ratio ~0.26
