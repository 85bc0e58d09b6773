"""One lattice sharded in t-slabs over R ranks (LGF_OPT_SHARD_WORLD, paper_1210_8018_b200/sharded.py) against
the oracle on ONE GPU: all R slabs live in this process, their kernel steps are launched one after another and the
exchanges between them are device copies (sharded.LocalComm), so nothing waits on a peer.  Same tolerances as the
unsharded path (BASELINE.json north_star)."""
import numpy as np
import pytest

import gen
import oracle
from test_golden import golden_path, read_golden

pytestmark = pytest.mark.gpu

ALPHA = 0.08


@pytest.fixture(scope="module")
def mods(cuda_device):
    from paper_1210_8018_b200 import lgf, sharded

    lgf.lib()
    return lgf, sharded


def _gather(parts):
    return np.concatenate(parts, axis=0)


CASES = [((8, 8, 8, 8), 1), ((8, 8, 8, 8), 2), ((8, 8, 8, 8), 4), ((16, 16, 8, 16), 2), ((12, 12, 12, 12), 3),
         ((8, 8, 32, 16), 4), ((16, 16, 16, 32), 8)]


@pytest.mark.parametrize("case", CASES, ids=lambda c: "x".join(map(str, c[0])) + f"-R{c[1]}")
@pytest.mark.parametrize("prec,recon", [("fp64", 18), ("fp64", 12), ("fp32", 18)])
def test_sharded_iterations_match_oracle(mods, case, prec, recon):
    lgf, sharded = mods
    N, R = case
    U = gen.gen_links(N, 0.5, 9000 + R)
    _, F0, th0 = oracle.measure(N, U, want_delta=False)
    Uo = U.copy()
    hist = oracle.iterate(N, Uo, ALPHA, 3)
    cdt = np.complex128 if prec == "fp64" else np.complex64
    tol_u, tol_s = (1e-12, 1e-10) if prec == "fp64" else (1e-5, 1e-4)
    sg = sharded.ShardedGaugeFixer(N, sharded.LocalComm(R), precision=prec, recon=recon)
    r0 = sg.load_links([np.ascontiguousarray(sharded.slab_of(U, N, R, r).astype(cdt)) for r in range(R)])
    assert abs(r0.F - F0) <= tol_s * max(abs(F0), 1e-3) and abs(r0.theta - th0) <= tol_s * th0 and r0.iterations == 0
    r = sg.iterate(ALPHA, 3)
    assert r.iterations == 3
    assert abs(r.F - hist[3, 0]) <= tol_s * abs(hist[3, 0]) and abs(r.theta - hist[3, 1]) <= 10 * tol_s * hist[3, 1]
    got = _gather(sg.get_links()).astype(np.complex128)
    assert got.shape == U.shape and np.abs(got - Uo).max() < 3 * tol_u
    sg.close()
    # the unsharded context on the same lattice: same links to rounding
    gf = lgf.GaugeFixer(N, precision=prec, recon=recon)
    gf.load_links(U.astype(cdt))
    gf.iterate(ALPHA, 3)
    assert np.abs(gf.get_links().astype(np.complex128) - got).max() < (1e-13 if prec == "fp64" else 1e-5)
    gf.close()


@pytest.mark.parametrize("R", [2, 4])
def test_sharded_fix_matches_golden(mods, R):
    lgf, sharded = mods
    n, seed = 8, gen.BASE_SEED + 8
    it, F, th, hist = read_golden(golden_path(n, seed))
    N = (n,) * 4
    U = gen.gen_links(n, 0.3, seed)
    sg = sharded.ShardedGaugeFixer(N, sharded.LocalComm(R), recon=12)
    sg.load_links([np.ascontiguousarray(sharded.slab_of(U, N, R, r)) for r in range(R)])
    r = sg.fix(ALPHA, 1e-15)
    assert r.converged == 1 and r.theta <= 1e-15 and r.iterations == it and abs(r.F - F) <= 1e-10
    Ufix = _gather(sg.get_links())
    assert abs(oracle.plaquette(n, Ufix) - oracle.plaquette(n, U)) < 1e-12      # a gauge transformation (pin P11)
    r2 = sg.fix(ALPHA, 1e-15)
    assert r2.iterations == 0 and r2.converged == 1 and r2.F == r.F               # already converged: no further step
    sg.close()


def test_sharded_option_validation(mods):
    lgf, sharded = mods
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer((8, 8, 8, 12), shard=(8, 0))           # 8 does not divide Nt = 12
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer((8, 8, 8, 8), shard=(2, 2))            # rank out of range
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer((8, 8, 8, 8), shard=(2, 0), accum_g=1) # default path only
    gf = lgf.GaugeFixer((8, 8, 8, 8), shard=(2, 1))
    i = gf.shard_info()
    assert i["world"] == 2 and i["rank"] == 1 and i["own_slices"] == 4 and i["sites"] == 8 * 8 * 8 * 4
    assert i["stored_sites"] == 8 * 8 * 8 * 6 and i["slice_sites"] == 512
    U = gen.gen_links((8, 8, 8, 8), 0.3, 5)
    gf.load_links(np.ascontiguousarray(U[2048:]))
    with pytest.raises(lgf.LgfError):
        gf.iterate(ALPHA, 1)                                   # the single-GPU drivers refuse a sharded context
    assert np.array_equal(gf.get_links(), U[2048:])           # round trip of the rank's own slices
    gf.close()
