"""GPU parity of the two SURVEY 8(f) variants of the hot path, through the C ABI, against the oracle:

  LGF_OPT_ACCUM_G (f1): the loaded links stay fixed and the accumulated transformation G(x) is
      carried instead; the same iteration as Alg. 1 lines 12-16 up to rounding, so
      the tolerances are those of the default path (BASELINE.json north_star).
  LGF_OPT_GMAP = 1 (f4): g = exp((alpha/2) w), eq. 1.2 as written; the oracle side is
      oracle.build_g_exp / oracle.set_exponential, pinned in tests/test_oracle_pins.py.
"""
import numpy as np
import pytest

import gen
import oracle
from test_golden import golden_path, read_golden

pytestmark = pytest.mark.gpu

ALPHA = 0.08


@pytest.fixture(scope="module")
def lgf(cuda_device):
    from paper_1210_8018_b200 import lgf as m

    m.lib()
    return m


@pytest.fixture
def exp_oracle():
    oracle.set_exponential(True)
    yield
    oracle.set_exponential(False)


ACC_LATTICES = [
    ((8, 8, 8, 8), 0.3, gen.BASE_SEED + 8),
    ((12, 12, 12, 12), 0.5, 79),
    ((16, 16, 16, 16), 0.5, gen.BASE_SEED + 16),
    ((32, 32, 32, 8), 0.5, 81),           # one of the paper's 32^3 x n lattices
    ((64, 64, 8, 8), 0.5, 1234),          # 64^2 FP64 planes: the 2-CTA cluster version of the last pass
]


def lid(v):
    return "x".join(map(str, v[0]))


# ------------------------------------------------------------------ ACCUM_G
@pytest.mark.parametrize("lat", ACC_LATTICES, ids=lid)
@pytest.mark.parametrize("recon", [18, 12])
def test_accum_g_iterations_match_oracle(lgf, lat, recon):
    """1 and then 3 more iterations: links (rewritten on demand), F, theta and the history."""
    N, sigma, seed = lat
    U = gen.gen_links(N, sigma, seed)
    Uo = U.copy()
    hist = oracle.iterate(N, Uo, ALPHA, 1)
    gf = lgf.GaugeFixer(N, recon=recon, accum_g=1)
    gf.load_links(U)
    r = gf.iterate(ALPHA, 1)
    assert r.iterations == 1
    assert abs(r.F - hist[1, 0]) <= 1e-10 * abs(hist[1, 0])
    assert abs(r.theta - hist[1, 1]) <= 1e-10 * hist[1, 1]
    assert np.abs(gf.get_links() - Uo).max() < 1e-12
    # carry on from the rewritten links (G was reset to 1), three iterations with G accumulating
    hist3 = oracle.iterate(N, Uo, ALPHA, 3)
    r = gf.iterate(ALPHA, 3)
    assert r.iterations == 3
    assert np.allclose(gf.history(), hist3, rtol=1e-9, atol=0)
    assert np.abs(gf.get_links() - Uo).max() < 1e-11
    # a plain measure of the rewritten links agrees with what the accumulated path reported
    F, th = gf.measure()
    assert abs(F - r.F) <= 1e-12 and abs(th - r.theta) <= 1e-10 * r.theta
    gf.close()


@pytest.mark.parametrize("n,sigma,seed", [(8, 0.3, gen.BASE_SEED + 8), (8, 0.3, gen.BASE_SEED + 1008),
                                          (16, 0.5, gen.BASE_SEED + 16)])
@pytest.mark.parametrize("recon", [18, 12])
def test_accum_g_convergence_matches_golden(lgf, n, sigma, seed, recon):
    it, F, th, hist = read_golden(golden_path(n, seed))
    U = gen.gen_links(n, sigma, seed)
    gf = lgf.GaugeFixer(n, recon=recon, accum_g=1)
    gf.load_links(U)
    r = gf.fix(ALPHA, 1e-15)
    assert r.converged == 1 and r.theta <= 1e-15
    assert abs(r.iterations - it) <= 0.02 * it
    assert abs(r.F - F) <= 1e-10
    h = gf.history()
    assert h.shape[0] == r.iterations + 1
    k = min(h.shape[0], hist.shape[0]) - 3
    assert np.allclose(h[:k, 0], hist[:k, 0], rtol=0, atol=1e-10)
    assert np.allclose(h[:k, 1], hist[:k, 1], rtol=1e-6, atol=1e-25)
    assert np.all(np.diff(h[:, 0]) >= -1e-15)
    Ufix = gf.get_links()
    I = np.eye(3)
    assert np.abs(Ufix @ np.conj(np.swapaxes(Ufix, -1, -2)) - I).max() < 1e-12
    assert np.abs(np.linalg.det(Ufix) - 1).max() < 1e-12
    if n == 8:
        assert abs(oracle.plaquette(n, Ufix) - oracle.plaquette(n, U)) < 1e-12
        # the fixed links agree with the oracle's fixed links (same gauge orbit, same minimum)
        Uo = U.copy()
        oracle.fix(n, Uo, ALPHA, 1e-15)
        assert np.abs(Ufix - Uo).max() < 1e-9
    r2 = gf.fix(ALPHA, 1e-15)
    assert r2.iterations == 0 and r2.converged == 1
    gf.close()


def test_accum_g_equals_default_path_and_stops_cleanly(lgf):
    """Same trajectory as the default path; kernels launched after convergence leave G alone."""
    n, seed = 8, gen.BASE_SEED + 2008
    U = gen.gen_links(n, 0.3, seed)
    a = lgf.GaugeFixer(n, recon=12)
    b = lgf.GaugeFixer(n, recon=12, accum_g=1, check_interval=64)   # many launches after `done`
    a.load_links(U)
    b.load_links(U)
    ra, rb = a.fix(ALPHA, 1e-15), b.fix(ALPHA, 1e-15)
    assert ra.iterations == rb.iterations
    assert abs(ra.F - rb.F) < 1e-13
    assert np.abs(a.get_links() - b.get_links()).max() < 1e-11
    Fb, thb = b.measure()
    assert abs(Fb - rb.F) < 1e-13 and thb <= 2e-15
    a.close()
    b.close()


def test_accum_g_fp32(lgf):
    N, sigma, seed = (16, 16, 16, 16), 0.5, gen.BASE_SEED + 16
    U = gen.gen_links(N, sigma, seed)
    U32 = U.astype(np.complex64)
    Uo = U32.astype(np.complex128)
    hist = oracle.iterate(N, Uo, ALPHA, 1)
    gf = lgf.GaugeFixer(N, precision="fp32", recon=12, accum_g=1)
    gf.load_links(U32)
    r = gf.iterate(ALPHA, 1)
    assert np.abs(gf.get_links().astype(np.complex128) - Uo).max() < 1e-5
    assert abs(r.theta - hist[1, 1]) <= 1e-4 * hist[1, 1]
    gf.load_links(U32)
    r = gf.fix(ALPHA, 1e-12)
    assert r.converged == 1 and r.theta <= 1e-12
    gf.close()


def test_accum_g_needs_the_tiled_packed_path(lgf):
    for kw in (dict(fft_batch=9), dict(fft_path=1), dict(fusion=0)):
        with pytest.raises(lgf.LgfError) as e:
            lgf.GaugeFixer(8, accum_g=1, **kw)
        assert e.value.code == lgf.ERR_INVALID_ARG
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer((4, 6, 8, 12), accum_g=1)           # generic FFT lattice


def test_accum_g_headline_32_12real(lgf):
    """BASELINE config 3 in the ACCUM_G launch configuration bench.py times."""
    n, seed = 32, gen.BASE_SEED + 32
    U = gen.gen_links(n, 0.5, seed)
    gf = lgf.GaugeFixer(n, recon=12, accum_g=1)
    gf.load_links(U)
    r1 = gf.iterate(ALPHA, 1)
    Uo = U.copy()
    hist = oracle.iterate(n, Uo, ALPHA, 1)
    assert np.abs(gf.get_links() - Uo).max() < 1e-12
    assert abs(r1.F - hist[1, 0]) <= 1e-10 * abs(hist[1, 0])
    assert abs(r1.theta - hist[1, 1]) <= 1e-10 * hist[1, 1]
    it, F, th, ghist = read_golden(golden_path(n, seed))
    gf.load_links(U)
    r = gf.fix(ALPHA, 1e-15)
    assert r.converged == 1 and abs(r.iterations - it) <= 0.02 * it and abs(r.F - F) <= 1e-10
    Ufix = gf.get_links()
    d = Ufix @ np.conj(np.swapaxes(Ufix, -1, -2)) - np.eye(3)
    assert np.abs(d).max() < 1e-12
    gf.close()


# ------------------------------------------------------------------ GMAP = exact exponential
EXP_VARIANTS = [dict(recon=18, fft_batch=4), dict(recon=12, fft_batch=4), dict(recon=18, fft_batch=9),
                dict(recon=12, fft_batch=4, fusion=0), dict(recon=18, fft_batch=4, fft_path=1),
                dict(recon=12, fft_batch=4, accum_g=1)]


def vid(v):
    return "-".join(f"{k}{x}" for k, x in v.items())


@pytest.mark.parametrize("var", EXP_VARIANTS[:4], ids=vid)
@pytest.mark.parametrize("scale", [1.0, 40.0])
def test_exp_g_tap_matches_oracle(lgf, var, scale):
    """g = exp((alpha/2) w) from an oracle w; scale = 40 makes |A| ~ 10 so that the halving and
    squaring steps run (alpha/2 * 40 = 1.6 times the natural size)."""
    N, sigma, seed = (8, 8, 8, 8), 0.5, 91
    U = gen.gen_links(N, sigma, seed)
    D, _, _ = oracle.measure(N, U)
    w = oracle.fourier_accelerate(N, D) * scale
    g = oracle.build_g_exp(w, ALPHA)
    gf = lgf.GaugeFixer(N, gmap=lgf.GMAP_EXP, **var)
    gf.load_links(U)
    gf.set_field(lgf.FIELD_W, w)
    g2 = gf.get_field(lgf.FIELD_G, alpha=ALPHA)
    # every squaring doubles the rounding error of the series: 4 (here) to 6 (oracle) squarings at scale 40
    tol = 5e-14 if scale == 1.0 else 5e-13
    assert np.abs(g2 - g).max() < tol
    assert np.abs(g2 @ np.conj(np.swapaxes(g2, -1, -2)) - np.eye(3)).max() < tol
    gf.stage(lgf.STAGE_UPDATE, alpha=ALPHA)
    U1 = oracle.update_links(N, U.copy(), g)
    assert np.abs(gf.get_links() - U1).max() < 4 * tol
    gf.close()


@pytest.mark.parametrize("var", EXP_VARIANTS, ids=vid)
@pytest.mark.parametrize("lat", [((8, 8, 8, 8), 0.3, gen.BASE_SEED + 8), ((16, 16, 16, 16), 0.5, gen.BASE_SEED + 16)], ids=lid)
def test_exp_one_iteration_matches_oracle(lgf, exp_oracle, var, lat):
    N, sigma, seed = lat
    U = gen.gen_links(N, sigma, seed)
    Uo = U.copy()
    hist = oracle.iterate(N, Uo, ALPHA, 1)
    gf = lgf.GaugeFixer(N, gmap=lgf.GMAP_EXP, **var)
    gf.load_links(U)
    r = gf.iterate(ALPHA, 1)
    assert np.abs(gf.get_links() - Uo).max() < 1e-12
    assert abs(r.F - hist[1, 0]) <= 1e-10 * abs(hist[1, 0])
    assert abs(r.theta - hist[1, 1]) <= 1e-10 * hist[1, 1]
    gf.close()


@pytest.mark.parametrize("var", [EXP_VARIANTS[1], EXP_VARIANTS[5]], ids=vid)
def test_exp_convergence_matches_oracle(lgf, exp_oracle, var):
    n, seed = 8, gen.BASE_SEED + 8
    U = gen.gen_links(n, 0.3, seed)
    Uo = U.copy()
    it, F, th, hist = oracle.fix(n, Uo, ALPHA, 1e-15)
    gf = lgf.GaugeFixer(n, gmap=lgf.GMAP_EXP, **var)
    gf.load_links(U)
    r = gf.fix(ALPHA, 1e-15)
    assert r.converged == 1 and abs(r.iterations - it) <= max(1, 0.02 * it)
    assert abs(r.F - F) <= 1e-10
    h = gf.history()
    k = min(h.shape[0], hist.shape[0]) - 3
    assert np.allclose(h[:k, 0], hist[:k, 0], rtol=0, atol=1e-10)
    # and the exponential map is not the first-order map: the trajectories differ at O(alpha^2 w^2)
    gf.set_option(lgf.OPT_GMAP, lgf.GMAP_FIRST_ORDER)
    gf.load_links(U)
    r0 = gf.iterate(ALPHA, 1)
    assert abs(r0.F - hist[1, 0]) > 1e-7
    gf.close()


# ------------------------------------------------------------------ LGF_LAYOUT_AOS12 interchange layout
@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_aos12_interchange_layout(lgf, recon, prec):
    """Rows 0, 1 as the exchange format: exact round trip of what was sent, row 2 is
    conj(row0 x row1), and an iteration from it matches the oracle run on the full links."""
    import torch

    N, sigma, seed = (8, 8, 8, 8), 0.3, gen.BASE_SEED + 8
    U = gen.gen_links(N, sigma, seed)
    cdt = np.complex128 if prec == "fp64" else np.complex64
    Uc = U.astype(cdt)
    U12 = np.ascontiguousarray(Uc[:, :, :2, :])
    gf = lgf.GaugeFixer(N, precision=prec, recon=recon)
    for src in (U12, torch.from_numpy(U12).cuda()):
        gf.load_links(src)
        two = gf.get_links(rows=2)
        assert two.shape == (8 ** 4, 4, 2, 3) and np.array_equal(two, U12)
        full = gf.get_links()
        assert np.array_equal(full[:, :, :2, :], U12)
        assert np.abs(full[:, :, 2, :] - Uc[:, :, 2, :]).max() < (5e-15 if prec == "fp64" else 1e-6)
        dev = gf.get_links(device=True, rows=2)
        assert np.array_equal(dev.cpu().numpy(), U12)
    r = gf.iterate(ALPHA, 1)
    Uo = Uc.astype(np.complex128)
    hist = oracle.iterate(N, Uo, ALPHA, 1)
    assert np.abs(gf.get_links().astype(np.complex128) - Uo).max() < (1e-12 if prec == "fp64" else 1e-5)
    assert abs(r.theta - hist[1, 1]) <= (1e-10 if prec == "fp64" else 1e-4) * hist[1, 1]
    gf.close()


# ------------------------------------------------------------------ LGF_OPT_GRAPH: graph replay == direct launches
@pytest.mark.parametrize("var", [dict(recon=12), dict(recon=18, fft_batch=9), dict(recon=12, fusion=0),
                                 dict(recon=18, fft_path=1), dict(recon=12, accum_g=1)], ids=vid)
def test_graph_replay_is_bitwise_the_direct_path(lgf, var):
    """The captured graph holds the same kernels with the same arguments: histories, links and launch
    counts are identical, for odd and even iteration counts and across fix / iterate / reload."""
    n, seed = 8, gen.BASE_SEED + 1008
    U = gen.gen_links(n, 0.3, seed)
    a = lgf.GaugeFixer(n, graph=1, **var)
    b = lgf.GaugeFixer(n, graph=0, **var)
    for gf in (a, b):
        gf.load_links(U)
    for steps in (19, 8, 1):
        ra, rb = a.iterate(ALPHA, steps), b.iterate(ALPHA, steps)
        assert ra.iterations == rb.iterations == steps
        assert ra.F == rb.F and ra.theta == rb.theta
        assert np.array_equal(a.history(), b.history())
    assert np.array_equal(a.get_links(), b.get_links())
    assert a.launch_count() == b.launch_count()
    ka, kb = a.kernel_times(), b.kernel_times()
    assert {k: v[1] for k, v in ka.items()} == {k: v[1] for k, v in kb.items()}
    for gf in (a, b):
        gf.load_links(U)
    ra, rb = a.fix(ALPHA, 1e-15), b.fix(ALPHA, 1e-15)
    assert ra.iterations == rb.iterations and ra.F == rb.F and ra.theta == rb.theta and ra.converged == 1
    assert np.array_equal(a.history(), b.history())
    assert np.array_equal(a.get_links(), b.get_links())
    # a different alpha re-captures; results still those of the direct path
    for gf in (a, b):
        gf.load_links(U)
    ra, rb = a.iterate(0.06, 10), b.iterate(0.06, 10)
    assert ra.F == rb.F and ra.theta == rb.theta
    a.close()
    b.close()


def test_graph_falls_back_on_the_legacy_default_stream(lgf):
    """The legacy default stream cannot be captured: the library must fall back to direct launches by
    itself and give the same results as on a capturable stream."""
    import torch

    n, seed = 8, gen.BASE_SEED + 8
    U = gen.gen_links(n, 0.3, seed)
    a = lgf.GaugeFixer(n, recon=12, stream=torch.cuda.default_stream())
    b = lgf.GaugeFixer(n, recon=12)
    for gf in (a, b):
        gf.load_links(U)
    ra, rb = a.iterate(ALPHA, 16), b.iterate(ALPHA, 16)
    assert ra.iterations == rb.iterations == 16 and ra.F == rb.F and ra.theta == rb.theta
    ra, rb = a.fix(ALPHA, 1e-15), b.fix(ALPHA, 1e-15)
    assert ra.iterations == rb.iterations and ra.F == rb.F and ra.converged == 1
    assert np.array_equal(a.get_links(), b.get_links())
    a.close()
    b.close()


# ------------------------------------------------------------------ LGF_OPT_ZBLOCK: (z,t)-blocked site walk
@pytest.mark.parametrize("var", [dict(recon=12), dict(recon=18, fusion=0), dict(recon=18, fft_batch=9, fft_path=1),
                                 dict(recon=12, accum_g=1)], ids=vid)
@pytest.mark.parametrize("N", [(8, 8, 8, 8), (12, 12, 12, 6), (4, 6, 8, 12)], ids=lambda n: "x".join(map(str, n)))
def test_site_walk_order_changes_nothing_but_the_sum_order(lgf, var, N):
    """Every z-block that divides Nz visits every site exactly once: the links after 3 iterations are
    bitwise those of the storage-order walk (same arithmetic per site), F and theta agree to rounding
    of the FP64 partial sums, and the first iteration matches the oracle."""
    if var.get("accum_g") and N != (8, 8, 8, 8):
        pytest.skip("ACCUM_G needs a lattice the tiled FFT covers")
    U = gen.gen_links(N, 0.5, 4242)
    Uo = U.copy()
    hist = oracle.iterate(N, Uo, ALPHA, 1)
    ref = None
    for zb in [N[2]] + [d for d in (1, 2, 3, 4, 6) if N[2] % d == 0 and d < N[2]]:
        gf = lgf.GaugeFixer(N, zblock=zb, **var)
        assert gf.zblock() == zb
        gf.load_links(U)
        r1 = gf.iterate(ALPHA, 1)
        assert np.abs(gf.get_links() - Uo).max() < 1e-12
        assert abs(r1.F - hist[1, 0]) <= 1e-10 * abs(hist[1, 0]) and abs(r1.theta - hist[1, 1]) <= 1e-10 * hist[1, 1]
        r3 = gf.iterate(ALPHA, 2)
        U3 = gf.get_links()
        if ref is None:
            ref = (U3, r3)
        else:
            assert np.array_equal(U3, ref[0]), zb
            assert abs(r3.F - ref[1].F) <= 1e-14 and abs(r3.theta - ref[1].theta) <= 1e-13 * ref[1].theta
        gf.close()


def test_zblock_option_validation_and_auto(lgf):
    gf = lgf.GaugeFixer((8, 8, 12, 8))
    assert gf.zblock() == 12                         # whole lattice far below the L2 budget: storage order
    gf.close()
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer((8, 8, 12, 8), zblock=5)     # must divide Nz
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer((8, 8, 12, 8), zblock=-1)
    big = lgf.GaugeFixer(64)                          # 64^4 FP64, 18-real: one time slice of links exceeds L2
    zb = big.zblock()
    big.close()
    assert 1 <= zb < 64 and 64 % zb == 0


# ------------------------------------------------------------------ LGF_OPT_ZT_PIPE: persistent (z,t) pass
@pytest.mark.parametrize("N", [(16, 16, 16, 16), (12, 12, 12, 12), (8, 8, 32, 16), (8, 8, 64, 64), (24, 24, 24, 24),
                               (8, 8, 16, 32)], ids=lambda n: "x".join(map(str, n)))
@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_zt_pipe_is_bitwise_the_plain_pass(lgf, N, prec):
    """The persistent (z,t) pass with cp.async prefetch does the same arithmetic in the same order: w is
    bitwise that of the plain kernel (and within the usual tolerance of the oracle); a pair without a
    persistent instantiation ((16, 32)) runs the plain kernel whatever the option says."""
    U = gen.gen_links(N, 0.5, 777)
    D, _, _ = oracle.measure(N, U)
    w = oracle.fourier_accelerate(N, D)
    cdt = np.complex128 if prec == "fp64" else np.complex64
    out = []
    for pipe in (0, 1):
        gf = lgf.GaugeFixer(N, precision=prec, zt_pipe=pipe)
        assert gf.uses_tiled_fft()
        gf.load_links(U.astype(cdt))
        gf.set_field(lgf.FIELD_DELTA, D.astype(cdt))
        gf.stage(lgf.STAGE_FOURIER)
        out.append(gf.get_field(lgf.FIELD_W))
        gf.load_links(U.astype(cdt))
        r = gf.iterate(ALPHA, 5)                   # several tiles per persistent CTA, graph replay on top
        out.append((r.F, r.theta))
        gf.close()
    assert np.array_equal(out[0], out[2]) and out[1] == out[3]
    assert np.abs(out[2].astype(np.complex128) - w).max() < (2e-13 if prec == "fp64" else 2e-5) * np.abs(w).max()


def test_zt_pipe_full_size_32(lgf):
    """The headline lattice: 1024 tiles over 296 persistent CTAs, three or four tiles each."""
    N = (32, 32, 32, 32)
    U = gen.gen_links(N, 0.5, gen.BASE_SEED + 32)
    res = []
    for pipe in (0, 1):
        gf = lgf.GaugeFixer(N, recon=12, zt_pipe=pipe)
        gf.load_links(U)
        r = gf.iterate(ALPHA, 3)
        res.append((r.F, r.theta, gf.get_links()))
        gf.close()
    assert res[0][0] == res[1][0] and res[0][1] == res[1][1] and np.array_equal(res[0][2], res[1][2])


# ------------------------------------------------------------------ LGF_OPT_FFT_PASSES: 2D + 2D and 4 x 1D structures
PASS_LATTICES = [((8, 8, 8, 8), 501), ((12, 12, 12, 12), 502), ((16, 16, 16, 16), 503), ((8, 8, 32, 16), 504),
                 ((8, 8, 64, 64), 505), ((48, 48, 8, 8), 506), ((16, 16, 16, 32), 507), ((8, 8, 24, 48), 508)]


@pytest.mark.parametrize("lat", PASS_LATTICES, ids=lambda v: "x".join(map(str, v[0])))
@pytest.mark.parametrize("passes", [4, 8])
def test_fft_pass_structures_match_oracle(lgf, lat, passes):
    """The 2D + 2D four-pass and the 4 x 1D eight-pass structures give the oracle's w
    (Alg. 1 lines 3-8) and the oracle's links after an iteration, FP64 and FP32, 4 and 9 fields."""
    N, seed = lat
    square_or_32xn = N[2] == N[3] or N[2] == 32
    U = gen.gen_links(N, 0.5, seed)
    D, _, _ = oracle.measure(N, U)
    w = oracle.fourier_accelerate(N, D)
    Uo = U.copy()
    hist = oracle.iterate(N, Uo, ALPHA, 1)
    if passes == 4 and not square_or_32xn:
        with pytest.raises(lgf.LgfError):
            lgf.GaugeFixer(N, fft_passes=4)          # the two-launch (z,t) pass is not instantiated for this tile
        return
    for prec, fb, tolw, tolu in (("fp64", 4, 2e-13, 1e-12), ("fp64", 9, 2e-13, 1e-12), ("fp32", 4, 2e-5, 1e-5)):
        cdt = np.complex128 if prec == "fp64" else np.complex64
        gf = lgf.GaugeFixer(N, precision=prec, fft_batch=fb, fft_passes=passes, recon=12 if fb == 4 else 18)
        assert gf.uses_tiled_fft() and gf.uses_gbuf() == (passes == 4 and fb == 4)
        gf.load_links(U.astype(cdt))
        gf.set_field(lgf.FIELD_DELTA, D.astype(cdt))
        gf.stage(lgf.STAGE_FOURIER)
        w2 = gf.get_field(lgf.FIELD_W).astype(np.complex128)
        assert np.abs(w2 - w).max() < tolw * np.abs(w).max()
        gf.load_links(U.astype(cdt))
        gf.reset_counters()
        r = gf.iterate(ALPHA, 1)
        kt = gf.kernel_times()
        nfft = sum(v[1] for k, v in kt.items() if k.startswith("fft_"))
        assert nfft == passes
        assert np.abs(gf.get_links().astype(np.complex128) - Uo).max() < tolu
        assert abs(r.theta - hist[1, 1]) <= (1e-10 if prec == "fp64" else 1e-4) * hist[1, 1]
        gf.close()


def test_fft_passes_validation(lgf):
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer(8, fft_passes=5)
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer((4, 6, 8, 12), fft_passes=8)            # not a tiled lattice
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer(8, fft_passes=8, accum_g=1)
    gf = lgf.GaugeFixer(8, fft_passes=4, accum_g=1)           # 2D + 2D keeps the g-building last pass
    gf.close()


# ------------------------------------------------------------------ 18-real storage and links that are not exactly SU(3)
def test_18_real_fused_path_projects_row_2_as_documented(lgf):
    """include/lgf.h (LGF_OPT_RECON) and DESIGN.md reading R15: links must be SU(3) to working precision.  With a
    deliberately non-unitary third row, FUSION = 0 multiplies all three rows like the oracle, while the fused kernel
    stores row 2 of g U g^dagger as conj(row0 x row1) of the product: rows 0, 1 agree with the oracle either way, row 2
    of the fused path differs by the size of the defect.  For exactly special unitary links both agree (other tests)."""
    N = (8, 8, 8, 8)
    U = gen.gen_links(N, 0.3, 31)
    U[:, :, 2, :] *= 1.0 + 1e-6                      # row 2 no longer conj(row0 x row1): defect 1e-6
    Uo = U.copy()
    oracle.iterate(N, Uo, ALPHA, 1)
    unf = lgf.GaugeFixer(N, recon=18, fusion=0)
    unf.load_links(U)
    unf.iterate(ALPHA, 1)
    assert np.abs(unf.get_links() - Uo).max() < 1e-12
    fus = lgf.GaugeFixer(N, recon=18)
    fus.load_links(U)
    fus.iterate(ALPHA, 1)
    Uf = fus.get_links()
    # rows 0, 1 of g U g^dagger only need rows 0, 1 of g and all of U ... whose row 2 enters through U g^dagger: first order in the defect
    assert np.abs(Uf[:, :, :2, :] - Uo[:, :, :2, :]).max() < 5e-6
    d2 = np.abs(Uf[:, :, 2, :] - Uo[:, :, 2, :]).max()
    assert 1e-7 < d2 < 5e-6                         # the projection is visible and of the size of the defect


# ------------------------------------------------------------------ LGF_OPT_TMARCH: several time slices per thread
@pytest.mark.parametrize("var", [dict(recon=12), dict(recon=18), dict(recon=18, precision="fp32"), dict(recon=12, accum_g=1),
                                 dict(recon=18, fft_batch=9), dict(recon=12, zblock=2)], ids=vid)
@pytest.mark.parametrize("tk", [2, 4])
def test_tmarch_gives_the_same_links(lgf, var, tk):
    """A thread of the link kernel that walks tk time slices takes the -t neighbour of its later sites from its own
    previous site: same products, so the links after 3 iterations are bitwise those of one site per thread, F and theta
    agree to the rounding of the partial sums, and the first iteration matches the oracle."""
    N = (8, 8, 8, 12) if tk == 4 else (8, 8, 8, 6)
    if var.get("accum_g") and N[3] == 6:
        N = (8, 8, 8, 8)
    fp32 = var.get("precision") == "fp32"
    U = gen.gen_links(N, 0.5, 606)
    Uo = U.copy()
    hist = oracle.iterate(N, Uo, ALPHA, 1)
    Uin = U.astype(np.complex64) if fp32 else U
    res = []
    for t in (1, tk):
        gf = lgf.GaugeFixer(N, tmarch=t, **var)
        gf.load_links(Uin)
        r1 = gf.iterate(ALPHA, 1)
        assert np.abs(gf.get_links().astype(np.complex128) - Uo).max() < (1e-5 if fp32 else 1e-12)
        assert abs(r1.theta - hist[1, 1]) <= (1e-4 if fp32 else 1e-10) * hist[1, 1]
        r3 = gf.iterate(ALPHA, 2)
        res.append((gf.get_links(), r3.F, r3.theta))
        gf.close()
    assert np.array_equal(res[0][0], res[1][0])
    assert abs(res[0][1] - res[1][1]) <= (1e-7 if fp32 else 1e-14) and abs(res[0][2] - res[1][2]) <= (1e-6 if fp32 else 1e-13) * res[0][2]


def test_tmarch_falls_back_when_it_does_not_divide(lgf):
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer(8, tmarch=3)
    N = (8, 8, 8, 6)                                  # 4 does not divide Nt = 6: one site per thread
    U = gen.gen_links(N, 0.5, 607)
    a, b = lgf.GaugeFixer(N, tmarch=4), lgf.GaugeFixer(N, tmarch=1)
    a.load_links(U); b.load_links(U)
    ra, rb = a.iterate(ALPHA, 2), b.iterate(ALPHA, 2)
    assert ra.F == rb.F and ra.theta == rb.theta and np.array_equal(a.get_links(), b.get_links())


# ------------------------------------------------------------------ LGF_OPT_LINK_TILE: the link kernel on 4D tiles
TILE_LATTICES = [(8, 8, 8, 8), (16, 16, 16, 16), (12, 12, 12, 12), (4, 6, 8, 12), (16, 8, 4, 6), (32, 32, 8, 8), (48, 48, 4, 4),
                 (64, 64, 4, 4), (24, 24, 6, 8), (8, 4, 4, 4), (32, 4, 4, 32), (64, 8, 8, 4)]


@pytest.mark.parametrize("var", [dict(recon=12), dict(recon=18), dict(recon=18, precision="fp32"), dict(recon=12, precision="fp32"),
                                 dict(recon=18, fft_batch=9), dict(recon=12, fft_path=1), dict(recon=12, zblock=2), dict(recon=12, gmap=1)], ids=vid)
@pytest.mark.parametrize("threads", [128, 256, 512])
def test_link_tile_gives_the_same_links(lgf, var, threads):
    """The tiled link kernel hands the anti-Hermitian parts of the new links to the +mu neighbours through shared memory
    instead of rebuilding the backward links: same link products, so the links after one iteration are bitwise those of the
    site kernel; Delta (hence F, theta) differs by the order of eight additions, and the iteration matches the oracle
    (links 1e-12 / 1e-5, F and theta 1e-10 / 1e-4 relative)."""
    fp32 = var.get("precision") == "fp32"
    for N in TILE_LATTICES:
        U = gen.gen_links(N, 0.5, 808 + N[0] + N[3])
        Uo = U.copy()
        if var.get("gmap"):
            oracle.set_exponential(1)
        try:
            hist = oracle.iterate(N, Uo, ALPHA, 1)
        finally:
            oracle.set_exponential(0)
        Uin = U.astype(np.complex64) if fp32 else U
        res = []
        for lt in (1, threads):
            gf = lgf.GaugeFixer(N, link_tile=lt, tmarch=1, **var)
            gf.load_links(Uin)
            r1 = gf.iterate(ALPHA, 1)
            assert np.abs(gf.get_links().astype(np.complex128) - Uo).max() < (1e-5 if fp32 else 1e-12), (N, lt)
            assert abs(r1.F - hist[1, 0]) <= (1e-4 if fp32 else 1e-10) * abs(hist[1, 0]), (N, lt)
            assert abs(r1.theta - hist[1, 1]) <= (1e-4 if fp32 else 1e-10) * hist[1, 1], (N, lt)
            D1 = gf.get_field(lgf.FIELD_DELTA)
            res.append((gf.get_links(), r1.F, r1.theta, D1))
            gf.close()
        assert np.array_equal(res[0][0], res[1][0]), N
        assert np.abs(res[0][3] - res[1][3]).max() <= (2e-5 if fp32 else 2e-14), N
        assert abs(res[0][1] - res[1][1]) <= (1e-6 if fp32 else 1e-14), N
        assert abs(res[0][2] - res[1][2]) <= (1e-5 if fp32 else 1e-13) * res[0][2], N


@pytest.mark.parametrize("threads", [128, 256, 512])
def test_link_tile_converges_to_the_golden_count(lgf, threads):
    """Algorithm 1 to theta <= 1e-15 with the tiled link kernel: the oracle's iteration count and final F (16^4 golden)."""
    it, F, th, ghist = read_golden(golden_path(16, gen.BASE_SEED + 16))
    U = gen.gen_links(16, 0.5, gen.BASE_SEED + 16)
    gf = lgf.GaugeFixer(16, recon=12, link_tile=threads)
    gf.load_links(U)
    r = gf.fix(ALPHA, 1e-15)
    assert r.converged == 1 and r.iterations == it
    assert abs(r.F - F) < 1e-10
    h = gf.history()
    assert np.abs(h[:, 0] - ghist[:, 0]).max() < 1e-10
    gf.close()


def test_link_tile_option_is_validated(lgf):
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer(8, link_tile=64)
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer(8, link_tile=-1)


# ------------------------------------------------------------------ LGF_OPT_LINK_STREAM: TMA-fed persistent link kernel
STREAM_LATTICES = [(16, 16, 16, 16), (16, 8, 4, 6), (32, 32, 8, 8), (32, 4, 4, 32), (48, 48, 4, 4), (64, 64, 4, 4), (64, 8, 8, 4),
                   (16, 16, 4, 24), (8, 8, 8, 8), (24, 24, 6, 8)]          # the last two: Nx Ny % 128 != 0, the option is ignored


@pytest.mark.parametrize("var", [dict(recon=12), dict(recon=18), dict(recon=18, precision="fp32"), dict(recon=12, precision="fp32"),
                                 dict(recon=12, zblock=2), dict(recon=12, gmap=1), dict(recon=12, graph=0)], ids=vid)
def test_link_stream_gives_the_same_links(lgf, var):
    """The streamed link kernel takes the thread's own links from a shared-memory ring filled by cp.async.bulk instead of
    loading them itself: same arithmetic per site, so the links after 1 and 3 iterations are bitwise those of the site
    kernel, F and theta agree to the order of the partial sums, and the first iteration matches the oracle."""
    fp32 = var.get("precision") == "fp32"
    for N in STREAM_LATTICES:
        U = gen.gen_links(N, 0.5, 909 + N[0] + N[3])
        Uo = U.copy()
        if var.get("gmap"):
            oracle.set_exponential(1)
        try:
            hist = oracle.iterate(N, Uo, ALPHA, 1)
        finally:
            oracle.set_exponential(0)
        Uin = U.astype(np.complex64) if fp32 else U
        res = []
        for ls in (0, 1):
            gf = lgf.GaugeFixer(N, link_stream=ls, tmarch=1, **var)
            gf.load_links(Uin)
            r1 = gf.iterate(ALPHA, 1)
            U1 = gf.get_links()
            assert np.abs(U1.astype(np.complex128) - Uo).max() < (1e-5 if fp32 else 1e-12), (N, ls)
            assert abs(r1.F - hist[1, 0]) <= (1e-4 if fp32 else 1e-10) * abs(hist[1, 0]), (N, ls)
            assert abs(r1.theta - hist[1, 1]) <= (1e-4 if fp32 else 1e-10) * hist[1, 1], (N, ls)
            D1 = gf.get_field(lgf.FIELD_DELTA)
            r3 = gf.iterate(ALPHA, 2)
            res.append((U1, D1, gf.get_links(), r3.F, r3.theta))
            gf.close()
        assert np.array_equal(res[0][0], res[1][0]), N
        if fp32:       # the FP32 site kernel adds the backward links in the order x, y, z, t, the streamed one in t, z, y, x
            assert np.abs(res[0][1] - res[1][1]).max() <= 2e-5, N
        else:
            assert np.array_equal(res[0][1], res[1][1]), N             # Delta: the same sums per site
        if fp32:       # a Delta that differs in the last place feeds the next g: the links stay equal to FP32 rounding
            assert np.abs(res[0][2] - res[1][2]).max() <= 2e-5, N
        else:
            assert np.array_equal(res[0][2], res[1][2]), N
        assert abs(res[0][3] - res[1][3]) <= (1e-6 if fp32 else 1e-14), N
        assert abs(res[0][4] - res[1][4]) <= (1e-5 if fp32 else 1e-13) * res[0][4], N


def test_link_stream_converges_to_the_golden_count(lgf):
    """Algorithm 1 to theta <= 1e-15 with the streamed link kernel: the oracle's iteration count, final F and F history
    (16^4 golden), with graph replay (default) and a stop decision taken by the persistent kernel's last CTA."""
    it, F, th, ghist = read_golden(golden_path(16, gen.BASE_SEED + 16))
    U = gen.gen_links(16, 0.5, gen.BASE_SEED + 16)
    for recon in (12, 18):
        gf = lgf.GaugeFixer(16, recon=recon, link_stream=1)
        gf.load_links(U)
        r = gf.fix(ALPHA, 1e-15)
        assert r.converged == 1 and r.iterations == it
        assert abs(r.F - F) < 1e-10
        h = gf.history()
        assert np.abs(h[:, 0] - ghist[:, 0]).max() < 1e-10
        gf.close()
    with pytest.raises(lgf.LgfError):
        lgf.GaugeFixer(16, link_stream=2)


# ------------------------------------------------------------------ ensemble.py: lattices pipelined through one GPU
def test_ensemble_pipeline_equals_one_lattice_at_a_time(lgf):
    """Seven different lattices through three slots (three contexts, streams and host threads): results and links
    are those of one context fixing them one after another, bitwise, and the first one matches the golden count."""
    import torch

    from paper_1210_8018_b200 import ensemble

    n = 8
    seeds = [gen.BASE_SEED + 8] + list(range(700, 706))
    ins = [torch.from_numpy(gen.gen_links(n, 0.3, s)).pin_memory() for s in seeds]
    outs = [torch.empty_like(t).pin_memory() for t in ins]
    ens = ensemble.EnsembleFixer(n, slots=3, recon=12)
    res = ens.run([t.numpy() for t in ins], [t.numpy() for t in outs], ALPHA, 1e-15)
    ens.close()
    it, F, th, hist = read_golden(golden_path(n, seeds[0]))
    assert res[0].iterations == it and abs(res[0].F - F) <= 1e-10
    gf = lgf.GaugeFixer(n, recon=12)
    for t, o, r in zip(ins, outs, res):
        gf.load_links(t.numpy())
        r1 = gf.fix(ALPHA, 1e-15)
        assert (r1.iterations, r1.F, r1.theta, r1.converged) == (r.iterations, r.F, r.theta, r.converged)
        assert np.array_equal(gf.get_links(), o.numpy())
    gf.close()
