"""GPU parity: the CUDA path (through the C ABI, liblgf.so) against the CPU oracle, element by
element, on the same seeded inputs.  Tolerances are BASELINE.json's north_star:
  after one iteration: links <= 1e-12 max abs, F and theta <= 1e-10 relative;
  after convergence:   iteration count within +-2 %, final F within 1e-10;
  FP32: links <= 1e-5 max abs after one iteration, converges to theta <= 1e-12.
Per-kernel taps use tighter, arithmetic-derived bounds."""
import os

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


def fixer(lgf, N, **kw):
    return lgf.GaugeFixer(N, **kw)


LATTICES = [
    # (extents, sigma, seed)            8^4 = BASELINE config 1; mixed extents span ragged tiles
    ((8, 8, 8, 8), 0.3, gen.BASE_SEED + 8),
    ((4, 6, 8, 12), 0.5, 77),
    ((16, 8, 4, 6), 0.5, 78),
    ((16, 16, 16, 16), 0.5, gen.BASE_SEED + 16),
    ((12, 12, 12, 12), 0.5, 79),        # radix-3 lines of the tiled FFT
]
VARIANTS = [dict(recon=18, fft_batch=4), dict(recon=12, fft_batch=4), dict(recon=18, fft_batch=9),
            dict(recon=12, fft_batch=9), dict(recon=18, fft_batch=4, fft_path=1),
            # the three separate kernels of the paper's kernel list instead of the fused default
            dict(recon=12, fft_batch=4, fusion=0), dict(recon=18, fft_batch=9, fusion=0)]


def ids(v):
    return "-".join(f"{k}{x}" for k, x in v.items()) if isinstance(v, dict) else "x".join(map(str, v[0]))


@pytest.mark.parametrize("recon", [18, 12])
def test_links_round_trip(lgf, recon):
    N = (4, 6, 8, 12)
    U = gen.gen_links(N, 0.5, 5)
    gf = fixer(lgf, N, recon=recon)
    gf.load_links(U)
    back = gf.get_links()
    if recon == 18:
        assert np.array_equal(back, U)
    else:
        assert np.array_equal(back[:, :, :2], U[:, :, :2])
        assert np.abs(back - U).max() < 1e-14            # row 2 rebuilt from unitarity
    # device-resident source and destination
    import torch
    Ud = torch.from_numpy(U).cuda()
    gf.load_links(Ud)
    assert np.abs(gf.get_links(device=True).cpu().numpy() - U).max() < 1e-14


@pytest.mark.parametrize("lat", LATTICES, ids=ids)
@pytest.mark.parametrize("var", VARIANTS, ids=ids)
def test_measure_matches_oracle(lgf, lat, var):
    N, sigma, seed = lat
    U = gen.gen_links(N, sigma, seed)
    D, F, th = oracle.measure(N, U)
    gf = fixer(lgf, N, **var)
    gf.load_links(U)
    F2, th2 = gf.measure()
    D2 = gf.get_field(lgf.FIELD_DELTA)
    assert np.abs(D2 - D).max() < 1e-13
    assert abs(F2 - F) <= 1e-12 * max(abs(F), 1e-3) + 1e-15
    assert abs(th2 - th) <= 1e-12 * th


@pytest.mark.parametrize("lat", LATTICES, ids=ids)
@pytest.mark.parametrize("var", VARIANTS, ids=ids)
def test_fourier_matches_oracle(lgf, lat, var):
    N, sigma, seed = lat
    U = gen.gen_links(N, sigma, seed)
    D, _, _ = oracle.measure(N, U)
    w = oracle.fourier_accelerate(N, D)
    gf = fixer(lgf, N, **var)
    gf.load_links(U)
    gf.set_field(lgf.FIELD_DELTA, D)
    gf.stage(lgf.STAGE_FOURIER)
    w2 = gf.get_field(lgf.FIELD_W)
    scale = np.abs(w).max()
    # row 2 of w is not needed by g (pin P15); the packed mode rebuilds it from anti-Hermiticity
    assert np.abs(w2 - w).max() < 2e-13 * scale


@pytest.mark.parametrize("var", VARIANTS[:4], ids=ids)
def test_g_and_update_match_oracle(lgf, var):
    N, sigma, seed = (4, 6, 8, 12), 0.5, 91
    U = gen.gen_links(N, sigma, seed)
    D, _, _ = oracle.measure(N, U)
    w = oracle.fourier_accelerate(N, D)
    g = oracle.build_g(w, ALPHA)
    gf = fixer(lgf, N, **var)
    gf.load_links(U)
    gf.set_field(lgf.FIELD_W, w)
    g2 = gf.get_field(lgf.FIELD_G, alpha=ALPHA)
    assert np.abs(g2 - g).max() < 1e-14
    gf.stage(lgf.STAGE_UPDATE, alpha=ALPHA)
    U1 = oracle.update_links(N, U.copy(), g)
    assert np.abs(gf.get_links() - U1).max() < 1e-13


@pytest.mark.parametrize("lat", LATTICES, ids=ids)
@pytest.mark.parametrize("var", VARIANTS, ids=ids)
def test_one_iteration_matches_oracle(lgf, lat, var):
    N, sigma, seed = lat
    U = gen.gen_links(N, sigma, seed)
    Uo = U.copy()
    hist = oracle.iterate(N, Uo, ALPHA, 1)
    gf = fixer(lgf, N, **var)
    gf.load_links(U)
    r = gf.iterate(ALPHA, 1)
    assert r.iterations == 1
    assert np.abs(gf.get_links() - Uo).max() < 1e-12
    assert abs(r.F - hist[1, 0]) <= 1e-10 * abs(hist[1, 0])
    assert abs(r.theta - hist[1, 1]) <= 1e-10 * hist[1, 1]
    h = gf.history()
    assert h.shape == (2, 2)
    assert np.allclose(h, hist, rtol=1e-10, atol=0)


@pytest.mark.parametrize("n,sigma,seed", [(8, 0.3, gen.BASE_SEED + 8), (8, 0.3, gen.BASE_SEED + 1008),
                                          (8, 0.3, gen.BASE_SEED + 2008), (16, 0.5, gen.BASE_SEED + 16),
                                          (16, 0.5, gen.BASE_SEED + 1016)])
@pytest.mark.parametrize("var", [VARIANTS[0], VARIANTS[1], VARIANTS[2], VARIANTS[4], VARIANTS[5]], ids=ids)
def test_convergence_matches_oracle_golden(lgf, n, sigma, seed, var):
    it, F, th, hist = read_golden(golden_path(n, seed))
    U = gen.gen_links(n, sigma, seed)
    gf = fixer(lgf, n, **var)
    gf.load_links(U)
    r = gf.fix(ALPHA, 1e-15)
    assert r.converged == 1 and r.theta <= 1e-15
    assert abs(r.iterations - it) <= 0.02 * it
    assert abs(r.F - F) <= 1e-10
    h = gf.history()
    assert h.shape[0] == r.iterations + 1
    k = min(h.shape[0], hist.shape[0]) - 3                  # the tail sits at the rounding floor
    assert np.allclose(h[:k, 0], hist[:k, 0], rtol=0, atol=1e-10)
    assert np.allclose(h[:k, 1], hist[:k, 1], rtol=1e-6, atol=1e-25)
    assert np.all(np.diff(h[:, 0]) >= -1e-15)              # F never decreases (pin P12)
    # the fixed links are unitary with det 1 and the plaquette is that of the input (pin P11)
    Ufix = gf.get_links()
    I = np.eye(3)
    assert np.abs(Ufix @ np.conj(np.swapaxes(Ufix, -1, -2)) - I).max() < 1e-12
    assert np.abs(np.linalg.det(Ufix) - 1).max() < 1e-12
    if n == 8:
        assert abs(oracle.plaquette(n, Ufix) - oracle.plaquette(n, U)) < 1e-12
    # calling fix again on converged links does nothing
    r2 = gf.fix(ALPHA, 1e-15)
    assert r2.iterations == 0 and r2.converged == 1 and r2.F == r.F


def test_iterate_equals_fix_prefix_and_is_deterministic(lgf):
    n, seed = 8, gen.BASE_SEED + 8
    U = gen.gen_links(n, 0.3, seed)
    a = fixer(lgf, n)
    a.load_links(U)
    ra = a.iterate(ALPHA, 12)
    b = fixer(lgf, n, check_interval=1)
    b.load_links(U)
    rb = b.iterate(ALPHA, 5)
    rb = b.iterate(ALPHA, 7)
    assert ra.iterations == 12 and rb.iterations == 7
    assert ra.F == rb.F and ra.theta == rb.theta            # bitwise: fixed-order reductions
    assert np.array_equal(a.get_links(), b.get_links())
    assert a.launch_count() > 12 * 3


def test_edge_cases(lgf):
    from helpers import unit_links
    n = (4, 4, 4, 4)
    gf = fixer(lgf, n, max_iter=3)
    # unit field: Delta = theta = 0, F = 1 exactly (pin P1): zero iterations
    gf.load_links(unit_links(n))
    r = gf.fix(ALPHA, 1e-15)
    assert (r.iterations, r.F, r.theta, r.converged) == (0, 1.0, 0.0, 1)
    # iteration cap: LGF_ERR_NOT_CONVERGED with the result still filled
    U = gen.gen_links(n, 0.5, 3)
    gf.load_links(U)
    with pytest.raises(lgf.LgfError) as e:
        gf.fix(ALPHA, 1e-15)
    assert e.value.code == lgf.ERR_NOT_CONVERGED
    r = gf.fix(ALPHA, 1e-15, allow_not_converged=True)
    assert r.iterations == 3 and r.converged == 0 and r.theta > 1e-15
    # stage order is checked
    with pytest.raises(lgf.LgfError):
        gf.stage(lgf.STAGE_UPDATE)
    # a NaN link is reported, not iterated on
    U[5, 2, 1, 1] = np.nan
    gf.load_links(U)
    with pytest.raises(lgf.LgfError) as e:
        gf.fix(ALPHA, 1e-15)
    assert e.value.code == lgf.ERR_NUMERIC
    # pure gauge field: F -> 1 (pin P13)
    gf2 = fixer(lgf, n)
    gf2.load_links(gen.gen_links(n, 0.0, 11))
    r = gf2.fix(ALPHA, 1e-15)
    assert r.converged and abs(r.F - 1) < 1e-12


@pytest.mark.parametrize("lat", [LATTICES[0], LATTICES[1], LATTICES[3]], ids=ids)
@pytest.mark.parametrize("var", [VARIANTS[0], VARIANTS[1]], ids=ids)
def test_fp32_variant(lgf, lat, var):
    N, sigma, seed = lat
    U = gen.gen_links(N, sigma, seed)
    Uo = U.copy()
    hist = oracle.iterate(N, Uo, ALPHA, 1)
    gf = fixer(lgf, N, precision="fp32", **var)
    gf.load_links(U.astype(np.complex64))
    r = gf.iterate(ALPHA, 1)
    assert np.abs(gf.get_links().astype(np.complex128) - Uo).max() < 1e-5
    assert abs(r.F - hist[1, 0]) < 1e-5 and abs(r.theta - hist[1, 1]) < 1e-4 * hist[1, 1]
    gf.load_links(U.astype(np.complex64))
    r = gf.fix(ALPHA, 1e-12)
    assert r.converged == 1 and r.theta <= 1e-12
    it_ref = oracle.fix(N, U.copy(), ALPHA, 1e-12)[0]
    assert abs(r.iterations - it_ref) <= max(1, 0.02 * it_ref)


def test_tiled_fft_is_taken_where_expected(lgf):
    for n, want in [(8, True), (12, True), (16, True), (24, True), (32, True), (48, True), (64, True), ((16, 16, 8, 8), True), ((32, 32, 32, 16), True), ((8, 8, 32, 64), True),
                    # N_s^3 x N_t and every other (Nz, Nt) pair of tiled extents
                    ((8, 8, 16, 32), True), ((8, 8, 8, 16), True), ((16, 16, 16, 32), True), ((24, 24, 24, 48), True),
                    ((32, 32, 32, 12), True), ((32, 32, 32, 24), True), ((12, 12, 32, 32), True), ((12, 12, 64, 8), True),
                    ((8, 16, 8, 8), False), (4, False), (36, False), ((8, 8, 8, 6), False), ((8, 8, 36, 8), False)]:
        gf = fixer(lgf, n)
        assert gf.uses_tiled_fft() == want, n
    assert not fixer(lgf, 16, fft_path=1).uses_tiled_fft()
    # FP32 tiles are 8 x-columns wide unless Nz = 12 (then 4): Nx = 12 with another Nz does not divide into
    # them and must take the generic transform instead of silently skipping x = 8..11
    for n, want in [(12, True), ((12, 12, 32, 32), False), ((12, 12, 16, 16), False), ((12, 12, 12, 48), True),
                    ((24, 24, 32, 32), True), ((8, 8, 12, 12), True)]:
        assert fixer(lgf, n, precision="fp32").uses_tiled_fft() == want, n


# Lines of 48 and 64 are shared by two threads (fft_tiled.cu, Line<T, N, 2>); lattices with
# Nx = Ny != Nz = Nt put them in the (x,y) passes or in the (z,t) pass at a size the oracle
# finishes in about a second.
SPLIT_LATTICES = [((64, 64, 8, 8), 81), ((8, 8, 64, 64), 82), ((48, 48, 12, 12), 83), ((16, 16, 48, 48), 84),
                  # (z,t) tiles with Nz = 32 != Nt: the paper's 32^3 x n lattices
                  ((32, 32, 32, 8), 85), ((8, 8, 32, 16), 86), ((8, 8, 32, 48), 87), ((8, 8, 32, 64), 88),
                  # every other (Nz, Nt) pair of tiled extents: N_s^3 x N_t shapes (T = 2L), mixed radix-3 / split
                  # lines on either axis, tiles that run one CTA per SM
                  ((16, 16, 16, 32), 89), ((8, 8, 24, 48), 90), ((8, 8, 32, 12), 91), ((8, 8, 32, 24), 92),
                  ((8, 8, 16, 64), 93), ((8, 8, 64, 16), 94), ((8, 8, 48, 64), 95), ((8, 8, 64, 48), 96),
                  ((16, 16, 8, 12), 97), ((8, 8, 12, 24), 98), ((8, 8, 48, 32), 99),
                  # Nx = 12: FP64 tiles (4 columns) divide it, FP32 tiles (8 columns) do not -> generic path in FP32
                  ((12, 12, 32, 32), 100), ((12, 12, 16, 16), 101)]
FP32_GENERIC = {(12, 12, 32, 32), (12, 12, 16, 16)}


@pytest.mark.parametrize("lat", SPLIT_LATTICES, ids=lambda v: "x".join(map(str, v[0])))
@pytest.mark.parametrize("fft_batch", [4, 9])
def test_split_line_fourier_matches_oracle(lgf, lat, fft_batch):
    N, seed = lat
    U = gen.gen_links(N, 0.5, seed)
    D, _, _ = oracle.measure(N, U)
    w = oracle.fourier_accelerate(N, D)
    for prec, tol in (("fp64", 2e-13), ("fp32", 2e-5)):
        gf = fixer(lgf, N, precision=prec, fft_batch=fft_batch)
        assert gf.uses_tiled_fft() == (not (prec == "fp32" and tuple(N) in FP32_GENERIC))
        gf.load_links(U if prec == "fp64" else U.astype(np.complex64))
        gf.set_field(lgf.FIELD_DELTA, D if prec == "fp64" else D.astype(np.complex64))
        gf.stage(lgf.STAGE_FOURIER)
        w2 = gf.get_field(lgf.FIELD_W).astype(np.complex128)
        assert np.abs(w2 - w).max() < tol * np.abs(w).max()


@pytest.mark.parametrize("lat", SPLIT_LATTICES, ids=lambda v: "x".join(map(str, v[0])))
def test_split_line_one_iteration(lgf, lat):
    N, seed = lat
    U = gen.gen_links(N, 0.5, seed)
    Uo = U.copy()
    hist = oracle.iterate(N, Uo, ALPHA, 1)
    for prec, recon, tol in (("fp64", 12, 1e-12), ("fp64", 18, 1e-12), ("fp32", 18, 1e-5)):
        gf = fixer(lgf, N, precision=prec, recon=recon)
        gf.load_links(U if prec == "fp64" else U.astype(np.complex64))
        r = gf.iterate(ALPHA, 1)
        assert np.abs(gf.get_links().astype(np.complex128) - Uo).max() < tol
        assert abs(r.theta - hist[1, 1]) <= (1e-10 if prec == "fp64" else 1e-4) * hist[1, 1]
        r = gf.iterate(ALPHA, 2)                       # three fused iterations stay on the oracle's trajectory
    Uo3 = U.copy()
    hist3 = oracle.iterate(N, Uo3, ALPHA, 3)
    gf = fixer(lgf, N, recon=12)
    gf.load_links(U)
    r = gf.iterate(ALPHA, 3)
    assert np.abs(gf.get_links() - Uo3).max() < 1e-12
    assert abs(r.F - hist3[3, 0]) <= 1e-10 * abs(hist3[3, 0]) and abs(r.theta - hist3[3, 1]) <= 1e-10 * hist3[3, 1]


def test_24_one_iteration(lgf):
    n = 24
    U = gen.gen_links(n, 0.5, 80)
    Uo = U.copy()
    hist = oracle.iterate(n, Uo, ALPHA, 1)
    for prec, tol in (("fp64", 1e-12), ("fp32", 1e-5)):
        gf = fixer(lgf, n, precision=prec, recon=12)
        gf.load_links(U if prec == "fp64" else U.astype(np.complex64))
        r = gf.iterate(ALPHA, 1)
        assert np.abs(gf.get_links().astype(np.complex128) - Uo).max() < tol
        assert abs(r.theta - hist[1, 1]) <= (1e-10 if prec == "fp64" else 1e-4) * hist[1, 1]


def test_headline_32_12real_one_iteration_and_golden(lgf):
    """BASELINE config 3 in the configuration bench.py times: 32^4, FP64, 12-real links."""
    n, seed = 32, gen.BASE_SEED + 32
    U = gen.gen_links(n, 0.5, seed)
    gf = fixer(lgf, n, recon=12)
    gf.load_links(U)
    r1 = gf.iterate(ALPHA, 1)
    U1 = gf.get_links()
    Uo = U.copy()
    hist = oracle.iterate(n, Uo, ALPHA, 1)
    assert np.abs(U1 - Uo).max() < 1e-12
    assert abs(r1.F - hist[1, 0]) <= 1e-10 * abs(hist[1, 0])
    assert abs(r1.theta - hist[1, 1]) <= 1e-10 * hist[1, 1]
    it, F, th, ghist = read_golden(golden_path(n, seed))
    assert np.array_equal(hist[1], ghist[1])                  # the golden file belongs to this input
    gf.load_links(U)
    r = gf.fix(ALPHA, 1e-15)
    assert r.converged == 1 and abs(r.iterations - it) <= 0.02 * it and abs(r.F - F) <= 1e-10
    h = gf.history()
    k = min(h.shape[0], ghist.shape[0]) - 3
    assert np.allclose(h[:k, 0], ghist[:k, 0], rtol=0, atol=1e-10) and np.allclose(h[:k, 1], ghist[:k, 1], rtol=1e-6, atol=1e-25)


def _mem_available_gb():
    try:
        with open("/proc/meminfo") as f:
            for line in f:
                if line.startswith("MemAvailable:"):
                    return int(line.split()[1]) / 1e6
    except OSError:
        pass
    return 0.0


def _unitarity_defect(U):
    I = np.eye(3)
    worst = 0.0
    for lo in range(0, U.shape[0], 1 << 20):                 # chunked: the full product would double the memory
        u = U[lo:lo + (1 << 20)].astype(np.complex128)
        worst = max(worst, float(np.abs(u @ np.conj(np.swapaxes(u, -1, -2)) - I).max()),
                    float(np.abs(np.linalg.det(u) - 1).max()))
    return worst


def _golden_count(hist, eps):
    """Iterations the oracle's trajectory needs to reach theta <= eps (R2: stop at the first theta <= eps)."""
    idx = np.nonzero(hist[:, 1] <= eps)[0]
    assert idx.size, "golden trajectory never reaches eps"
    return int(idx[0])


@pytest.mark.slow
def test_full_size_48_fp32(lgf):
    """BASELINE config 4 in the configuration bench.py times: 48^4, FP32 storage and FFT, FP64 sums,
    18-real links.  One iteration against the oracle element by element (north_star: 1e-5), then
    Algorithm 1 to theta <= 1e-12 against the oracle's golden trajectory (tests/golden/fix_48_*.txt, FP64
    oracle on the same generator output): iteration count within +-2 %, final F within 1e-5, the (F, theta)
    prefix, plus the invariants that hold at any size.  The ACCUM_G leg is held to the same golden."""
    n, seed = 48, gen.BASE_SEED + 48
    git, gF, gth, ghist = read_golden(golden_path(n, seed))
    n12 = _golden_count(ghist, 1e-12)
    U = gen.gen_links(n, 0.5, seed)
    gf = fixer(lgf, n, precision="fp32", recon=18)
    assert gf.uses_tiled_fft() and gf.uses_gbuf()
    U32 = U.astype(np.complex64)
    gf.load_links(U32)
    _, F0, th0 = oracle.measure(n, U, want_delta=False)
    assert F0 == ghist[0, 0] and th0 == ghist[0, 1]           # the golden file belongs to this input
    Fg, thg = gf.measure()
    assert abs(Fg - F0) < 1e-6 and abs(thg - th0) <= 1e-5 * th0
    r1 = gf.iterate(ALPHA, 1)
    U1 = gf.get_links().astype(np.complex128)
    Uo = U.copy()
    hist = oracle.iterate(n, Uo, ALPHA, 1)
    assert np.array_equal(hist[1], ghist[1])
    assert np.abs(U1 - Uo).max() < 1e-5
    assert abs(r1.F - hist[1, 0]) < 1e-5 and abs(r1.theta - hist[1, 1]) <= 1e-4 * hist[1, 1]
    del Uo, U1

    def check_against_golden(fx):
        fx.load_links(U32)
        r = fx.fix(ALPHA, 1e-12)
        assert r.converged == 1 and r.theta <= 1e-12
        assert abs(r.iterations - n12) <= max(1, int(0.02 * n12)), (r.iterations, n12)
        assert abs(r.F - ghist[r.iterations, 0]) < 1e-5 and abs(r.F - gF) < 1e-5
        h = fx.history()
        assert h.shape[0] == r.iterations + 1
        k = min(h.shape[0], n12) - 6                          # FP32 theta leaves the FP64 trajectory near its floor
        assert np.allclose(h[:k, 0], ghist[:k, 0], rtol=0, atol=1e-5)
        # theta = mean |Delta|^2 and an element of Delta carries about 2e-7 of absolute FP32 rounding (8 sums of O(1)
        # links), i.e. a relative error of 2e-7 / sqrt(theta) in Delta and twice that in theta: 2e-3 while theta >= 1e-4
        # (measured 3e-5 at theta = 1e-3), a few per cent further down (measured 3e-3 at theta = 3e-7)
        big = ghist[:k, 1] >= 1e-4
        assert np.allclose(h[:k, 1][big], ghist[:k, 1][big], rtol=2e-3, atol=0)
        assert np.allclose(h[:k, 1][~big], ghist[:k, 1][~big], rtol=5e-2, atol=0)
        assert np.all(np.diff(h[:, 0]) >= -1e-6)              # F never decreases (pin P12), FP32 rounding
        Ufix = fx.get_links()
        assert _unitarity_defect(Ufix) < 5e-5                 # no reunitarisation of links (reading R18)
        assert abs(oracle.plaquette(n, Ufix.astype(np.complex128)) - oracle.plaquette(n, U)) < 1e-5
        return r, Ufix

    r, Ufix = check_against_golden(gf)
    gf.close()
    # LGF_OPT_ACCUM_G at the same size (the configuration `bench.py --accum-g 1 --workload 48^4` times)
    ga = fixer(lgf, n, precision="fp32", recon=18, accum_g=1)
    ga.load_links(U32)
    ra1 = ga.iterate(ALPHA, 1)
    assert abs(ra1.F - hist[1, 0]) < 1e-5 and abs(ra1.theta - hist[1, 1]) <= 1e-4 * hist[1, 1]
    ra, Ua = check_against_golden(ga)
    assert np.abs(Ua - Ufix).max() < 5e-3                     # same minimum; FP32 rounding differs along the way
    ga.close()


@pytest.mark.slow
def test_full_size_64_fp64(lgf):
    """BASELINE config 5 in the configuration bench.py times: 64^4, FP64, 18-real links (9.7 GB of
    links).  Measure and one iteration against the oracle element by element, then Algorithm 1 to
    theta <= 1e-15 against the oracle's golden trajectory (tests/golden/fix_64_*.txt): iteration count within
    +-2 %, final F within 1e-10, the (F, theta) prefix, plus the invariants that hold at any size.  The
    ACCUM_G leg is held to the same golden.  Needs about 45 GB of host memory (explicit skip otherwise)."""
    if _mem_available_gb() < 48:
        pytest.skip("needs about 45 GB of host memory")
    n, seed = 64, gen.BASE_SEED + 64
    git, gF, gth, ghist = read_golden(golden_path(n, seed))
    U = gen.gen_links(n, 0.6, seed)
    gf = fixer(lgf, n, recon=18)
    assert gf.uses_tiled_fft() and gf.uses_gbuf()             # 64^2 planes: 2-CTA cluster variant of the last pass
    assert gf.zblock() < 64                                   # one time slice of links exceeds L2: blocked site walk
    gf.load_links(U)
    D, F0, th0 = oracle.measure(n, U)
    assert F0 == ghist[0, 0] and th0 == ghist[0, 1]           # the golden file belongs to this input
    Fg, thg = gf.measure()
    assert abs(Fg - F0) <= 1e-12 * max(abs(F0), 1e-3) + 1e-15 and abs(thg - th0) <= 1e-12 * th0
    assert np.abs(gf.get_field(lgf.FIELD_DELTA) - D).max() < 1e-13
    del D
    p0 = oracle.plaquette(n, U)
    r1 = gf.iterate(ALPHA, 1)
    U1 = gf.get_links()
    hist = oracle.iterate(n, U, ALPHA, 1)                     # in place: U becomes the oracle's links after one iteration
    assert np.array_equal(hist[1], ghist[1])
    worst = 0.0
    for lo in range(0, U.shape[0], 1 << 20):
        worst = max(worst, float(np.abs(U1[lo:lo + (1 << 20)] - U[lo:lo + (1 << 20)]).max()))
    assert worst < 1e-12
    assert abs(r1.F - hist[1, 0]) <= 1e-10 * abs(hist[1, 0]) and abs(r1.theta - hist[1, 1]) <= 1e-10 * hist[1, 1]
    assert abs(oracle.plaquette(n, U1) - p0) < 1e-12          # a gauge transformation (pin P11)
    del U1

    def check_against_golden(fx):
        """fx holds the links after one iteration: the rest of the trajectory is rows 1.. of the golden file"""
        r = fx.fix(ALPHA, 1e-15)
        assert r.converged == 1 and r.theta <= 1e-15
        assert abs(1 + r.iterations - git) <= int(0.02 * git), (r.iterations, git)
        assert abs(r.F - gF) <= 1e-10
        h = fx.history()
        assert h.shape[0] == r.iterations + 1
        k = min(h.shape[0], ghist.shape[0] - 1) - 3           # the tail sits at the rounding floor
        assert np.allclose(h[:k, 0], ghist[1:1 + k, 0], rtol=0, atol=1e-10)
        assert np.allclose(h[:k, 1], ghist[1:1 + k, 1], rtol=1e-6, atol=1e-25)
        assert np.all(np.diff(h[:, 0]) >= -1e-15)
        return r

    r = check_against_golden(gf)                              # continues from the links after one iteration
    Ufix = gf.get_links()
    assert _unitarity_defect(Ufix) < 1e-12
    assert abs(oracle.plaquette(n, Ufix) - p0) < 1e-12
    gf.close()
    # LGF_OPT_ACCUM_G at the same size, from the oracle's links after one iteration, against the same golden rows
    ga = fixer(lgf, n, recon=18, accum_g=1)
    ga.load_links(U)
    ra = check_against_golden(ga)
    del U
    Ua = ga.get_links()
    assert _unitarity_defect(Ua) < 1e-12
    worst = 0.0
    for lo in range(0, Ua.shape[0], 1 << 20):
        worst = max(worst, float(np.abs(Ua[lo:lo + (1 << 20)] - Ufix[lo:lo + (1 << 20)]).max()))
    assert worst < 1e-9                                       # the same minimum
    ga.close()
