"""Pins for the CPU oracle (oracle/lgf_oracle.c): what the paper and the mathematics fix.

The paper (arXiv 1210.8018) prints no worked numeric example, so the oracle is pinned to
closed forms, brute force, a library FFT and invariants.
Each test names the part of the oracle a plausible mistake in which it would catch.
CPU only (-m "not gpu").
"""
import numpy as np
import pytest

import gen
import oracle
from helpers import (GELL_MANN, dag, dft4d_bruteforce, expm_batch, gauge_transform, lat,
                     random_su3_algebra, shift, unit_links, volume)

ALPHA = 0.08
MIXED = (4, 4, 6, 8)


def rough_links(N, sigma=0.5, seed=7):
    return gen.gen_links(N, sigma, seed)


# ---------------------------------------------------------------- O0 tables / mask

def test_tables_closed_form_and_pmax():
    """s_mu[k] = 4 sin^2(pi k/N) = 2 - 2 cos(2 pi k/N) (eigenvalues of -d^2 on plane waves);
    p_max^2 = 16 for even extents, 4 sin^2(pi/3)=3 per odd axis of extent 3 (R5, R6)."""
    tabs, pmax2 = oracle.momentum_tables((4, 6, 8, 3))
    for n, t in zip((4, 6, 8, 3), tabs):
        k = np.arange(n)
        assert np.allclose(t, 2 - 2 * np.cos(2 * np.pi * k / n), atol=1e-14)
    assert abs(pmax2 - (4 + 4 + 4 + 3)) < 1e-13
    assert abs(oracle.momentum_tables(8)[1] - 16) < 1e-14


def test_mask_is_eigenvalue_ratio_of_lattice_laplacian():
    """Apply -d^2 (second differences) to a plane wave and read off p^2: M = p_max^2/p^2 (R5, R7)."""
    N = (4, 6, 2, 8)
    V = volume(N)
    M = oracle.mask(N)
    assert M[0] == 0.0
    idx = np.arange(V)
    c = [(idx // int(np.prod(N[:d]))) % N[d] for d in range(4)]
    for k in [(1, 0, 0, 0), (2, 3, 1, 4), (3, 5, 0, 7), (0, 0, 1, 0)]:
        wave = np.exp(2j * np.pi * sum(k[d] * c[d] / N[d] for d in range(4)))
        lap = sum(2 * wave - shift(N, wave, mu, 1) - shift(N, wave, mu, -1) for mu in range(4))
        p2 = (lap / wave).real
        assert np.ptp(p2) < 1e-12
        kk = k[0] + N[0] * (k[1] + N[1] * (k[2] + N[2] * k[3]))
        assert abs(M[kk] - 16.0 / p2[0]) < 1e-12
    assert abs(M[2 + N[0] * (3 + N[1] * (1 + N[2] * 4))] - 1.0) < 1e-14  # the corner mode


# ---------------------------------------------------------------- O1 measure

def test_P1_unit_field():
    D, F, th = oracle.measure(MIXED, unit_links(MIXED))
    assert F == 1.0 and th == 0.0 and np.all(D == 0)


def test_P2_constant_field():
    """U_mu(x) = C_mu: Delta = 0 (needs the periodic wrap of x - nu), F = (1/12) sum Re Tr C_mu."""
    rng = np.random.default_rng(1)
    C = expm_batch(random_su3_algebra(rng, (4,))[0])
    U = np.ascontiguousarray(np.broadcast_to(C, (volume(MIXED), 4, 3, 3)))
    D, F, th = oracle.measure(MIXED, U)
    assert np.abs(D).max() < 1e-14 and th < 1e-28
    assert abs(F - np.trace(C, axis1=1, axis2=2).real.sum() / 12) < 1e-14


def test_P3_cartan_links_closed_form():
    """Diagonal links: Delta_aa = 2i sum_nu[sin phi_a,nu(x-nu) - sin phi_a,nu(x)] minus the mean over a.
    Catches sign / neighbour-direction / trace / normalisation mistakes with no matrix code."""
    N = MIXED
    V = volume(N)
    rng = np.random.default_rng(2)
    phi = rng.uniform(-np.pi, np.pi, size=(V, 4, 3))
    phi[..., 2] = -phi[..., 0] - phi[..., 1]
    U = np.zeros((V, 4, 3, 3), dtype=np.complex128)
    for a in range(3):
        U[:, :, a, a] = np.exp(1j * phi[..., a])
    D, F, th = oracle.measure(N, U)
    d = np.zeros((V, 3))
    for nu in range(4):
        sn = np.sin(phi[:, nu, :])
        d += shift(N, sn, nu, -1) - sn
    d = 2 * d
    d -= d.mean(axis=1, keepdims=True)
    expect = np.zeros((V, 3, 3), dtype=np.complex128)
    for a in range(3):
        expect[:, a, a] = 1j * d[:, a]
    assert np.abs(D - expect).max() < 1e-13
    assert abs(F - np.cos(phi).sum() / (12 * V)) < 1e-14
    assert abs(th - (d ** 2).sum() / (3 * V)) < 1e-12 * th


def test_P4_delta_structure():
    """sum_x Delta = 0 (telescoping, periodic), Delta anti-Hermitian and traceless."""
    U = rough_links(MIXED)
    D, F, th = oracle.measure(MIXED, U)
    assert np.abs(D.sum(axis=0)).max() < 1e-12
    assert np.abs(D + dag(D)).max() == 0 or np.abs(D + dag(D)).max() < 1e-15
    assert np.abs(np.trace(D, axis1=1, axis2=2)).max() < 1e-14
    assert abs(th - (np.abs(D) ** 2).sum() / (3 * volume(MIXED))) < 1e-13 * th


def test_P17_global_colour_rotation():
    U = rough_links(MIXED)
    rng = np.random.default_rng(3)
    h = expm_batch(random_su3_algebra(rng, ())[0])
    Uh = np.ascontiguousarray(h @ U @ dag(h))
    D, F, th = oracle.measure(MIXED, U)
    Dh, Fh, thh = oracle.measure(MIXED, Uh)
    assert abs(F - Fh) < 1e-14 and abs(th - thh) < 1e-13 * th
    assert np.abs(Dh - h @ D @ dag(h)).max() < 1e-13


def test_P19_delta_is_the_gradient_of_F():
    """g = exp(eps Delta): dF/d eps = theta/8 (sign and scale of Delta, independent of any FFT)."""
    N = (4, 4, 4, 6)
    U = rough_links(N, sigma=0.4)
    D, F, th = oracle.measure(N, U)
    eps = 1e-5
    Fp = oracle.measure(N, gauge_transform(N, U, expm_batch(eps * D)), want_delta=False)[1]
    Fm = oracle.measure(N, gauge_transform(N, U, expm_batch(-eps * D)), want_delta=False)[1]
    assert abs((Fp - Fm) / (2 * eps) - th / 8) < 1e-6 * th


# ---------------------------------------------------------------- O3-O5 FFT

@pytest.mark.parametrize("n", [1, 2, 3, 4, 6, 8, 9, 12, 16, 18, 24, 32, 36, 48, 54, 64, 5, 7, 30])
def test_fft1d_against_definition_and_numpy(n):
    rng = np.random.default_rng(n)
    x = rng.normal(size=n) + 1j * rng.normal(size=n)
    j = np.arange(n)
    direct = np.exp(-2j * np.pi * np.outer(j, j) / n) @ x
    assert np.abs(oracle.fft1d(x, -1) - direct).max() < 1e-13 * n
    assert np.abs(oracle.fft1d(x, -1) - np.fft.fft(x)).max() < 1e-13 * n
    assert np.abs(oracle.fft1d(x, +1) - np.fft.ifft(x) * n).max() < 1e-13 * n


@pytest.mark.parametrize("N", [(4, 4, 4, 4), (2, 4, 6, 3)])
def test_P5_fft4d_bruteforce(N):
    """O(V^2) DFT from the definition: pins the axis <-> index mapping and the sign."""
    rng = np.random.default_rng(5)
    V = volume(N)
    f = rng.normal(size=V) + 1j * rng.normal(size=V)
    for sign in (-1, +1):
        ref = dft4d_bruteforce(N, f, sign)
        assert np.abs(oracle.fft4d(N, f, sign) - ref).max() < 1e-13 * np.abs(ref).max()


def test_P6_roundtrip_parseval_P16_numpy():
    N = (8, 6, 4, 12)
    V = volume(N)
    rng = np.random.default_rng(6)
    f = rng.normal(size=V) + 1j * rng.normal(size=V)
    fk = oracle.fft4d(N, f, -1)
    assert np.abs(oracle.fft4d(N, fk, +1) / V - f).max() < 1e-14 * 10
    assert abs((np.abs(f) ** 2).sum() - (np.abs(fk) ** 2).sum() / V) < 1e-13 * V
    assert np.abs(fk - np.fft.fftn(lat(N, f)).reshape(V)).max() < 1e-13 * np.abs(fk).max()


# ---------------------------------------------------------------- O0-O5 together

def test_P7_fft_free_laplacian_identity():
    """-lap w = p_max^2 (Delta - mean Delta): pins lattice p^2, p_max^2, zero mode, 1/V, axis mapping."""
    N = MIXED
    D = oracle.measure(N, rough_links(N))[0]
    w = oracle.fourier_accelerate(N, D)
    lap = sum(2 * w - shift(N, w, mu, 1) - shift(N, w, mu, -1) for mu in range(4))
    rhs = 16.0 * (D - D.mean(axis=0))
    assert np.abs(lap - rhs).max() < 1e-12
    assert np.abs(w.mean(axis=0)).max() < 1e-13          # zero mode removed (M(0) = 0)


def test_P9_w_antihermitian_traceless_and_P14_sign_independence():
    N = MIXED
    V = volume(N)
    D = oracle.measure(N, rough_links(N))[0]
    w = oracle.fourier_accelerate(N, D)
    assert np.abs(w + dag(w)).max() < 1e-13
    assert np.abs(np.trace(w, axis1=1, axis2=2)).max() < 1e-13
    M = oracle.mask(N)
    for (i, j) in [(0, 1), (1, 1), (2, 0)]:
        f = np.ascontiguousarray(D[:, i, j])
        flipped = oracle.fft4d(N, oracle.fft4d(N, f, +1) * M, -1) / V
        assert np.abs(flipped - w[:, i, j]).max() < 1e-13


# ---------------------------------------------------------------- O6 g

def test_P10_g_is_SU3_and_is_gram_schmidt_on_rows():
    N = MIXED
    w = oracle.fourier_accelerate(N, oracle.measure(N, rough_links(N))[0])
    g = oracle.build_g(w, ALPHA)
    assert np.abs(g @ dag(g) - np.eye(3)).max() < 1e-13
    assert np.abs(np.linalg.det(g) - 1).max() < 1e-13
    # m = 1 + (alpha/2) w;  Gram-Schmidt on rows <=> m g^dagger lower triangular with real
    # positive diagonal on rows 0, 1 (pins rows-not-columns, the order 0,1 and the inner product)
    m = np.eye(3) + (ALPHA / 2) * w
    L = m @ dag(g)
    assert np.abs(L[:, 0, 1]).max() < 1e-13 and np.abs(L[:, 0, 2]).max() < 1e-13
    assert np.abs(L[:, 1, 2]).max() < 1e-13
    assert np.abs(L[:, 0, 0].imag).max() < 1e-13 and L[:, 0, 0].real.min() > 0
    assert np.abs(L[:, 1, 1].imag).max() < 1e-13 and L[:, 1, 1].real.min() > 0
    # coefficient alpha/2 (R10): |m_row0| = L00 must equal |row 0 of 1 + 0.04 w|
    assert np.abs(L[:, 0, 0].real - np.linalg.norm(m[:, 0, :], axis=1)).max() < 1e-13


def test_P15_third_row_of_w_is_irrelevant():
    N = (4, 4, 4, 4)
    w = oracle.fourier_accelerate(N, oracle.measure(N, rough_links(N))[0])
    w2 = w.copy()
    w2[:, 2, :] = 123.0
    assert np.array_equal(oracle.build_g(w, ALPHA), oracle.build_g(w2, ALPHA))


# ---------------------------------------------------------------- O7 update

def test_update_is_the_gauge_transformation_and_P11_plaquette():
    N = MIXED
    U = rough_links(N)
    g = gen.gen_haar_field(N, 99)
    expect = gauge_transform(N, U, g)
    p0 = oracle.plaquette(N, U)
    U2 = oracle.update_links(N, U.copy(), g)
    assert np.abs(U2 - expect).max() < 1e-14
    assert abs(oracle.plaquette(N, U2) - p0) < 1e-13
    # plaquette against an np.roll re-derivation, so that P11 does not rest on itself
    acc = 0.0
    for mu in range(4):
        for nu in range(mu + 1, 4):
            P = U[:, mu] @ shift(N, U[:, nu], mu, 1) @ dag(shift(N, U[:, mu], nu, 1)) @ dag(U[:, nu])
            acc += np.trace(P, axis1=1, axis2=2).real.sum()
    assert abs(p0 - acc / (18 * volume(N))) < 1e-13
    assert abs(oracle.plaquette(N, unit_links(N)) - 1.0) < 1e-15


# ---------------------------------------------------------------- whole loop

def test_P8_closed_form_contraction_factor():
    """Unit field transformed by exp(i eps omega.lambda/2): theta_1/theta_0 -> (1 - 16 alpha)^2 = 0.0784.
    Pins alpha/2 (not alpha or alpha/4), the sign of the step, p_max^2 = 16 and the update ordering."""
    N = (4, 4, 6, 8)
    rng = np.random.default_rng(8)
    a, _ = random_su3_algebra(rng, (volume(N),))
    ratios = []
    for eps in (1e-3, 1e-5):
        U = gauge_transform(N, unit_links(N), expm_batch(eps * a))
        h = oracle.iterate(N, U, ALPHA, 1)
        ratios.append(h[1, 1] / h[0, 1])
    assert abs(ratios[0] - 0.0784) < 2e-5
    assert abs(ratios[1] - 0.0784) < 1e-8
    # a different alpha moves it as (1 - 16 alpha)^2
    U = gauge_transform(N, unit_links(N), expm_batch(1e-5 * a))
    h = oracle.iterate(N, U, 0.05, 1)
    assert abs(h[1, 1] / h[0, 1] - (1 - 16 * 0.05) ** 2) < 1e-8


def test_P12_F_monotone_and_P11_plaquette_along_a_run():
    N = (4, 4, 4, 8)
    U = rough_links(N, sigma=0.5, seed=11)
    p0 = oracle.plaquette(N, U)
    for _ in range(6):
        h = oracle.iterate(N, U, ALPHA, 1)
        assert h[1, 0] >= h[0, 0]
        assert abs(oracle.plaquette(N, U) - p0) < 1e-12
    assert np.abs(U @ dag(U) - np.eye(3)).max() < 1e-13


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_P13_pure_gauge_field_is_fixed_to_F_equal_1(seed):
    N = (4, 4, 4, 4)
    U = gen.gen_links(N, 0.0, seed)                      # Haar-random gauge transform of U = 1
    assert abs(oracle.plaquette(N, U) - 1) < 1e-13
    it, F, th, hist = oracle.fix(N, U, ALPHA, 1e-15)
    assert 0 < it < 100 and th <= 1e-15
    assert abs(F - 1) < 1e-12
    assert np.all(np.diff(hist[:, 0]) >= -1e-15)
    assert hist.shape[0] == it + 1


def test_fix_semantics():
    """iterations = executions of the loop body (R16); 0 if already fixed; -1 at the cap (R17);
    stop test is theta <= eps (R2)."""
    N = (4, 4, 4, 4)
    it, F, th, hist = oracle.fix(N, unit_links(N), ALPHA, 1e-15)
    assert it == 0 and F == 1.0 and th == 0.0 and hist.shape[0] == 1
    U = rough_links(N, sigma=0.3)
    it, F, th, hist = oracle.fix(N, U.copy(), ALPHA, 1e-15, max_iter=3)
    assert it == -1 and th > 1e-15
    it2, F2, th2, hist2 = oracle.fix(N, U.copy(), ALPHA, 1e-15)
    assert it2 > 3 and th2 <= 1e-15 and hist2[it2 - 1, 1] > 1e-15
    h = oracle.iterate(N, U.copy(), ALPHA, 5)
    assert np.array_equal(h, hist2[:6])
    # eps equal to a theta on the trajectory stops there
    it3 = oracle.fix(N, U.copy(), ALPHA, hist2[4, 1])[0]
    assert it3 == 4


def test_P18_iteration_count_is_robust_to_rounding_noise():
    N = (4, 4, 4, 4)
    U = rough_links(N, sigma=0.3, seed=5)
    rng = np.random.default_rng(18)
    Un = U * (1 + 1e-15 * rng.normal(size=U.shape))
    a = oracle.fix(N, U.copy(), ALPHA, 1e-15)
    b = oracle.fix(N, np.ascontiguousarray(Un), ALPHA, 1e-15)
    assert a[0] == b[0] and abs(a[1] - b[1]) < 1e-13


# ---------------------------------------------------------------- variant: exact exponential
def _random_ah_traceless(rng, n, scale):
    a = rng.normal(size=(n, 3, 3)) + 1j * rng.normal(size=(n, 3, 3))
    a = a - np.conj(np.swapaxes(a, -1, -2))
    a = a - (np.trace(a, axis1=-2, axis2=-1) / 3)[:, None, None] * np.eye(3)
    return scale * a


def test_exp_variant_closed_form_library_and_group():
    """g = exp((alpha/2) w), eq. 1.2 as written: closed form on diagonal w, scipy's expm
    (a library routine, Pade) on random anti-Hermitian traceless w over a wide range of norms, SU(3)."""
    from scipy.linalg import expm

    rng = np.random.default_rng(5)
    alpha = 0.08
    ph = rng.normal(size=(64, 2)) * 5
    w = np.zeros((64, 3, 3), dtype=np.complex128)
    w[:, 0, 0] = 1j * ph[:, 0]
    w[:, 1, 1] = 1j * ph[:, 1]
    w[:, 2, 2] = -1j * (ph[:, 0] + ph[:, 1])
    g = oracle.build_g_exp(w, alpha)
    want = np.zeros_like(g)
    for k in range(3):
        want[:, k, k] = np.exp(alpha / 2 * w[:, k, k])
    assert np.abs(g - want).max() < 1e-15
    for scale in (1e-3, 1.0, 10.0, 200.0):
        w = _random_ah_traceless(rng, 50, scale)
        g = oracle.build_g_exp(w, alpha)
        ref = np.stack([expm(alpha / 2 * m) for m in w])
        # squarings amplify rounding with |A|: both routines carry an error of a few |A| eps
        assert np.abs(g - ref).max() < (2e-14 if scale <= 10 else 2e-13)
        assert np.abs(g @ np.conj(np.swapaxes(g, -1, -2)) - np.eye(3)).max() < 1e-13
        assert np.abs(np.linalg.det(g) - 1).max() < 1e-13


def test_exp_variant_agrees_with_first_order_to_second_order():
    """reunit(1 + A) and exp(A) differ at O(|A|^2): halving alpha divides the difference by 4."""
    rng = np.random.default_rng(6)
    w = _random_ah_traceless(rng, 200, 1.0)
    d = [np.abs(oracle.build_g_exp(w, a) - oracle.build_g(w, a)).max() for a in (0.02, 0.01)]
    assert 3.5 < d[0] / d[1] < 4.5 and d[0] < 0.02


def test_exp_variant_iteration_is_a_gauge_transformation_and_converges():
    """With the exact exponential the update is still a gauge transformation (plaquette), F rises
    monotonically, theta reaches 1e-15, and the linear contraction factor is the same (1 - 16 alpha)^2."""
    n = 4
    U = gen.gen_links(n, 0.4, 21)
    p0 = oracle.plaquette(n, U)
    oracle.set_exponential(True)
    try:
        it, F, th, hist = oracle.fix(n, U, 0.08, 1e-15)
        assert 0 < it < 200 and th <= 1e-15
        assert np.all(np.diff(hist[:, 0]) >= -1e-15)
        assert abs(oracle.plaquette(n, U) - p0) < 1e-12
        eps = 1e-4
        om = np.random.default_rng(3).normal(size=(n ** 4, 8))
        from helpers import GELL_MANN, expm_batch, shift, dag, unit_links
        g0 = expm_batch(1j * eps * np.einsum("xa,aij->xij", om, GELL_MANN) / 2)
        V0 = unit_links(n)
        for mu in range(4):
            V0[:, mu] = g0 @ dag(shift(n, g0, mu, 1))
        h = oracle.iterate(n, V0, 0.08, 1)
        assert abs(h[1, 1] / h[0, 1] - (1 - 16 * 0.08) ** 2) < 1e-3
    finally:
        oracle.set_exponential(False)
    it0 = oracle.fix(n, gen.gen_links(n, 0.4, 21), 0.08, 1e-15)[0]
    assert abs(it - it0) <= 0.25 * it0            # same fixed points, trajectories differ at O(alpha^2)
