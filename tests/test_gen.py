"""The seeded input generator (gen/): group properties, determinism, and the statistics the
recipe in DESIGN.md / SURVEY.md 8(d) states.  CPU only."""
import numpy as np

import gen
from helpers import dag, gauge_transform, volume


def test_links_are_SU3_and_deterministic():
    N = (4, 6, 4, 8)
    U = gen.gen_links(N, 0.5, 42)
    assert U.shape == (volume(N), 4, 3, 3)
    assert np.abs(U @ dag(U) - np.eye(3)).max() < 1e-14
    assert np.abs(np.linalg.det(U) - 1).max() < 1e-14
    assert np.array_equal(U, gen.gen_links(N, 0.5, 42))
    assert not np.array_equal(U, gen.gen_links(N, 0.5, 43))


def test_haar_transform_is_the_stated_gauge_transform():
    """U = g0 V g0^dag(x+mu) with V the un-transformed field of the same seed."""
    N = (4, 4, 4, 6)
    V_ = gen.gen_links(N, 0.5, 5, haar=False)
    g0 = gen.gen_haar_field(N, 5)
    assert np.abs(g0 @ dag(g0) - np.eye(3)).max() < 1e-14
    assert np.abs(np.linalg.det(g0) - 1).max() < 1e-14
    assert np.abs(gen.gen_links(N, 0.5, 5) - gauge_transform(N, V_, g0)).max() < 1e-14


def test_roughness_statistics():
    """mean Re Tr V / 3 for sigma = 0.3 / 0.5 / 0.6 (0.941 / 0.842 / 0.778, ~1%)."""
    for sigma, expect in ((0.3, 0.941), (0.5, 0.842), (0.6, 0.778)):
        V_ = gen.gen_links(8, sigma, 1, haar=False)
        m = np.trace(V_, axis1=2, axis2=3).real.mean() / 3
        assert abs(m - expect) < 0.01
    # after the Haar transform the links are uniformly distributed: mean trace ~ 0
    U = gen.gen_links(8, 0.3, 1)
    assert abs(np.trace(U, axis1=2, axis2=3).real.mean()) < 0.02


def test_haar_moments():
    """Haar SU(3): E|g_ij|^2 = 1/3, E g_ij = 0."""
    g = gen.gen_haar_field(8, 3)
    assert np.abs((np.abs(g) ** 2).mean(axis=0) - 1 / 3).max() < 0.02
    assert np.abs(g.mean(axis=0)).max() < 0.03
