"""numpy helpers for the tests: special fields and independent re-derivations.

Nothing here is imported by the oracle or by the CUDA package.  Shapes follow the
interchange layout: links [V,4,3,3], site fields [V,3,3], s = ix + Nx*(iy + Ny*(iz + Nz*it)).
A field reshaped to N[::-1] + (...) is indexed [it, iz, iy, ix, ...], so lattice axis mu is
numpy axis 3 - mu.
"""
import numpy as np


def dims(N):
    return (N,) * 4 if isinstance(N, int) else tuple(N)


def volume(N):
    N = dims(N)
    return N[0] * N[1] * N[2] * N[3]


def lat(N, f):
    """[V, ...] -> [Nt, Nz, Ny, Nx, ...]"""
    N = dims(N)
    return f.reshape(N[::-1] + f.shape[1:])


def shift(N, f, mu, d):
    """Field evaluated at x + d*mu_hat: returns h with h(x) = f(x + d mu_hat)."""
    return np.roll(lat(N, f), -d, axis=3 - mu).reshape(f.shape)


def dag(m):
    return np.conj(np.swapaxes(m, -1, -2))


GELL_MANN = np.zeros((8, 3, 3), dtype=np.complex128)
GELL_MANN[0][0, 1] = GELL_MANN[0][1, 0] = 1
GELL_MANN[1][0, 1] = -1j
GELL_MANN[1][1, 0] = 1j
GELL_MANN[2][0, 0] = 1
GELL_MANN[2][1, 1] = -1
GELL_MANN[3][0, 2] = GELL_MANN[3][2, 0] = 1
GELL_MANN[4][0, 2] = -1j
GELL_MANN[4][2, 0] = 1j
GELL_MANN[5][1, 2] = GELL_MANN[5][2, 1] = 1
GELL_MANN[6][1, 2] = -1j
GELL_MANN[6][2, 1] = 1j
GELL_MANN[7] = np.diag([1, 1, -2]) / np.sqrt(3)


def expm_batch(a):
    """exp of a batch of 3x3 matrices [..., 3, 3]: scaling and squaring + Taylor."""
    nrm = np.abs(a).sum(axis=(-1, -2)).max()
    sq = 0
    while nrm > 0.125:
        nrm *= 0.5
        sq += 1
    a = a / 2.0 ** sq
    e = np.broadcast_to(np.eye(3, dtype=np.complex128), a.shape).copy()
    term = e.copy()
    for n in range(1, 20):
        term = term @ a / n
        e = e + term
    for _ in range(sq):
        e = e @ e
    return e


def unit_links(N):
    U = np.zeros((volume(N), 4, 3, 3), dtype=np.complex128)
    U[..., 0, 0] = U[..., 1, 1] = U[..., 2, 2] = 1
    return U


def gauge_transform(N, U, g):
    """U_mu(x) -> g(x) U_mu(x) g(x+mu)^dagger, written with np.roll."""
    out = np.empty_like(U)
    for mu in range(4):
        out[:, mu] = g @ U[:, mu] @ dag(shift(N, g, mu, +1))
    return np.ascontiguousarray(out)


def random_su3_algebra(rng, shape, scale=1.0):
    """i * sum_a omega^a lambda_a / 2 with omega ~ N(0, scale^2): anti-Hermitian traceless."""
    om = rng.normal(0.0, scale, size=shape + (8,))
    return 1j * np.einsum("...a,aij->...ij", om, GELL_MANN) / 2, om


def dft4d_bruteforce(N, f, sign):
    """O(V^2) 4D DFT straight from the definition: F(k) = sum_x f(x) exp(sign 2 pi i sum_mu k_mu x_mu / N_mu)."""
    N = dims(N)
    V = volume(N)
    idx = np.arange(V)
    c = []
    for d in range(4):
        c.append(idx % N[d])
        idx = idx // N[d]
    phase = np.zeros((V, V))
    for d in range(4):
        phase += np.outer(c[d], c[d]) / N[d]
    return np.exp(sign * 2j * np.pi * phase) @ f
