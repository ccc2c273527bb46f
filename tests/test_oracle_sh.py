"""Pin T7 (reading S8): the oracle's SH basis is the orthonormal real SH with sign (-1)^m."""
import numpy as np
import scipy.special as sp

from oracle import oracle


def _grid(n_th=64, n_ph=128):
    x, w = np.polynomial.legendre.leggauss(n_th)           # cos(theta) nodes: exact for polynomials
    ph = (np.arange(n_ph) + 0.5) * 2 * np.pi / n_ph
    ct, phg = np.meshgrid(x, ph, indexing="ij")
    st = np.sqrt(1 - ct ** 2)
    d = np.stack([st * np.cos(phg), st * np.sin(phg), ct], -1).reshape(-1, 3)
    wt = (w[:, None] * np.full(n_ph, 2 * np.pi / n_ph)[None]).reshape(-1)
    return d, wt, np.arccos(ct).reshape(-1), phg.reshape(-1)


def test_sh_orthonormal_by_quadrature():
    d, wt, _, _ = _grid()
    Y = np.stack([oracle.sh_basis(3, v) for v in d])
    G = (Y * wt[:, None]).T @ Y
    assert np.abs(G - np.eye(16)).max() < 1e-10


def test_sh_unsoeld_theorem():
    rng = np.random.default_rng(1)
    for _ in range(100):
        v = rng.standard_normal(3); v /= np.linalg.norm(v)
        Y = oracle.sh_basis(3, v)
        for l in range(4):
            assert abs((Y[l * l:(l + 1) ** 2] ** 2).sum() - (2 * l + 1) / (4 * np.pi)) < 1e-12


def test_sh_matches_library_real_harmonics_with_condon_shortley_sign():
    """basis[l^2+l+m] == (-1)^m * (orthonormal real SH Y_lm), the latter built from scipy's complex harmonics."""
    d, _, theta, phi = _grid(12, 16)
    have = np.stack([oracle.sh_basis(3, v) for v in d])
    f = getattr(sp, "sph_harm_y", None)
    for l in range(4):
        for m in range(-l, l + 1):
            am = abs(m)
            Yc = f(l, am, theta, phi) if f is not None else sp.sph_harm(am, l, phi, theta)
            if m == 0:
                real = Yc.real
            elif m > 0:
                real = np.sqrt(2) * (-1) ** m * Yc.real
            else:
                real = np.sqrt(2) * (-1) ** m * Yc.imag
            assert np.abs(have[:, l * l + l + m] - (-1) ** m * real).max() < 1e-12, (l, m)


def test_degree0_colour():
    assert abs(oracle.sh_basis(0, [0, 0, 1])[0] - 1 / (2 * np.sqrt(np.pi))) < 1e-15
    assert np.all(oracle.sh_basis(0, [0, 0, 1])[1:] == 0)
