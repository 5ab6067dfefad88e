"""P1 — the taper O2 pinned against an independent recipe and printed values."""
import numpy as np

from oracle import taper


def legendre_pswf(x, c, nterms=40):
    """Independent recipe: psi ∝ sum_{k even} beta_k Pbar_k(x),
    Pbar_k = sqrt(k + 1/2) P_k, beta = eigenvector of the smallest eigenvalue of the
    symmetric tridiagonal matrix of the prolate differential operator in that basis."""
    k = 2.0 * np.arange(nterms)
    diag = k * (k + 1) + c * c * (2 * k * (k + 1) - 1) / ((2 * k + 3) * (2 * k - 1))
    off = c * c * (k + 2) * (k + 1) / ((2 * k + 3) * np.sqrt((2 * k + 1) * (2 * k + 5)))
    A = np.diag(diag) + np.diag(off[:-1], 1) + np.diag(off[:-1], -1)
    _, vec = np.linalg.eigh(A)
    beta = vec[:, 0]
    coef = np.zeros(2 * nterms)
    coef[::2] = beta * np.sqrt(k + 0.5)
    val = np.polynomial.legendre.legval(np.asarray(x, float), coef)
    return val / np.polynomial.legendre.legval(0.0, coef)


def test_p1_library_vs_legendre_recipe():
    x = np.linspace(-0.999, 0.999, 801)
    assert np.max(np.abs(taper.psi(x) - legendre_pswf(x, taper.C_PSWF))) <= 1e-13


def test_p1_printed_values(golden):
    for nu, val in golden("p1_taper_values.txt"):
        nu, val = float(nu), float(val)
        if nu < 1.0:
            assert abs(taper.psi(np.array([nu]))[0] - val) <= 1e-13
        # the independent recipe reproduces the printed value, including the limit at 1
        assert abs(legendre_pswf(nu, taper.C_PSWF) - val) <= 1e-13


def test_taper_shape_and_cutoff():
    x = np.linspace(0, 0.999, 200)
    p = taper.psi(x)
    assert p[0] == 1.0
    assert np.all(np.diff(p) < 0)              # monotone decreasing on [0, 1)
    assert np.all(taper.psi(np.array([1.0, -1.0, 1.5, -3.0])) == 0.0)
    assert np.allclose(taper.psi(-x), p)       # even
    assert taper.C_PSWF == 3 * np.pi
    T = taper.taper2d(np.array([0.0, 0.01]), np.array([0.0, 0.02, 0.03]), 0.08)
    assert T.shape == (3, 2) and T[0, 0] == 1.0
    assert np.isclose(T[1, 1], taper.psi(np.array([0.5]))[0] * taper.psi(np.array([0.25]))[0])
