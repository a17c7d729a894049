"""Pins for oracle/sph.py (Cartesian -> real solid harmonics).  CPU only.
Each pin is independent of the recurrences the oracle generates the harmonics with."""
import numpy as np
import pytest

from oracle import sph


def _comps(l):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def test_p18a_cartesian_overlap_by_quadrature():
    """cart_overlap(l) against Gauss-Hermite quadrature of a CONTRACTED shell's Cartesian functions (two primitives):
    the ratio to the (L,0,0) self-overlap does not depend on exponents or coefficients."""
    x, wx = np.polynomial.hermite.hermgauss(40)               # int f(x) e^{-x^2} dx
    expo, coef = np.array([0.8, 2.3]), np.array([0.6, 0.5])
    for l in range(5):
        cs = _comps(l)

        def ov(a, b):
            s = 0.0
            for ei, ci in zip(expo, coef):
                for ej, cj in zip(expo, coef):
                    p = ei + ej
                    m = [np.sum(wx * (x / np.sqrt(p)) ** (a[k] + b[k])) / np.sqrt(p) for k in range(3)]
                    s += ci * cj * m[0] * m[1] * m[2]
            return s
        ref = np.array([[ov(a, b) for b in cs] for a in cs]) / ov((l, 0, 0), (l, 0, 0))
        np.testing.assert_allclose(sph.cart_overlap(l), ref, rtol=1e-12, atol=1e-14)


@pytest.mark.parametrize("l", range(5))
def test_p18b_orthonormal_and_harmonic(l):
    T = sph.shell_transform(l)
    M = sph.cart_overlap(l)
    np.testing.assert_allclose(T.T @ M @ T, np.eye(2 * l + 1), atol=1e-13)
    # every column is a harmonic polynomial: its Laplacian vanishes identically
    cs = _comps(l)
    for c in range(2 * l + 1):
        lap = {}
        for (a, b, d), v in zip(cs, T[:, c]):
            for ax, n in enumerate((a, b, d)):
                if n >= 2:
                    k = [a, b, d]; k[ax] -= 2
                    lap[tuple(k)] = lap.get(tuple(k), 0.0) + n * (n - 1) * v
        assert all(abs(v) < 1e-13 for v in lap.values()), (l, c, lap)


def test_p18c_textbook_forms():
    """p: (y, z, x); d: xy, yz, 2zz-xx-yy, xz, xx-yy, each with a positive factor (order m = -l..l)."""
    T1 = sph.shell_transform(1)                                # Cartesian order x, y, z
    np.testing.assert_allclose(T1, [[0, 0, 1], [1, 0, 0], [0, 1, 0]], atol=1e-15)
    T2 = sph.shell_transform(2)                                # xx, xy, xz, yy, yz, zz
    form = np.array([[0, 1, 0, 0, 0, 0], [0, 0, 0, 0, 1, 0], [-1, 0, 0, -1, 0, 2], [0, 0, 1, 0, 0, 0],
                     [1, 0, 0, -1, 0, 0]], float).T
    for c in range(5):
        f = T2[:, c] @ form[:, c] / (form[:, c] @ form[:, c])
        assert f > 0
        np.testing.assert_allclose(T2[:, c], f * form[:, c], atol=1e-14)
    # normalised d functions: xy carries sqrt(3) relative to the (2,0,0) norm; 2zz-xx-yy the factor 1/2
    assert T2[1, 0] == pytest.approx(np.sqrt(3.0)) and T2[5, 2] == pytest.approx(1.0) and T2[0, 2] == pytest.approx(-0.5)


@pytest.mark.parametrize("l", range(1, 5))
def test_p18d_unsoeld_sum_is_rotation_invariant(l):
    """sum_m S_lm(r)^2 depends on |r| only (Unsoeld): fails if one m has the wrong relative norm or a wrong term."""
    T = sph.shell_transform(l)
    rng = np.random.default_rng(l)
    cs = _comps(l)
    vals = []
    for _ in range(12):
        r = rng.normal(size=3); r /= np.linalg.norm(r)
        v = np.array([r[0] ** a * r[1] ** b * r[2] ** c for (a, b, c) in cs])
        vals.append(float(np.sum((T.T @ v) ** 2)))
    np.testing.assert_allclose(vals, vals[0], rtol=1e-12)


def test_p18e_block_structure():
    T = sph.transform_matrix([0, 2, 1, 3])
    assert T.shape == (1 + 6 + 3 + 10, 1 + 5 + 3 + 7)
    assert T[0, 0] == 1.0 and not T[0, 1:].any() and not T[1:7, 6:].any()
    M = np.arange(400, dtype=float).reshape(20, 20)
    np.testing.assert_allclose(sph.cart_to_spherical([0, 2, 1, 3], M), T.T @ M @ T)
