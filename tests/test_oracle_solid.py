"""Pins of the oracle's real solid harmonics (oracle/solid.py; SURVEY.md §8(a) row a6, §8(c) "pure-X variant"):
harmonicity, the textbook forms for l <= 2, and orthonormality on the unit sphere in Racah normalisation
(int S_lm S_lm' dOmega = 4 pi / (2l+1) delta_mm')."""
import numpy as np
import pytest

from oracle import solid


def _poly(l, row):
    """dict monomial -> coefficient of one solid harmonic."""
    return {c: row[i] for i, c in enumerate(solid.components(l)) if row[i] != 0.0}


@pytest.mark.parametrize("l", range(7))
def test_harmonic(l):
    """Laplacian of every S_lm vanishes identically (a dropped or mis-signed term breaks it)."""
    S = solid.solid_matrix(l)
    for m in range(2 * l + 1):
        lap = {}
        for (x, y, z), v in _poly(l, S[m]).items():
            for ax, p in enumerate((x, y, z)):
                if p >= 2:
                    q = [x, y, z]
                    q[ax] -= 2
                    lap[tuple(q)] = lap.get(tuple(q), 0.0) + v * p * (p - 1)
        assert all(abs(v) < 1e-12 for v in lap.values()), (l, m - l, lap)


def test_low_l_closed_forms():
    s3 = np.sqrt(3.0)
    assert np.allclose(solid.solid_matrix(0), [[1.0]])
    # l = 1: m = -1, 0, 1 -> y, z, x  (components x, y, z)
    assert np.allclose(solid.solid_matrix(1), [[0, 1, 0], [0, 0, 1], [1, 0, 0]])
    # l = 2, components xx xy xz yy yz zz: m = -2..2 -> sqrt3 xy, sqrt3 yz, zz - xx/2 - yy/2, sqrt3 xz, sqrt3/2 (xx - yy)
    want = [[0, s3, 0, 0, 0, 0], [0, 0, 0, 0, s3, 0], [-0.5, 0, 0, -0.5, 0, 1.0], [0, 0, s3, 0, 0, 0], [s3 / 2, 0, 0, -s3 / 2, 0, 0]]
    assert np.allclose(solid.solid_matrix(2), want)


@pytest.mark.parametrize("l", range(1, 7))
def test_orthonormal_on_sphere(l):
    nt, nph = 48, 96
    ct, wt = np.polynomial.legendre.leggauss(nt)
    ph = (np.arange(nph) + 0.5) * 2 * np.pi / nph
    st = np.sqrt(1 - ct ** 2)
    X = np.outer(st, np.cos(ph)).ravel()
    Y = np.outer(st, np.sin(ph)).ravel()
    Z = np.outer(ct, np.ones(nph)).ravel()
    W = np.outer(wt, np.full(nph, 2 * np.pi / nph)).ravel()
    mono = np.stack([X ** a * Y ** b * Z ** c for (a, b, c) in solid.components(l)])
    vals = solid.solid_matrix(l) @ mono
    G = (vals * W) @ vals.T
    assert np.allclose(G, 4 * np.pi / (2 * l + 1) * np.eye(2 * l + 1), atol=1e-10)
