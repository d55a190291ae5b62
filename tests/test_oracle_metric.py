"""Pins for the oracle's two-centre metric V_XY = (X|Y) and fit solve."""
import numpy as np
from scipy.special import erf

import lx_inputs as gen
from helpers import table


def _f0(T):
    return 1.0 if T < 1e-14 else 0.5 * np.sqrt(np.pi / T) * erf(np.sqrt(T))


def _ss(q1, q2, R):
    """[s|s](R) = 2 pi^{5/2} / (q1 q2 sqrt(q1+q2)) F_0(q1 q2/(q1+q2) R^2) for unnormalised s primitives."""
    return 2 * np.pi ** 2.5 / (q1 * q2 * np.sqrt(q1 + q2)) * _f0(q1 * q2 / (q1 + q2) * float(np.dot(R, R)))


def test_metric_ss_closed_form(oracle):
    A, B = np.array([0.1, -0.4, 0.25]), np.array([1.3, 0.6, -0.7])
    aux = table([(0, A, [0.9], [1.0]), (0, B, [0.35, 2.2], [0.7, 0.4])])
    V = oracle.metric_2c(aux)
    ex01 = 0.7 * _ss(0.9, 0.35, A - B) + 0.4 * _ss(0.9, 2.2, A - B)
    ex11 = sum(c1 * c2 * _ss(q1, q2, np.zeros(3)) for q1, c1 in zip([0.35, 2.2], [0.7, 0.4])
               for q2, c2 in zip([0.35, 2.2], [0.7, 0.4]))
    assert abs(V[0, 1] - ex01) < 1e-14 * ex01 and abs(V[1, 0] - ex01) < 1e-14 * ex01
    assert abs(V[0, 0] - _ss(0.9, 0.9, np.zeros(3))) < 1e-14 * V[0, 0]
    assert abs(V[1, 1] - ex11) < 1e-14 * ex11


def test_metric_ps_and_pp_by_centre_derivatives(oracle):
    """p_i = (1/2q) d/dA_i of the s primitive, so (p_i|s) and (p_i|p_j) are centre derivatives of the closed form
    [s|s](A−B); taken by central differences of step h (error O(h^2) relative 1e-7 at h = 1e-3)."""
    A, B, q1, q2, h = np.array([0.2, 0.1, -0.3]), np.array([-0.6, 0.9, 0.5]), 0.8, 1.7, 1e-3
    aux = table([(1, A, [q1], [1.0]), (0, B, [q2], [1.0]), (1, B, [q2], [1.0])])
    V = oracle.metric_2c(aux)                      # bf: p(A) 0..2, s(B) 3, p(B) 4..6; component order x, y, z
    e = np.eye(3)
    for i in range(3):
        d1 = (_ss(q1, q2, A + h * e[i] - B) - _ss(q1, q2, A - h * e[i] - B)) / (2 * h) / (2 * q1)
        assert abs(V[i, 3] - d1) < 1e-6 * abs(d1), (i, V[i, 3], d1)
        assert abs(V[3, i] - V[i, 3]) < 1e-15
        for j in range(3):
            f = lambda sa, sb: _ss(q1, q2, A + sa * h * e[i] - B - sb * h * e[j])
            d2 = (f(1, 1) - f(1, -1) - f(-1, 1) + f(-1, -1)) / (4 * h * h) / (4 * q1 * q2)
            assert abs(V[i, 4 + j] - d2) < 2e-6 * max(abs(d2), 1e-3), (i, j, V[i, 4 + j], d2)


def test_metric_symmetric_diagonal_and_definite(oracle):
    """V = V^T although (X|Y 1) and (Y|X 1) take different routes through the 3-centre routine (X on the Hermite side
    of one electron, Y on the product side of the other); diagonal blocks reproduce the separate Schwarz routine;
    V is positive definite (a Coulomb metric of linearly independent functions)."""
    rng = np.random.default_rng(11)
    xs = []
    for l in range(7):
        k = 1 + l % 2
        z = np.exp(rng.uniform(np.log(0.2), np.log(5.0), k))
        xs.append((l, rng.uniform(0, 2.5, 3), z, rng.uniform(0.3, 1.0, k) * gen.prim_norm(z, l)))
    aux = table(xs)
    V = oracle.metric_2c(aux)
    assert np.max(np.abs(V - V.T)) <= 1e-14 * np.max(np.abs(V))
    q = oracle.schwarz_aux(aux)
    for x in range(aux.nshell):
        blk = np.diag(V[aux.bf_off[x]:aux.bf_off[x + 1], aux.bf_off[x]:aux.bf_off[x + 1]])
        assert abs(np.sqrt(blk.max()) - q[x]) <= 1e-13 * q[x]
    # Cartesian shells with l >= 2 hold the lower-l contaminants (x²+y²+z² is an s function), still independent here
    small = table(xs[:4])
    w = np.linalg.eigvalsh(oracle.metric_2c(small))
    assert w.min() > 0


def test_fit_solve_residual_and_identity(oracle):
    rng = np.random.default_rng(3)
    prim, aux = gen._cluster(rng, 3, 5.0, gen._PRIM4, gen._AUX4[:3])
    V = oracle.metric_2c(aux)
    g = rng.normal(size=aux.nbf)
    d = oracle.fit_solve(V, g)
    assert np.max(np.abs(V @ d - g)) <= 1e-9 * np.max(np.abs(g)) * np.linalg.cond(V) * 1e-4 + 1e-10
    assert np.allclose(oracle.fit_solve(np.eye(5) * 2.0, np.arange(5.0)), np.arange(5.0) / 2.0, rtol=0, atol=1e-15)
