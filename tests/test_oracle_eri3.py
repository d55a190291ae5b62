"""Pins for the oracle integrals (Appendix A eqs. 12-19; SURVEY.md §8(c) pins).

Each pin is chosen so that a plausible mistake (dropped term, wrong sign/index, transposed operand) fails it.
"""
import itertools
import os

import numpy as np
import pytest

import lx_inputs as gen
from helpers import bruteforce_primitive, comp_index, table

HERE = os.path.dirname(os.path.abspath(__file__))
A = np.array([0.3, -0.7, 1.1])
B = np.array([-1.2, 0.4, 0.2])
C = np.array([0.9, 1.3, -0.8])
ZA, ZB, ZC = 1.3, 0.45, 0.8


def _prim_val(oracle, c, a, b, Cc=C, Aa=A, Bb=B, zc=ZC, za=ZA, zb=ZB):
    lx, la, lb = sum(c), sum(a), sum(b)
    aux = table([(lx, Cc, [zc], [1.0])])
    prim = table([(la, Aa, [za], [1.0]), (lb, Bb, [zb], [1.0])])
    o = oracle.eri3_batch(lx, la, lb, aux, prim, [0], [[0, 1]])
    return o[0, 0, comp_index(lx, c), comp_index(la, a), comp_index(lb, b)]


def _set(oracle, lx, la, lb, Cc=C, Aa=A, Bb=B, zc=(ZC,), za=(ZA,), zb=(ZB,), cc=None, ca=None, cb=None):
    aux = table([(lx, Cc, list(zc), cc if cc is not None else [1.0] * len(zc))])
    prim = table([(la, Aa, list(za), ca if ca is not None else [1.0] * len(za)),
                  (lb, Bb, list(zb), cb if cb is not None else [1.0] * len(zb))])
    return oracle.eri3_batch(lx, la, lb, aux, prim, [0], [[0, 1]])[0, 0]


def test_worked_example_golden(oracle):
    rows = [l.split() for l in open(os.path.join(HERE, "golden", "worked_example_primitives.txt")) if not l.startswith("#")]
    assert len(rows) == 10
    for r in rows:
        c, a, b = tuple(map(int, r[0:3])), tuple(map(int, r[3:6])), tuple(map(int, r[6:9]))
        ex = float(r[9])
        assert abs(_prim_val(oracle, c, a, b) - ex) < 2e-15 * max(1.0, abs(ex)), (c, a, b)


def test_sss_closed_form(oracle):
    """(s|ss) = 2 pi^{5/2}/(p q sqrt(p+q)) exp(-mu|AB|^2) F_0(rho|PC|^2), F_0 = sqrt(pi/T) erf(sqrt T)/2 (eq. 4, m=0)."""
    from scipy import special
    rng = np.random.default_rng(5)
    for _ in range(20):
        a, b, c = rng.uniform(-2, 2, 3), rng.uniform(-2, 2, 3), rng.uniform(-3, 3, 3)
        za, zb, zc = np.exp(rng.uniform(np.log(0.1), np.log(10), 3))
        p = za + zb
        P = (za * a + zb * b) / p
        T = p * zc / (p + zc) * np.sum((P - c) ** 2)
        F0 = 0.5 * np.sqrt(np.pi / T) * special.erf(np.sqrt(T))
        ex = 2 * np.pi ** 2.5 / (p * zc * np.sqrt(p + zc)) * np.exp(-za * zb / p * np.sum((a - b) ** 2)) * F0
        got = _prim_val(oracle, (0, 0, 0), (0, 0, 0), (0, 0, 0), c, a, b, zc, za, zb)
        assert abs(got - ex) < 1e-14 * abs(ex)


@pytest.mark.parametrize("c,a,b", [((0, 0, 0), (0, 0, 0), (0, 0, 0)), ((0, 1, 0), (0, 0, 0), (0, 0, 0)),
                                   ((0, 0, 1), (0, 0, 0), (1, 0, 0)), ((1, 0, 1), (0, 2, 0), (0, 0, 1)),
                                   ((1, 1, 0), (1, 0, 1), (0, 1, 0)), ((0, 3, 0), (1, 1, 0), (0, 1, 1))])
def test_bruteforce_quadrature(oracle, c, a, b):
    """Independent of Boys and of the E/R recursions (helpers.bruteforce_primitive)."""
    ex = bruteforce_primitive(c, a, b, C, A, B, ZC, ZA, ZB)
    got = _prim_val(oracle, c, a, b)
    assert abs(got - ex) < 5e-13 * max(abs(ex), 1e-3)


def test_bruteforce_second_geometry(oracle):
    A2, B2, C2 = np.array([0.0, 0.1, -0.4]), np.array([0.5, -0.3, 0.2]), np.array([-0.2, 0.6, 0.1])
    for c, a, b in [((2, 0, 0), (0, 1, 1), (1, 0, 0)), ((0, 1, 1), (2, 0, 0), (0, 0, 2))]:
        ex = bruteforce_primitive(c, a, b, C2, A2, B2, 2.1, 0.7, 3.3)
        got = _prim_val(oracle, c, a, b, C2, A2, B2, 2.1, 0.7, 3.3)
        assert abs(got - ex) < 5e-13 * max(abs(ex), 1e-3)


def test_hrr_identity_contracted(oracle):
    """(X|a b+1_i) = (X|a+1_i b) + AB_i (X|ab)   (eq. 1) on contracted shells."""
    za, zb, zc = [1.3, 0.4, 3.0], [0.45, 2.2], [0.8, 0.3]
    ca, cb, cc = [0.7, 0.5, 0.2], [1.1, 0.3], [0.9, 0.6]
    AB = A - B
    for lx, la, lb in [(0, 0, 0), (1, 1, 0), (2, 1, 1), (3, 2, 1), (2, 2, 2)]:
        base = _set(oracle, lx, la, lb, zc=zc, za=za, zb=zb, cc=cc, ca=ca, cb=cb)
        up_b = _set(oracle, lx, la, lb + 1, zc=zc, za=za, zb=zb, cc=cc, ca=ca, cb=cb)
        up_a = _set(oracle, lx, la + 1, lb, zc=zc, za=za, zb=zb, cc=cc, ca=ca, cb=cb)
        scale = np.max(np.abs(up_b))
        for ia, a in enumerate(gen_components(la)):
            for ib, b in enumerate(gen_components(lb)):
                for i in range(3):
                    bp = list(b); bp[i] += 1
                    ap = list(a); ap[i] += 1
                    lhs = up_b[:, ia, comp_index(lb + 1, bp)]
                    rhs = up_a[:, comp_index(la + 1, ap), ib] + AB[i] * base[:, ia, ib]
                    assert np.max(np.abs(lhs - rhs)) < 1e-14 * scale


def gen_components(l):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def test_translational_sum_rule(oracle):
    """2 zc [c+1_i|ab] - c_i [c-1_i|ab] + 2 za [c|a+1_i b] - a_i [c|a-1_i b] + 2 zb [c|a b+1_i] - b_i [c|a b-1_i] = 0
    per primitive triple (SURVEY.md §8(c) pins): couples all three indices and all three exponents."""
    def v(c, a, b):
        if min(c) < 0 or min(a) < 0 or min(b) < 0:
            return 0.0
        return _prim_val(oracle, tuple(c), tuple(a), tuple(b))
    for c, a, b in [((0, 0, 0), (0, 0, 0), (0, 0, 0)), ((1, 0, 1), (0, 1, 0), (1, 0, 0)), ((2, 1, 0), (1, 1, 0), (0, 0, 2)),
                    ((0, 2, 2), (2, 0, 0), (1, 1, 0))]:
        for i in range(3):
            e = np.eye(3, dtype=int)[i]
            terms = [2 * ZC * v(np.add(c, e), a, b), -c[i] * v(np.subtract(c, e), a, b),
                     2 * ZA * v(c, np.add(a, e), b), -a[i] * v(c, np.subtract(a, e), b),
                     2 * ZB * v(c, a, np.add(b, e)), -b[i] * v(c, a, np.subtract(b, e))]
            assert abs(sum(terms)) < 2e-15 * max(1.0, max(abs(t) for t in terms))


def test_bra_swap_symmetry(oracle):
    """(X|ab) = (X|ba) with the shells swapped: transpose of the last two indices."""
    za, zb, zc = [1.3, 0.4], [0.45], [0.8, 2.0]
    for lx, la, lb in [(1, 2, 0), (2, 1, 2), (3, 2, 1), (4, 0, 2)]:
        x = _set(oracle, lx, la, lb, za=za, zb=zb, zc=zc)
        y = _set(oracle, lx, lb, la, Aa=B, Bb=A, za=zb, zb=za, zc=zc)
        assert np.max(np.abs(x - np.swapaxes(y, 1, 2))) < 1e-15 * np.max(np.abs(x))


def test_translation_invariance(oracle):
    t = np.array([3.7, -11.2, 5.9])
    for lx, la, lb in [(2, 1, 1), (3, 2, 2)]:
        x = _set(oracle, lx, la, lb)
        y = _set(oracle, lx, la, lb, Cc=C + t, Aa=A + t, Bb=B + t)
        assert np.max(np.abs(x - y)) < 5e-14 * np.max(np.abs(x))


def test_axis_permutation_and_reflection(oracle):
    """Permuting / reflecting the axes of all centres permutes / sign-flips components exactly."""
    lx, la, lb = 3, 2, 1
    x = _set(oracle, lx, la, lb)
    perm = [2, 0, 1]                                  # new axis k holds old axis perm[k]
    y = _set(oracle, lx, la, lb, Cc=C[perm], Aa=A[perm], Bb=B[perm])
    for (ic, c), (ia, a), (ib, b) in itertools.product(enumerate(gen_components(lx)), enumerate(gen_components(la)),
                                                       enumerate(gen_components(lb))):
        cp, ap, bp = [c[k] for k in perm], [a[k] for k in perm], [b[k] for k in perm]
        assert abs(y[comp_index(lx, cp), comp_index(la, ap), comp_index(lb, bp)] - x[ic, ia, ib]) < 1e-15
    s = np.array([1.0, -1.0, 1.0])
    z = _set(oracle, lx, la, lb, Cc=C * s, Aa=A * s, Bb=B * s)
    for (ic, c), (ia, a), (ib, b) in itertools.product(enumerate(gen_components(lx)), enumerate(gen_components(la)),
                                                       enumerate(gen_components(lb))):
        assert abs(z[ic, ia, ib] - (-1) ** (c[1] + a[1] + b[1]) * x[ic, ia, ib]) < 1e-15


def test_far_field_limit(oracle):
    """|PC| -> inf: (s|ss) -> (pi/p)^{3/2} (pi/q)^{3/2} exp(-mu|AB|^2)/|PC|; (p_z|ss) -> that * d/dC_z-type decay."""
    Cf = np.array([0.0, 0.0, 200.0])
    p = ZA + ZB
    P = (ZA * A + ZB * B) / p
    R = np.linalg.norm(P - Cf)
    ex = (np.pi / p) ** 1.5 * (np.pi / ZC) ** 1.5 * np.exp(-ZA * ZB / p * np.sum((A - B) ** 2)) / R
    got = _prim_val(oracle, (0, 0, 0), (0, 0, 0), (0, 0, 0), Cc=Cf)
    assert abs(got - ex) < 1e-14 * ex
    # dipole of a p function on C: charge moment int z^2 e^{-q r^2} = (pi/q)^{3/2}/(2q); field of the bra charge
    q_bra = (np.pi / p) ** 1.5 * np.exp(-ZA * ZB / p * np.sum((A - B) ** 2))
    mom = (np.pi / ZC) ** 1.5 / (2 * ZC)
    ex_p = q_bra * mom * (P - Cf)[2] / R ** 3
    got_p = _prim_val(oracle, (0, 0, 1), (0, 0, 0), (0, 0, 0), Cc=Cf)
    assert abs(got_p - ex_p) < 1e-13 * abs(ex_p)


def test_degenerate_geometries(oracle):
    """A = B, P = C (T = 0), all centres equal (reading G15): finite, symmetric, and equal to the quadrature."""
    z = np.zeros(3)
    v = _prim_val(oracle, (0, 0, 0), (0, 0, 0), (0, 0, 0), Cc=z, Aa=z, Bb=z)
    p = ZA + ZB
    assert abs(v - 2 * np.pi ** 2.5 / (p * ZC * np.sqrt(p + ZC))) < 1e-15 * v      # F_0(0) = 1
    # odd total power on an axis vanishes when everything is concentric
    assert abs(_prim_val(oracle, (1, 0, 0), (0, 0, 0), (0, 0, 0), Cc=z, Aa=z, Bb=z)) < 1e-17
    ex = bruteforce_primitive((2, 0, 0), (1, 0, 0), (1, 0, 0), z, z, z, ZC, ZA, ZB)
    assert abs(_prim_val(oracle, (2, 0, 0), (1, 0, 0), (1, 0, 0), Cc=z, Aa=z, Bb=z) - ex) < 1e-13 * abs(ex)
    ex = bruteforce_primitive((1, 0, 0), (1, 0, 0), (0, 0, 0), C, A, A, ZC, ZA, ZB)   # A = B
    assert abs(_prim_val(oracle, (1, 0, 0), (1, 0, 0), (0, 0, 0), Bb=A) - ex) < 1e-13 * abs(ex)


def test_contraction_is_linear(oracle):
    """(X|ab) = sum_kij c_k c_i c_j [..]_kij: contracted set = weighted sum of primitive sets."""
    za, zb, zc = [1.3, 0.4, 3.0], [0.45, 2.2], [0.8, 0.3]
    ca, cb, cc = [0.7, -0.5, 0.2], [1.1, 0.3], [0.9, 0.6]
    full = _set(oracle, 2, 2, 1, zc=zc, za=za, zb=zb, cc=cc, ca=ca, cb=cb)
    acc = 0.0
    for k, i, j in itertools.product(range(2), range(3), range(2)):
        acc = acc + cc[k] * ca[i] * cb[j] * _set(oracle, 2, 2, 1, zc=[zc[k]], za=[za[i]], zb=[zb[j]])
    assert np.max(np.abs(full - acc)) < 1e-15 * np.max(np.abs(full))


def test_double_instantiation_close(oracle):
    cfg = gen.config1(npair=8, nx=4)
    a = oracle.eri3_batch(2, 1, 1, cfg["aux"], cfg["prim"], cfg["x_idx"], cfg["pair_idx"], real="ld")
    b = oracle.eri3_batch(2, 1, 1, cfg["aux"], cfg["prim"], cfg["x_idx"], cfg["pair_idx"], real="d")
    assert np.max(np.abs(a - b)) < 1e-13 * np.max(np.abs(a))
    assert a.shape == (8, 4, 6, 3, 3)


def test_batch_rejects_wrong_class(oracle):
    cfg = gen.config1(npair=2, nx=2)
    with pytest.raises(ValueError):
        oracle.eri3_batch(1, 1, 1, cfg["aux"], cfg["prim"], cfg["x_idx"], cfg["pair_idx"])
