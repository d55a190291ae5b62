"""The chain form of the ket recurrence (lx_chain.cuh header) checked against the oracle on the CPU.

A plain Python restatement of the identity the team / chain kernels evaluate,

    [a0|c]^(0) = sum_{n <= c/2} beta(c,n) (2 zc)^-|n| ( prod_i B_i^(c_i - 2 n_i)  Y_|n| )[a],
    Y_p = Delta^p Z^(Lx-2p),  (Delta Z)^(m) = Z^(m) - (rho/zc) Z^(m+1),  Z^(m)[a] = [a0|0]^(m)  (eq. 3),

in the basis u[a] = f[a]/a! where one step is u[a] <- r_i u[a] + u[a-1_i], r_i = 2 gamma PC_i.  It shares no code with
the CUDA path; it pins the derivation (the resummation of the c-1 terms that eq. 2, drops) to the
McMurchie-Davidson oracle for uncontracted primitives."""
import itertools
import math

import numpy as np
import pytest
from scipy.special import hyp1f1

from helpers import table


def comps(l):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def boys(m, T):
    return hyp1f1(m + 0.5, m + 1.5, -T) / (2 * m + 1)


def fact3(a):
    return math.factorial(a[0]) * math.factorial(a[1]) * math.factorial(a[2])


def chain_eval(E, LX, A, B, Cc, za, zb, zc):
    A, B, Cc = map(np.asarray, (A, B, Cc))
    g = za + zb
    P = (za * A + zb * B) / g
    rho = g * zc / (g + zc)
    PA, PC = P - A, P - Cc
    T = rho * PC @ PC
    L = E + LX
    pref = 2 * math.pi ** 2.5 / (g * zc * math.sqrt(g + zc)) * math.exp(-za * zb / g * ((A - B) @ (A - B)))
    Z = {(m, (0, 0, 0)): pref * boys(m, T) for m in range(L + 1)}           # eq. 4
    WP = -(rho / g) * PC
    for e in range(1, E + 1):                                               # eq. 3 (VRR1)
        for a in comps(e):
            i = min((d for d in range(3) if a[d] > 0), key=lambda d: a[d])
            a1 = tuple(a[d] - (d == i) for d in range(3))
            for m in range(L - e + 1):
                v = PA[i] * Z[(m, a1)] + WP[i] * Z[(m + 1, a1)]
                if a1[i] > 0:
                    a2 = tuple(a1[d] - (d == i) for d in range(3))
                    v += a1[i] / (2 * g) * (Z[(m, a2)] - rho / g * Z[(m + 1, a2)])
                Z[(m, a)] = v
    allA = [a for e in range(E + 1) for a in comps(e)]
    cs, r = 1 / (2 * (g + zc)), 2 * g * PC
    out = {}
    for c in comps(LX):
        for a in allA:
            out[(c, a)] = 0.0
        for n in itertools.product(*[range(ci // 2 + 1) for ci in c]):
            t = tuple(ci - 2 * ni for ci, ni in zip(c, n))
            p, k = sum(n), sum(t)
            beta = 1.0
            for ci, ni in zip(c, n):
                beta *= math.factorial(ci) / (math.factorial(ni) * math.factorial(ci - 2 * ni) * 2 ** ni)
            u = {a: sum(math.comb(p, s) * (-rho / zc) ** s * Z[(k + s, a)] for s in range(p + 1)) / fact3(a) for a in allA}
            for i in range(3):
                for _ in range(t[i]):
                    u = {a: r[i] * u[a] + (u[tuple(a[d] - (d == i) for d in range(3))] if a[i] > 0 else 0.0) for a in allA}
            for a in allA:
                out[(c, a)] += beta * (2 * zc) ** (-p) * cs ** k * u[a] * fact3(a)
    return out


@pytest.mark.parametrize("E,LX", [(0, 2), (1, 1), (2, 2), (2, 3), (3, 4), (4, 4), (4, 3), (2, 5), (1, 6)])
def test_chain_form_equals_oracle(oracle, E, LX):
    rng = np.random.default_rng(100 * E + LX)
    A, B, Cc = rng.uniform(-1, 1, 3), rng.uniform(-1, 1, 3), rng.uniform(-1, 1, 3)
    za, zb, zc = rng.uniform(0.3, 2, 3)
    out = chain_eval(E, LX, A, B, Cc, za, zb, zc)
    worst, scale = 0.0, 0.0
    for e in range(E + 1):
        prim = table([(e, A, [za], [1.0]), (0, B, [zb], [1.0])])
        aux = table([(LX, Cc, [zc], [1.0])])
        ref = oracle.eri3_batch(LX, e, 0, aux, prim, [0], [[0, 1]])[0, 0, :, :, 0]
        for ic, c in enumerate(comps(LX)):
            for ia, a in enumerate(comps(e)):
                worst = max(worst, abs(out[(c, a)] - ref[ic, ia]))
                scale = max(scale, abs(ref[ic, ia]))
    assert worst <= 1e-13 * scale, (worst, scale)


def test_closed_n_quantal_form_g5_g6():
    """Reading G5/G6: the corrected closed form of the paper's eq. 8,
        (B^t z)[a] = sum_{u <= min(a,t)} prod_i C(t_i,u_i) C(a_i,u_i) u_i!  w^(t-u) c^|u| z[a-u],
    is the expansion of the chain operator B_i = w_i + c S_i, and its integer coefficients for a = t = (2,0,0) are the
    1, 4, 2 of the worked example eq. 9 (the printed last coefficient 1 is a typo: tests/golden/cvrr2_example.txt)."""
    import os
    rng = np.random.default_rng(8)
    E, LX = 4, 4
    allA = [a for e in range(E + 1) for a in comps(e)]
    z = {a: rng.normal() for a in allA}
    w, cs = rng.normal(size=3), 0.37
    for t in comps(LX) + comps(2) + comps(3):
        # stepping: f <- w_i f[a] + c a_i f[a - 1_i]
        f = dict(z)
        for i in range(3):
            for _ in range(t[i]):
                f = {a: w[i] * f[a] + (cs * a[i] * f[tuple(a[d] - (d == i) for d in range(3))] if a[i] > 0 else 0.0) for a in allA}
        for a in allA:
            closed = 0.0
            for u in itertools.product(*[range(min(a[i], t[i]) + 1) for i in range(3)]):
                coef = 1
                for i in range(3):
                    coef *= math.comb(t[i], u[i]) * math.comb(a[i], u[i]) * math.factorial(u[i])
                closed += coef * np.prod([w[i] ** (t[i] - u[i]) for i in range(3)]) * cs ** sum(u) * z[tuple(a[i] - u[i] for i in range(3))]
            assert abs(closed - f[a]) <= 1e-12 * max(1.0, abs(f[a])), (t, a)
    gold = [tuple(int(v) for v in ln.split()) for ln in open(os.path.join(os.path.dirname(__file__), "golden", "cvrr2_example.txt"))
            if ln.strip() and not ln.startswith("#")]
    assert gold == [(u, math.comb(2, u) ** 2 * math.factorial(u)) for u in range(3)] == [(0, 1), (1, 4), (2, 2)]
