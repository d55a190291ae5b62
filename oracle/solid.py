"""ORACLE — test infrastructure only.  Real solid harmonics and the Cartesian -> solid-harmonic transform of the
auxiliary index (HGPA step 5; reading G1: "pure X = Cartesian result x the
real-solid-harmonic matrix").

Plain restatement of the closed formula of the real solid harmonics (Helgaker, Jorgensen, Olsen, "Molecular
Electronic-Structure Theory", eq. 6.4.47), Racah normalisation (S_l0 = r^l P_l(cos theta), e.g. S_20 = z^2 - x^2/2 - y^2/2):

    S_lm = N_lm  sum_{t=0}^{[(l-|m|)/2]} sum_{u=0}^{t} sum_{v}  C^{lm}_{tuv}  x^{2t+|m|-2(u+v)} y^{2(u+v)} z^{l-2t-|m|}
    C^{lm}_{tuv} = (-1)^{t+v-v_m} (1/4)^t binom(l,t) binom(l-t,|m|+t) binom(t,u) binom(|m|,2v)
    N_lm = 1/(2^|m| l!) sqrt( 2 (l+|m|)! (l-|m|)! / 2^{delta_m0} ),   v = v_m, v_m+1, ..., [|m|/2 - v_m] + v_m,
    v_m = 0 for m >= 0 and 1/2 for m < 0.

Components are ordered m = -l, ..., 0, ..., +l; Cartesian components in ABI order (reading G2).  Pinned by
tests/test_oracle_solid.py (harmonicity, low-l closed forms, orthogonality on the sphere).  Shares nothing with the
CUDA path, which builds its own matrix by the recurrences of the regular solid harmonics.
"""
from fractions import Fraction
from math import comb, factorial, sqrt

import numpy as np


def components(l):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def solid_matrix(l):
    """S[m + l, c]: coefficient of the Cartesian monomial c (ABI order) in S_lm; shape (2l+1, (l+1)(l+2)/2)."""
    comps = components(l)
    index = {c: i for i, c in enumerate(comps)}
    S = np.zeros((2 * l + 1, len(comps)))
    for m in range(-l, l + 1):
        am = abs(m)
        norm = sqrt(2.0 * factorial(l + am) * factorial(l - am) / (2.0 if m == 0 else 1.0)) / (2 ** am * factorial(l))
        two_vm = 0 if m >= 0 else 1                      # 2 v_m
        for t in range((l - am) // 2 + 1):
            for u in range(t + 1):
                # v = v_m + k, k = 0 .. floor(|m|/2 - v_m)
                kmax = (am - two_vm) // 2
                for k in range(kmax + 1):
                    two_v = two_vm + 2 * k               # 2 v (an integer)
                    sign = -1 if (t + k) % 2 else 1      # (-1)^(t + v - v_m)
                    coef = Fraction(sign, 4 ** t) * comb(l, t) * comb(l - t, am + t) * comb(t, u) * comb(am, two_v)
                    px = 2 * t + am - 2 * u - two_v
                    py = 2 * u + two_v
                    pz = l - 2 * t - am
                    S[m + l, index[(px, py, pz)]] += norm * float(coef)
    return S


def cart_to_pure(lx, cart):
    """Apply the transform to the aux index of out[npair, nx, nc(lx), na, nb] -> [npair, nx, 2lx+1, na, nb]."""
    return np.einsum("mc,pxcab->pxmab", solid_matrix(lx), np.asarray(cart, dtype=np.float64))
