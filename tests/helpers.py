"""Test helpers: tiny shell-table builders and an independent brute-force quadrature of eq. 12."""
import numpy as np

import lx_inputs as gen


def table(shells):
    """shells: list of (l, centre(3), zetas, coefs)."""
    return gen.make_shells([s[0] for s in shells], [s[1] for s in shells],
                           [np.atleast_1d(s[2]) for s in shells], [np.atleast_1d(s[3]) for s in shells])


def comp_index(l, c):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)].index(tuple(c))


def bruteforce_primitive(c, a, b, C, A, B, zc, za, zb, nt=48, nh=12.0, step=0.22):
    """[c|ab] of PAPER.md eq. 12 for unnormalised primitives (eq. 13) by plain quadrature, independent of the
    Boys function and of every recurrence:
        1/r12 = (2/sqrt(pi)) int_0^inf exp(-u^2 r12^2) du ,  u = sqrt(rho) t / sqrt(1-t^2)   (Gauss-Legendre in t)
        per axis  I(u) = iint (x1-C)^c e^{-zc (x1-C)^2} e^{-u^2 (x1-x2)^2} (x2-A)^a (x2-B)^b e^{-za(x2-A)^2 - zb(x2-B)^2}
    with the trapezoid rule (spectrally accurate for Gaussians) in x2 and in s = x1-x2, the s grid scaled to the
    width 1/sqrt(u^2+zc) and centred on the maximum of the s-Gaussian.
    """
    p = za + zb
    rho = p * zc / (p + zc)
    tn, tw = np.polynomial.legendre.leggauss(nt)
    tn = 0.5 * (tn + 1.0)
    tw = 0.5 * tw
    total = 0.0
    for t, w in zip(tn, tw):
        u2 = rho * t * t / (1.0 - t * t)
        dudt = np.sqrt(rho) * (1.0 - t * t) ** -1.5
        prod = 1.0
        for ax in range(3):
            P = (za * A[ax] + zb * B[ax]) / p
            h2 = step / np.sqrt(p)
            n2 = int(np.ceil(nh / step)) + 8 * (a[ax] + b[ax] + c[ax] + 1)
            x2 = P + h2 * np.arange(-n2, n2 + 1)
            al = u2 + zc
            hs = step / np.sqrt(al)
            ns = int(np.ceil(nh / step)) + 8 * (c[ax] + 1)
            k = hs * np.arange(-ns, ns + 1)
            s0 = -zc * (x2 - C[ax]) / al
            s = s0[:, None] + k[None, :]
            x1 = x2[:, None] + s
            f = ((x1 - C[ax]) ** c[ax]) * np.exp(-zc * (x1 - C[ax]) ** 2 - u2 * s * s)
            g = ((x2 - A[ax]) ** a[ax]) * ((x2 - B[ax]) ** b[ax]) * np.exp(-za * (x2 - A[ax]) ** 2 - zb * (x2 - B[ax]) ** 2)
            prod *= h2 * hs * float(np.sum(f * g[:, None]))
        total += w * dudt * prod
    return 2.0 / np.sqrt(np.pi) * total


def bruteforce_pair_diagonal(a, b, A, B, za, zb, nt=48, nh=12.0, step=0.22):
    """(ab|ab) for ONE unnormalised primitive pair by the same plain quadrature as bruteforce_primitive (no Boys
    function, no recurrence): both electrons carry the product (x-A)^a (x-B)^b exp(-za (x-A)^2 - zb (x-B)^2).
        1/r12 = (2/sqrt(pi)) int_0^inf exp(-u^2 r12^2) du,  u = sqrt(rho) t / sqrt(1-t^2),  rho = p/2, p = za + zb."""
    p = za + zb
    rho = 0.5 * p
    tn, tw = np.polynomial.legendre.leggauss(nt)
    tn = 0.5 * (tn + 1.0)
    tw = 0.5 * tw
    total = 0.0
    for t, w in zip(tn, tw):
        u2 = rho * t * t / (1.0 - t * t)
        dudt = np.sqrt(rho) * (1.0 - t * t) ** -1.5
        prod = 1.0
        for ax in range(3):
            P = (za * A[ax] + zb * B[ax]) / p
            deg = a[ax] + b[ax]
            h2 = step / np.sqrt(p)
            n2 = int(np.ceil(nh / step)) + 8 * (2 * deg + 1)
            x2 = P + h2 * np.arange(-n2, n2 + 1)
            al = u2 + p
            hs = step / np.sqrt(al)
            ns = int(np.ceil(nh / step)) + 8 * (deg + 1)
            k = hs * np.arange(-ns, ns + 1)
            s0 = -p * (x2 - P) / al
            s = s0[:, None] + k[None, :]
            x1 = x2[:, None] + s
            f = ((x1 - A[ax]) ** a[ax]) * ((x1 - B[ax]) ** b[ax]) * np.exp(-za * (x1 - A[ax]) ** 2 - zb * (x1 - B[ax]) ** 2 - u2 * s * s)
            g = ((x2 - A[ax]) ** a[ax]) * ((x2 - B[ax]) ** b[ax]) * np.exp(-za * (x2 - A[ax]) ** 2 - zb * (x2 - B[ax]) ** 2)
            prod *= h2 * hs * float(np.sum(f * g[:, None]))
        total += w * dudt * prod
    return 2.0 / np.sqrt(np.pi) * total
