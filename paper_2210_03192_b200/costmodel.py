"""Algorithmic FLOP / byte model per shell-set, used only to turn measured times into roofline
fractions.  Counted on the uni-quantal, component-level DAG of the HGPA scheme (§2.5.1): what the method
must compute, each needed intermediate once, every multiply-add as one FMA = 2 flops.

    flops/set = K * (40 + 4 (L+1) + 2 VRR_FMA + 2 sum_{e=La}^{La+Lb} nc(e) nc(Lx)) + 2 HRR_FMA
    bytes/set = 8 nc(Lx) nc(La) nc(Lb)          (the stored shell-set; zero for the DF digestions)

VRR_FMA counts eq. 3 (VRR1) and the full Obara-Saika ket relation (reading G4) over the nodes [e0|c]^(m) reachable
from the targets [e0|c]^(0), La <= e <= La+Lb, |c| = Lx, recursing along the axis with the smallest positive power;
HRR_FMA counts eq. 1 over the nodes reachable from (X|ab).
"""
from functools import lru_cache


def ncart(l):
    return (l + 1) * (l + 2) // 2


def comps(l):
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def _dir(v):
    best, d = 99, 0
    for i in range(3):
        if 0 < v[i] < best:
            best, d = v[i], i
    return d


def _dec(v, i, n=1):
    w = list(v)
    w[i] -= n
    return tuple(w)


@lru_cache(maxsize=None)
def vrr_fma(lx, la, lb):
    """FMAs per primitive triple for all VRR1+VRR2 nodes needed by the targets."""
    seen = {}

    def need(a, c, m):
        key = (a, c, m)
        if key in seen:
            return
        cost = 0
        if sum(c) > 0:                      # VRR2: raise the ket along i
            i = _dir(c)
            c1 = _dec(c, i)
            need(a, c1, m + 1)
            cost += 1
            if a[i] > 0:
                need(_dec(a, i), c1, m + 1)
                cost += 1
            if c[i] > 1:
                c2 = _dec(c, i, 2)
                need(a, c2, m)
                need(a, c2, m + 1)
                cost += 2
        elif sum(a) > 0:                    # VRR1 (eq. 3)
            i = _dir(a)
            a1 = _dec(a, i)
            need(a1, c, m)
            need(a1, c, m + 1)
            cost += 2
            if a[i] > 1:
                a2 = _dec(a, i, 2)
                need(a2, c, m)
                need(a2, c, m + 1)
                cost += 2
        seen[key] = cost

    for e in range(la, la + lb + 1):
        for a in comps(e):
            for c in comps(lx):
                need(a, c, 0)
    return sum(seen.values())


@lru_cache(maxsize=None)
def hrr_fma(lx, la, lb):
    seen = set()

    def need(a, b):
        if sum(b) == 0 or (a, b) in seen:
            return
        seen.add((a, b))
        i = _dir(b)
        b1 = _dec(b, i)
        a1 = list(a)
        a1[i] += 1
        need(tuple(a1), b1)
        need(a, b1)

    for a in comps(la):
        for b in comps(lb):
            need(a, b)
    return len(seen) * ncart(lx)


def flops_per_set(lx, la, lb, K):
    if la < lb:
        la, lb = lb, la
    L = lx + la + lb
    contr = sum(ncart(e) * ncart(lx) for e in range(la, la + lb + 1))
    return K * (40 + 4 * (L + 1) + 2 * vrr_fma(lx, la, lb) + 2 * contr) + 2 * hrr_fma(lx, la, lb)


def bytes_per_set(lx, la, lb):
    return 8 * ncart(lx) * ncart(la) * ncart(lb)


def nint_per_set(lx, la, lb):
    return ncart(lx) * ncart(la) * ncart(lb)
