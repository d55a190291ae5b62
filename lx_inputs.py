"""Seeded synthetic inputs shared by the oracle tests and the CUDA path (and by nothing else).

This module holds NO integral arithmetic: it only draws shell tables, shell-pair lists, densities and fit
vectors with the shapes and value distributions of BASELINE.json's five configs (the paper's workloads,
PAPER.md Table 5 lines 369-397 and Table 6, whose molecules and basis-set files are not
available and are not reproduced).  The recipe is restated in DESIGN.md ("Input recipe").

Draw order for every config: primary centres, primary exponents, primary coefficients, then the same three
for the aux table, all from one ``numpy.random.default_rng`` (PCG64) stream.
"""
from dataclasses import dataclass
from math import pi

import numpy as np


def ncart(l):
    return (l + 1) * (l + 2) // 2


def dfact(n):
    r = 1.0
    while n > 1:
        r *= n
        n -= 2
    return r


def prim_norm(zeta, l):
    """Normalisation of the x^l primitive, folded into ``coef`` by the generator (reading G3):
    N(zeta,l) = (2 zeta/pi)^(3/4) (4 zeta)^(l/2) / sqrt((2l-1)!!).  The library itself adds none."""
    zeta = np.asarray(zeta, dtype=np.float64)
    return (2.0 * zeta / pi) ** 0.75 * (4.0 * zeta) ** (0.5 * l) / np.sqrt(dfact(2 * l - 1))


@dataclass
class Shells:
    """SoA shell table (same fields as lx_shells_t in include/lx.h)."""
    L: np.ndarray          # [nshell] int32
    K: np.ndarray          # [nshell] int32
    prim_off: np.ndarray   # [nshell+1] int32
    center: np.ndarray     # [nshell*3] float64 (bohr)
    zeta: np.ndarray       # [nprim]
    coef: np.ndarray       # [nprim]  (includes normalisation)
    bf_off: np.ndarray     # [nshell+1] int32, Cartesian basis-function offsets

    @property
    def nshell(self):
        return len(self.L)

    @property
    def nbf(self):
        return int(self.bf_off[-1])


def make_shells(Ls, centers, zetas, coefs):
    """Assemble a table from per-shell lists (zetas[i], coefs[i] are 1-D arrays of equal length)."""
    Ls = np.asarray(Ls, dtype=np.int32)
    K = np.array([len(z) for z in zetas], dtype=np.int32)
    prim_off = np.zeros(len(Ls) + 1, dtype=np.int32)
    prim_off[1:] = np.cumsum(K)
    bf_off = np.zeros(len(Ls) + 1, dtype=np.int32)
    bf_off[1:] = np.cumsum([ncart(int(l)) for l in Ls])
    return Shells(L=Ls, K=K, prim_off=prim_off,
                  center=np.ascontiguousarray(np.asarray(centers, dtype=np.float64).reshape(-1)),
                  zeta=np.concatenate([np.asarray(z, dtype=np.float64) for z in zetas]) if len(zetas) else np.zeros(0),
                  coef=np.concatenate([np.asarray(c, dtype=np.float64) for c in coefs]) if len(coefs) else np.zeros(0),
                  bf_off=bf_off)


def _log_uniform(rng, lo, hi, n):
    return np.exp(rng.uniform(np.log(lo), np.log(hi), size=n))


def _min_sep_points(rng, n, box, dmin):
    """Random sequential placement of n points in [0,box]^3 with pairwise distance >= dmin."""
    pts = np.zeros((0, 3))
    while len(pts) < n:
        cand = rng.uniform(0.0, box, size=(max(4 * (n - len(pts)), 16), 3))
        for c in cand:
            if len(pts) == 0 or np.min(np.sum((pts - c) ** 2, axis=1)) >= dmin * dmin:
                pts = np.vstack([pts, c])
                if len(pts) == n:
                    break
    return pts


# ----------------------------------------------------------------------------------------------------------
# Config 1: single class (d|pp), K=1, 64 pairs x 32 aux shells, 10-bohr cube, seed 0
# ----------------------------------------------------------------------------------------------------------
def config1(seed=0, npair=64, nx=32):
    rng = np.random.default_rng(seed)
    n = 2 * npair
    pc = rng.uniform(0.0, 10.0, size=(n, 3))
    pz = _log_uniform(rng, 0.1, 10.0, n)
    prim = make_shells([1] * n, pc, [[z] for z in pz], [[float(prim_norm(z, 1))] for z in pz])
    xc = rng.uniform(0.0, 10.0, size=(nx, 3))
    xz = _log_uniform(rng, 0.1, 10.0, nx)
    aux = make_shells([2] * nx, xc, [[z] for z in xz], [[float(prim_norm(z, 2))] for z in xz])
    pair_idx = np.stack([2 * np.arange(npair), 2 * np.arange(npair) + 1], axis=1).astype(np.int32)
    return dict(lx=2, la=1, lb=1, aux=aux, prim=prim, x_idx=np.arange(nx, dtype=np.int32), pair_idx=pair_idx)


# ----------------------------------------------------------------------------------------------------------
# Config 2: class sweep, primary K=3 (ratio-3 geometric, smallest log-U[0.1,0.5], c ~ U[0.2,1] x N),
#           aux K=1 (log-U[0.05,20]), 1024 pairs x 256 aux per class, 20-bohr cube
# ----------------------------------------------------------------------------------------------------------
CONFIG2_CLASSES = [(lx, la, lb) for lx in range(5) for la in range(3) for lb in range(3)]


def config2(lx, la, lb, npair=1024, nx=256, seed=2):
    rng = np.random.default_rng([seed, 1000 * lx + 100 * la + 10 * lb])
    n = 2 * npair
    Ls = [la] * npair + [lb] * npair
    pc = rng.uniform(0.0, 20.0, size=(n, 3))
    zmin = _log_uniform(rng, 0.1, 0.5, n)
    zs = [zmin[i] * 3.0 ** np.arange(3) for i in range(n)]
    cu = rng.uniform(0.2, 1.0, size=(n, 3))
    cs = [cu[i] * prim_norm(zs[i], Ls[i]) for i in range(n)]
    prim = make_shells(Ls, pc, zs, cs)
    xc = rng.uniform(0.0, 20.0, size=(nx, 3))
    xz = _log_uniform(rng, 0.05, 20.0, nx)
    aux = make_shells([lx] * nx, xc, [[z] for z in xz], [[float(prim_norm(z, lx))] for z in xz])
    pair_idx = np.stack([np.arange(npair), npair + np.arange(npair)], axis=1).astype(np.int32)
    return dict(lx=lx, la=la, lb=lb, aux=aux, prim=prim, x_idx=np.arange(nx, dtype=np.int32), pair_idx=pair_idx)


# ----------------------------------------------------------------------------------------------------------
# Config 3: high angular momentum.  (6|33) (6|22) (5|33) (4|44) at K=1; (5|22) with primary K=5 geometric over
#           [0.05,50]; 4096 pairs x 128 aux; centres in a 15-bohr cube with min separation 1.5 bohr.
#           8192+128 distinct centres cannot keep 1.5 bohr apart in 15^3 bohr^3 (packing bound ~1400), so the
#           shells sit on 256 min-separated "atom" centres drawn first; each shell picks an atom (R3).
# ----------------------------------------------------------------------------------------------------------
CONFIG3_CLASSES = [(6, 3, 3, 1), (6, 2, 2, 1), (5, 3, 3, 1), (4, 4, 4, 1), (5, 2, 2, 5)]


def config3(lx, la, lb, kprim=1, npair=4096, nx=128, seed=3, natom=256):
    rng = np.random.default_rng([seed, 1000 * lx + 100 * la + 10 * lb])
    atoms = _min_sep_points(rng, natom, 15.0, 1.5)
    n = 2 * npair
    Ls = [la] * npair + [lb] * npair
    pc = atoms[rng.integers(0, natom, size=n)]
    if kprim == 1:
        pz = _log_uniform(rng, 0.1, 10.0, n)
        zs = [[z] for z in pz]
        cs = [[float(prim_norm(z, l))] for z, l in zip(pz, Ls)]
    else:
        zgeo = 0.05 * (50.0 / 0.05) ** (np.arange(kprim) / (kprim - 1))
        zs = [zgeo.copy() for _ in range(n)]
        cu = rng.uniform(0.2, 1.0, size=(n, kprim))
        cs = [cu[i] * prim_norm(zs[i], Ls[i]) for i in range(n)]
    prim = make_shells(Ls, pc, zs, cs)
    xc = atoms[rng.integers(0, natom, size=nx)]
    xz = _log_uniform(rng, 0.05, 20.0, nx)
    aux = make_shells([lx] * nx, xc, [[z] for z in xz], [[float(prim_norm(z, lx))] for z in xz])
    pair_idx = np.stack([np.arange(npair), npair + np.arange(npair)], axis=1).astype(np.int32)
    return dict(lx=lx, la=la, lb=lb, aux=aux, prim=prim, x_idx=np.arange(nx, dtype=np.int32), pair_idx=pair_idx)


# ----------------------------------------------------------------------------------------------------------
# Configs 4 and 5: DF Coulomb on synthetic atom clusters
# ----------------------------------------------------------------------------------------------------------
def _geo(lo, hi, n):
    if n == 1:
        return np.array([np.sqrt(lo * hi)])
    return lo * (hi / lo) ** (np.arange(n) / (n - 1))


# (l, smallest exponent, K, ratio) per primary shell of one atom; contracted shells geometric upward
_PRIM4 = [(0, 4000.0 / 3.2 ** 7, 8, 3.2), (0, 0.5, 1, 1.0), (0, 0.15, 1, 1.0),
          (1, 0.625, 3, 4.0), (1, 0.18, 1, 1.0), (2, 0.8, 1, 1.0)]
_AUX4 = [(0, 7), (1, 5), (2, 4), (3, 3), (4, 2)]
_PRIM5 = [(0, 1.5, 10, 3.0), (0, 0.9, 3, 3.0), (0, 0.35, 1, 1.0), (0, 0.12, 1, 1.0),
          (1, 0.7, 3, 3.0), (1, 0.25, 1, 1.0), (1, 0.09, 1, 1.0),
          (2, 0.6, 2, 3.0), (2, 0.2, 1, 1.0), (3, 0.5, 1, 1.0)]
_AUX5 = [(0, 8), (1, 6), (2, 5), (3, 4), (4, 3), (5, 2), (6, 1)]


def _cluster(rng, natom, box, prim_spec, aux_spec):
    atoms = _min_sep_points(rng, natom, box, 1.8)
    Ls, cen, zs = [], [], []
    for at in atoms:
        for (l, zmin, k, ratio) in prim_spec:
            Ls.append(l)
            cen.append(at)
            zs.append(zmin * ratio ** np.arange(k))
    cs = []
    for l, z in zip(Ls, zs):
        c = rng.uniform(0.2, 1.0, size=len(z)) if len(z) > 1 else np.ones(1)
        cs.append(c * prim_norm(z, l))
    prim = make_shells(Ls, cen, zs, cs)
    xL, xcen, xz = [], [], []
    for at in atoms:
        for (l, n) in aux_spec:
            for z in _geo(0.1, 30.0, n):
                xL.append(l)
                xcen.append(at)
                xz.append([z])
    aux = make_shells(xL, xcen, xz, [[float(prim_norm(z[0], l))] for z, l in zip(xz, xL)])
    return prim, aux


def unique_pairs(nshell):
    """All unique shell pairs (a >= b), including a == b."""
    a, b = np.tril_indices(nshell)
    return np.stack([a, b], axis=1).astype(np.int32)


def _df_config(seed, natom, box, prim_spec, aux_spec):
    rng = np.random.default_rng(seed)
    prim, aux = _cluster(rng, natom, box, prim_spec, aux_spec)
    nbf, naux = prim.nbf, aux.nbf
    Cm = rng.normal(0.0, np.sqrt(1.0 / nbf), size=(nbf, max(nbf // 4, 1)))
    D = Cm @ Cm.T
    D = 0.5 * (D + D.T)
    d = rng.normal(0.0, 1.0, size=naux)
    return dict(aux=aux, prim=prim, pair_idx=unique_pairs(prim.nshell), D=D, d=d, tau=1e-12)


def config4(seed=4, natom=64):
    """64-atom cluster, 30-bohr box: primary s(K=8) s s p(K=3) p d; aux 7s5p4d3f2g over [0.1,30]."""
    return _df_config(seed, natom, 30.0, _PRIM4, _AUX4)


def config5(seed=5, natom=256):
    """256-atom cluster, 50-bohr box: primary 4s3p2d1f (first s K=10); aux 8s6p5d4f3g2h1i."""
    return _df_config(seed, natom, 50.0, _PRIM5, _AUX5)


def fit_subset(aux, zmin=0.15):
    """The aux shells usable as a FIT basis: the synthetic aux sets of configs 4/5 put ζ = 0.1 functions of every L on
    every atom, which makes the two-centre metric numerically singular (config 4: λmin/λmax = 7e-19 by the oracle);
    without the shells of smallest exponent < zmin the condition number is ~1e8.  Returns (table of the kept shells,
    basis-function indices of the kept shells in the full table)."""
    keep = [i for i in range(aux.nshell) if float(np.min(aux.zeta[aux.prim_off[i]:aux.prim_off[i + 1]])) >= zmin]
    ctr = aux.center.reshape(-1, 3)
    sub = make_shells([aux.L[i] for i in keep], [ctr[i] for i in keep],
                      [aux.zeta[aux.prim_off[i]:aux.prim_off[i + 1]] for i in keep],
                      [aux.coef[aux.prim_off[i]:aux.prim_off[i + 1]] for i in keep])
    idx = np.concatenate([np.arange(aux.bf_off[i], aux.bf_off[i + 1]) for i in keep]) if keep else np.zeros(0, np.int64)
    return sub, idx
