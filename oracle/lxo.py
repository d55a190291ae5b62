"""ORACLE — test infrastructure only.  ctypes binding of oracle/md_eri3.c (see its header).

Every function takes plain numpy arrays; a "shell table" is any object with the attributes
``L, prim_off, center, zeta, coef`` (and ``bf_off`` for the DF calls) — the oracle does not import the
module that defines the tables, it only reads these attributes.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liblxo.so")
_lib = None


def build(force=False):
    """Compile the C oracle with gcc (building the checker is not using it)."""
    srcs = [os.path.join(_HERE, "md_eri3.c"), os.path.join(_HERE, "md_impl.h")]
    if (not force) and os.path.exists(_SO) and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in srcs):
        return _SO
    cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", _SO, srcs[0], "-lm"]
    subprocess.check_call(cmd)
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_SO)
        _lib.lxo_max_threads.restype = C.c_int
        for n in ("lxo_eri3_batch_ld", "lxo_eri3_batch_d", "lxo_df_ld", "lxo_df_d"):
            getattr(_lib, n).restype = C.c_int
    return _lib


def max_threads():
    return int(_load().lxo_max_threads())


def ncart(l):
    return (l + 1) * (l + 2) // 2


def components(l):
    """Cartesian components of a shell in ABI order (reading G2): lx = l..0, ly = l-lx..0."""
    return [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def boys_ld(mmax, T):
    """F_m(T), m = 0..mmax, evaluated and returned in long double (eq. 19)."""
    out = np.zeros(mmax + 1, dtype=np.longdouble)
    _load().lxo_boys_ld(C.c_int(mmax), C.c_longdouble(T), _p(out, C.c_longdouble))
    return out


def boys(mmax, T):
    """F_m(T) in plain double arithmetic (the timed-baseline instantiation)."""
    out = np.zeros(mmax + 1, dtype=np.float64)
    _load().lxo_boys_d(C.c_int(mmax), C.c_double(T), _p(out, C.c_double))
    return out


def _tab(t):
    return (_i32(t.L), _i32(t.prim_off), _f64(t.center), _f64(t.zeta), _f64(t.coef))


def eri3_batch(lx, la, lb, aux, prim, x_idx, pair_idx, real="ld"):
    """(X|ab) for every listed pair × aux shell; returns out[npair, nx, nc(lx), nc(la), nc(lb)] (float64).

    real="ld": long double inside (parity);  real="d": double inside (timed baseline).
    """
    lib = _load()
    x_idx = _i32(x_idx)
    pair_idx = _i32(pair_idx).reshape(-1, 2)
    nx, npair = len(x_idx), len(pair_idx)
    out = np.zeros((npair, nx, ncart(lx), ncart(la), ncart(lb)), dtype=np.float64)
    xa, pa = _tab(aux), _tab(prim)
    fn = lib.lxo_eri3_batch_ld if real == "ld" else lib.lxo_eri3_batch_d
    i32, f64 = C.c_int32, C.c_double
    rc = fn(C.c_int(lx), C.c_int(la), C.c_int(lb),
            _p(xa[0], i32), _p(xa[1], i32), _p(xa[2], f64), _p(xa[3], f64), _p(xa[4], f64),
            _p(pa[0], i32), _p(pa[1], i32), _p(pa[2], f64), _p(pa[3], f64), _p(pa[4], f64),
            _p(x_idx, i32), C.c_int(nx), _p(pair_idx, i32), C.c_int(npair), _p(out, f64))
    if rc != 0:
        raise ValueError("oracle: a listed shell does not have the stated angular momentum")
    return out


def schwarz_aux(aux):
    """Q_X = sqrt(max_c (X_c|X_c)) per aux shell (Schwarz factors)."""
    xa = _tab(aux)
    q = np.zeros(len(xa[0]), dtype=np.float64)
    i32, f64 = C.c_int32, C.c_double
    _load().lxo_schwarz_aux(C.c_int(len(q)), _p(xa[0], i32), _p(xa[1], i32), _p(xa[3], f64), _p(xa[4], f64), _p(q, f64))
    return q


def schwarz_pair(prim, pair_idx):
    """Q_ab = sqrt(max_{a,b} (ab|ab)) per listed primary shell pair."""
    pa = _tab(prim)
    pair_idx = _i32(pair_idx).reshape(-1, 2)
    q = np.zeros(len(pair_idx), dtype=np.float64)
    i32, f64 = C.c_int32, C.c_double
    _load().lxo_schwarz_pair(_p(pa[0], i32), _p(pa[1], i32), _p(pa[2], f64), _p(pa[3], f64), _p(pa[4], f64),
                             _p(pair_idx, i32), C.c_int(len(pair_idx)), _p(q, f64))
    return q


def df_gamma_J(aux, prim, pair_idx, q_aux, q_pair, tau, D=None, d=None, x_sel=None, p_sel=None, real="ld"):
    """γ_X = Σ_ab (X|ab) D_ab and J_ab = Σ_X (X|ab) d_X over unique shell pairs with Schwarz screening
    ``q_aux[X]*q_pair[ab] < tau`` → skipped (readings G13, G16).

    Returns (gamma or None, J or None, n_sets, n_integrals).  x_sel / p_sel restrict the aux shells / pairs
    visited (sampled runs): gamma is then a partial sum over p_sel, J holds only the p_sel blocks.
    """
    lib = _load()
    xa, pa = _tab(aux), _tab(prim)
    xbf, pbf = _i32(aux.bf_off), _i32(prim.bf_off)
    pair_idx = _i32(pair_idx).reshape(-1, 2)
    nbf, naux = int(pbf[-1]), int(xbf[-1])
    i32, f64 = C.c_int32, C.c_double
    gamma = np.zeros(naux, dtype=np.float64) if D is not None else None
    J = np.zeros((nbf, nbf), dtype=np.float64) if d is not None else None
    Dm = _f64(D) if D is not None else None
    dv = _f64(d) if d is not None else None
    qa = _f64(q_aux) if q_aux is not None else None
    qp = _f64(q_pair) if q_pair is not None else None
    xs = _i32(x_sel) if x_sel is not None else None
    ps = _i32(p_sel) if p_sel is not None else None
    nsets, nints = C.c_int64(0), C.c_int64(0)
    null_f, null_i = C.POINTER(f64)(), C.POINTER(i32)()
    fn = lib.lxo_df_ld if real == "ld" else lib.lxo_df_d
    fn(C.c_int(len(xa[0])), _p(xa[0], i32), _p(xa[1], i32), _p(xa[2], f64), _p(xa[3], f64), _p(xa[4], f64),
       _p(xbf, i32), _p(pa[0], i32), _p(pa[1], i32), _p(pa[2], f64), _p(pa[3], f64), _p(pa[4], f64), _p(pbf, i32),
       _p(pair_idx, i32), C.c_int(len(pair_idx)),
       _p(qa, f64) if qa is not None else null_f, _p(qp, f64) if qp is not None else null_f, C.c_double(tau),
       _p(Dm, f64) if Dm is not None else null_f, C.c_int(nbf), _p(dv, f64) if dv is not None else null_f,
       _p(gamma, f64) if gamma is not None else null_f, _p(J, f64) if J is not None else null_f, C.c_int(nbf),
       _p(xs, i32) if xs is not None else null_i, C.c_int(len(xs) if xs is not None else 0),
       _p(ps, i32) if ps is not None else null_i, C.c_int(len(ps) if ps is not None else 0),
       C.byref(nsets), C.byref(nints))
    return gamma, J, int(nsets.value), int(nints.value)


class _Tab:
    pass


def metric_2c(aux):
    """Two-centre Coulomb metric of the fit, V[bf(X)+c, bf(Y)+c'] = (X_c|Y_c') = ∬ X_c(r1) Y_c'(r2) / r12 (PAPER.md:21,
    :365 "the two-center ... integrals"), Cartesian components, [naux_bf, naux_bf] float64.

    Written out from the definition with the 3-centre routine: Y_c'(r2) = Y_c'(r2) · 1 and the constant 1 is an s
    Gaussian of exponent 0 and coefficient 1 (any centre), so (X|Y) = (X|Y 1) — eq. 12 with ζ_b = 0, where the product
    centre P = A and the overlap factor is 1.  Pins: tests/test_oracle_metric.py (closed forms for s and p shells,
    symmetry between the two routes (X|Y 1) and (Y|X 1), the diagonal against the separate Schwarz routine, positive
    definiteness)."""
    L = _i32(aux.L)
    n = len(L)
    ext = _Tab()
    ext.L = np.concatenate([L, np.zeros(1, np.int32)])
    po = _i32(aux.prim_off)
    ext.prim_off = np.concatenate([po, np.asarray([po[-1] + 1], np.int32)])
    ext.center = np.concatenate([_f64(aux.center).reshape(-1), np.zeros(3)])
    ext.zeta = np.concatenate([_f64(aux.zeta), np.zeros(1)])
    ext.coef = np.concatenate([_f64(aux.coef), np.ones(1)])
    bf = _i32(aux.bf_off)
    nbf = int(bf[-1])
    V = np.zeros((nbf, nbf), dtype=np.float64)
    for lx in sorted(set(L.tolist())):
        xs = np.nonzero(L == lx)[0]
        for ly in sorted(set(L.tolist())):
            ys = np.nonzero(L == ly)[0]
            out = eri3_batch(lx, ly, 0, aux, ext, xs, [[int(y), n] for y in ys])      # [ny, nx, nc(lx), nc(ly), 1]
            for iy, y in enumerate(ys):
                for ix, x in enumerate(xs):
                    V[bf[x]:bf[x + 1], bf[y]:bf[y + 1]] = out[iy, ix, :, :, 0]
    return V


def fit_solve(V, gamma):
    """Fit coefficients d = V⁻¹ γ (PAPER.md:21 robust fit, :365) by the LAPACK Cholesky
    factorisation V = L Lᵀ and two triangular solves (numpy/scipy library routine as the step)."""
    import scipy.linalg as sl
    c = sl.cho_factor(np.asarray(V, dtype=np.float64), lower=True)
    return sl.cho_solve(c, np.asarray(gamma, dtype=np.float64))
