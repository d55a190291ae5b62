"""GPU two-centre metric V_XY = (X|Y) and fit solve d = V^-1 gamma (lx_metric_2c / lx_fit_solve; SURVEY.md §8(f) NEXT-2,
PAPER.md:21, :365) against the long-double oracle.

Tolerances.  Metric: |V_ij - ref_ij| <= 1e-12 sqrt(ref_ii ref_jj) — the Cauchy-Schwarz scale of the entry; the Hermite sums
of a high-L pair cancel against terms of that size, so an entry-relative bound would be the wrong yardstick for entries that
are small by symmetry.  Solve: Cholesky is backward stable, the residual obeys |V d - gamma| <= c n eps |V| |d|; against the
oracle's solution the error is bounded by cond(V) times that."""
import numpy as np
import pytest

import lx_inputs as gen
from helpers import table

pytestmark = pytest.mark.gpu

TOL_V = 1e-12


@pytest.fixture(scope="module")
def lx():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2210_03192_b200 import lx as _lx
    _lx.lx_init(0)
    return _lx


def _scaled_err(got, ref):
    s = np.sqrt(np.diag(ref))
    return float(np.max(np.abs(got - ref) / np.outer(s, s)))


def _all_l_table(seed, per_l=2):
    rng = np.random.default_rng(seed)
    xs = []
    shared = rng.uniform(0, 3, 3)
    for l in range(7):
        for r in range(per_l):
            k = 1 + (l + r) % 3
            z = np.exp(rng.uniform(np.log(0.1), np.log(8.0), k))
            ctr = shared if r == 0 else rng.uniform(0, 3, 3)          # every L also meets the others on ONE centre (R = 0)
            xs.append((l, ctr, z, rng.uniform(0.3, 1.0, k) * gen.prim_norm(z, l)))
    return table(xs)


def test_metric_every_class(lx, oracle):
    """All 28 (Lx, Ly) classes, contracted shells (K = 1..3), coinciding and distinct centres; exact symmetry."""
    import torch
    aux = _all_l_table(21)
    V = lx.lx_metric_2c(lx.HostShells(aux))
    assert torch.equal(V, V.T)
    err = _scaled_err(V.cpu().numpy(), oracle.metric_2c(aux))
    assert err <= TOL_V, err


def test_metric_padded_leading_dimension_and_shell_order(lx, oracle):
    """ld > n leaves the padding untouched; a shuffled shell order moves blocks, nothing else."""
    import torch
    aux = _all_l_table(22, per_l=1)
    n = aux.nbf
    buf = torch.full((n, n + 5), -7.0, dtype=torch.float64, device="cuda")
    lx.lx_metric_2c(lx.HostShells(aux), buf)
    assert torch.all(buf[:, n:] == -7.0)
    ref = oracle.metric_2c(aux)
    assert _scaled_err(buf[:, :n].cpu().numpy(), ref) <= TOL_V
    perm = np.random.default_rng(1).permutation(aux.nshell)
    sh = gen.make_shells([aux.L[i] for i in perm], [aux.center.reshape(-1, 3)[i] for i in perm],
                         [aux.zeta[aux.prim_off[i]:aux.prim_off[i + 1]] for i in perm],
                         [aux.coef[aux.prim_off[i]:aux.prim_off[i + 1]] for i in perm])
    Vp = lx.lx_metric_2c(lx.HostShells(sh)).cpu().numpy()
    idx = np.concatenate([np.arange(aux.bf_off[i], aux.bf_off[i + 1]) for i in perm])
    assert _scaled_err(Vp, ref[np.ix_(idx, idx)]) <= TOL_V


def test_metric_config4_sampled_and_fit_residual(lx, oracle):
    """Config 4's aux basis in full on the GPU (6784 functions); 160 sampled shells against the oracle block by block;
    then d = V^-1 gamma on the conditioned fit subset (4544 functions) with the backward-stability residual bound."""
    import torch
    c4 = gen.config4()
    aux = c4["aux"]
    V = lx.lx_metric_2c(lx.HostShells(aux))
    assert torch.equal(V, V.T)
    rng = np.random.default_rng(8)
    pick = np.sort(rng.choice(aux.nshell, 160, replace=False))
    ctr = aux.center.reshape(-1, 3)
    sub = gen.make_shells([aux.L[i] for i in pick], [ctr[i] for i in pick],
                          [aux.zeta[aux.prim_off[i]:aux.prim_off[i + 1]] for i in pick],
                          [aux.coef[aux.prim_off[i]:aux.prim_off[i + 1]] for i in pick])
    idx = torch.as_tensor(np.concatenate([np.arange(aux.bf_off[i], aux.bf_off[i + 1]) for i in pick]), device="cuda")
    got = V[idx][:, idx].cpu().numpy()
    err = _scaled_err(got, oracle.metric_2c(sub))
    assert err <= TOL_V, err
    # the full synthetic basis is numerically singular (lx_inputs.fit_subset): the fit runs on its conditioned subset,
    # whose metric is a principal submatrix of V
    sub, keep = gen.fit_subset(aux)
    keep = torch.as_tensor(keep, device="cuda")
    Vs = V[keep][:, keep].contiguous()
    assert torch.equal(Vs, lx.lx_metric_2c(lx.HostShells(sub)))       # same shell pairs, same arithmetic: bit-identical
    n = sub.nbf
    g = torch.as_tensor(rng.normal(size=n), device="cuda")
    F = Vs.clone()
    d = lx.lx_fit_solve(F, g.clone())
    res = float(torch.max(torch.abs(Vs @ d - g)))
    bound = 1e-14 * n * float(torch.max(torch.abs(Vs))) * float(torch.max(torch.abs(d)))
    print(f"config 4 fit: n = {n}, residual {res:.2e}, backward-stability bound {bound:.2e}")
    assert res <= bound
    g2 = torch.as_tensor(rng.normal(size=(2, n)), device="cuda")                 # factor reused, two right-hand sides
    d2 = lx.lx_fit_solve(F, g2.clone(), factored=True)
    assert float(torch.max(torch.abs(d2 @ Vs - g2))) <= 1e-14 * n * float(torch.max(torch.abs(Vs))) * float(torch.max(torch.abs(d2)))
    d1 = lx.lx_fit_solve(F, g.clone(), factored=True)
    assert torch.equal(d1, d)


def test_fit_solve_against_oracle(lx, oracle):
    import torch
    rng = np.random.default_rng(3)
    prim, aux = gen._cluster(rng, 3, 5.0, gen._PRIM4, gen._AUX4[:3])
    Vo = oracle.metric_2c(aux)
    g = rng.normal(size=aux.nbf)
    do = oracle.fit_solve(Vo, g)
    V = lx.lx_metric_2c(lx.HostShells(aux))
    d = lx.lx_fit_solve(V, torch.as_tensor(g, device="cuda")).cpu().numpy()
    cond = np.linalg.cond(Vo)
    err = float(np.max(np.abs(d - do)) / np.max(np.abs(do)))
    print(f"fit solve: n = {aux.nbf}, cond(V) = {cond:.2e}, error against the oracle {err:.2e}")
    assert err <= 1e-14 * cond * np.sqrt(aux.nbf)


def test_fit_solve_errors_and_empty(lx):
    import torch
    Vneg = -torch.eye(4, dtype=torch.float64, device="cuda")
    with pytest.raises(lx.LxError) as e:
        lx.lx_fit_solve(Vneg, torch.ones(4, dtype=torch.float64, device="cuda"))
    assert e.value.status == lx.LX_ENOTPD
    V0 = torch.empty((0, 0), dtype=torch.float64, device="cuda")
    lx.lx_fit_solve(V0, None)
    aux = _all_l_table(5, per_l=1)
    small = torch.empty((aux.nbf, aux.nbf - 1), dtype=torch.float64, device="cuda")
    import ctypes as C
    hs = lx.HostShells(aux)
    assert lx._lib.lx_metric_2c(C.byref(hs.struct), small.data_ptr(), aux.nbf - 1) == lx.LX_EINVAL
    bad = table([(7, [0, 0, 0], [1.0], [1.0])])
    with pytest.raises(lx.LxError) as e:
        lx.lx_metric_2c(lx.HostShells(bad))
    assert e.value.status == lx.LX_EUNSUPPORTED


def test_two_pass_df_j_against_oracle(lx, oracle):
    """The whole density-fitted Coulomb build through the C ABI: Schwarz factors -> schedule -> gamma = (X|ab) D
    -> d = V^-1 gamma -> J = (X|ab) d, every step on the GPU, against the same chain in the oracle.  d carries the factor
    cond(V) of the solve, J inherits it: the bound is eps cond(V) sqrt(naux) (eps = 2.2e-16) on the scale of the largest
    element (measured: d 5e-11 at cond 4e7, J 1.5e-13 — the error of d lies along the weakly weighted directions of V)."""
    import torch
    rng = np.random.default_rng(12)
    prim, aux = gen._cluster(rng, 4, 6.0, gen._PRIM4, gen._AUX4[:3])
    pairs = gen.unique_pairs(prim.nshell)
    nbf = prim.nbf
    Cm = rng.normal(0, 1 / np.sqrt(nbf), size=(nbf, max(nbf // 4, 1)))
    D = Cm @ Cm.T
    tau = 1e-12
    # oracle chain
    qx_o, qp_o = oracle.schwarz_aux(aux), oracle.schwarz_pair(prim, pairs)
    g_o, _, nsets_o, _ = oracle.df_gamma_J(aux, prim, pairs, qx_o, qp_o, tau, D=D)
    V_o = oracle.metric_2c(aux)
    d_o = oracle.fit_solve(V_o, g_o)
    _, J_o, _, _ = oracle.df_gamma_J(aux, prim, pairs, qx_o, qp_o, tau, d=d_o)
    # GPU chain
    ha, hp = lx.HostShells(aux), lx.HostShells(prim)
    qx, qp = lx.lx_schwarz_aux_host(ha), lx.lx_schwarz_pair_host(hp, pairs)
    sched = lx.Schedule(ha, hp, qx, qp, pairs, tau)
    assert sched.num_sets == nsets_o
    da, dp = lx.DeviceShells(ha, "cuda:0"), lx.DeviceShells(hp, "cuda:0")
    gam = lx.lx_df_gamma(sched, da, dp, torch.as_tensor(D, device="cuda"))
    V = lx.lx_metric_2c(ha)
    d = lx.lx_fit_solve(V, gam.clone())
    J = lx.lx_df_J(sched, da, dp, d)
    torch.cuda.synchronize()
    cond = np.linalg.cond(V_o)
    tol = 2.2e-16 * cond * np.sqrt(aux.nbf)
    eg = float(np.max(np.abs(gam.cpu().numpy() - g_o)) / np.max(np.abs(g_o)))
    ed = float(np.max(np.abs(d.cpu().numpy() - d_o)) / np.max(np.abs(d_o)))
    eJ = float(np.max(np.abs(J.cpu().numpy() - J_o)) / np.max(np.abs(J_o)))      # both sides mirror J to (b, a)
    print(f"two-pass DF-J: naux = {aux.nbf}, cond(V) = {cond:.2e}; errors gamma {eg:.1e}, d {ed:.1e}, J {eJ:.1e} (bound {tol:.1e})")
    assert eg <= 1e-12 and ed <= tol and eJ <= tol
