"""GPU parity of the integral-direct DF contractions at the stated configurations:
BASELINE.json configs[3] (64 atoms) in full, configs[4] (256 atoms, aux L up to 6, primary up to f) on the seeded
sample SURVEY.md §8(d) prescribes, and small clusters built from the config-5 basis so that the digestion of every
kernel family is compared element by element.  Tolerance (north_star): relative Frobenius <= 1e-11 for gamma and J.
Schwarz factors are the ORACLE's (long double) and are passed to both sides (reading G13: identical screening,
PAPER.md:365)."""
import numpy as np
import pytest

import lx_inputs as gen

pytestmark = pytest.mark.gpu

TOL_DF = 1e-11


@pytest.fixture(scope="module")
def lx():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2210_03192_b200 import lx as _lx
    _lx.lx_init(0)
    return _lx


def _relerr(got, ref):
    return float(np.linalg.norm(got - ref) / np.linalg.norm(ref))


def _gpu_df(lx, aux, prim, pairs, qx, qp, tau, D, d):
    import torch
    ha, hp = lx.HostShells(aux), lx.HostShells(prim)
    sched = lx.Schedule(ha, hp, qx, qp, pairs, tau)
    da, dp = lx.DeviceShells(ha), lx.DeviceShells(hp)
    ws = torch.empty(sched.workspace_bytes, dtype=torch.uint8, device="cuda")
    gamma = lx.lx_df_gamma(sched, da, dp, torch.from_numpy(np.ascontiguousarray(D)).cuda(), workspace=ws)
    J = lx.lx_df_J(sched, da, dp, torch.from_numpy(np.ascontiguousarray(d)).cuda(), workspace=ws)
    torch.cuda.synchronize()
    return sched, gamma.cpu().numpy(), J.cpu().numpy()


@pytest.mark.parametrize("natom,box,tau", [(2, 4.0, 1e-12), (3, 6.0, 1e-12), (3, 9.0, 1e-6), (2, 3.0, None)])
def test_df_high_L_small_cluster(lx, oracle, natom, box, tau):
    """Clusters of 2-3 atoms with the config-5 basis (primary up to f, aux up to i): every (Lx|LaLb) class with
    Lx <= 6, La,Lb <= 3 goes through lx_df_gamma / lx_df_J, i.e. MODE 1/2 of the team, chain, lane and group families,
    with and without screening, against the oracle element by element; the schedule's integer counts are bit-exact."""
    rng = np.random.default_rng(31 + natom)
    prim, aux = gen._cluster(rng, natom, box, gen._PRIM5, gen._AUX5)
    pairs = gen.unique_pairs(prim.nshell)
    D = rng.normal(size=(prim.nbf, prim.nbf))
    D = D + D.T
    d = rng.normal(size=aux.nbf)
    if tau is None:
        qx = qp = None
        tau = 0.0
    else:
        qx, qp = oracle.schwarz_aux(aux), oracle.schwarz_pair(prim, pairs)
    g_ref, J_ref, nsets, nints = oracle.df_gamma_J(aux, prim, pairs, qx, qp, tau, D=D, d=d)
    sched, gamma, J = _gpu_df(lx, aux, prim, pairs, qx, qp, tau, D, d)
    assert sched.num_sets == nsets and sched.num_integrals == nints
    assert np.isfinite(gamma).all() and np.isfinite(J).all()
    eg, eJ = _relerr(gamma, g_ref), _relerr(J, J_ref)
    assert eg <= TOL_DF and eJ <= TOL_DF, (eg, eJ)
    assert np.linalg.norm(J - J.T) <= 1e-13 * np.linalg.norm(J)      # mirrored atomics: equal up to summation order (G14)
    assert abs(gamma @ d - np.sum(J * D)) <= 1e-10 * abs(gamma @ d)


@pytest.mark.parametrize("cls", [(6, 3, 3), (5, 3, 2), (6, 2, 2), (5, 3, 0), (0, 3, 3), (3, 3, 2), (6, 3, 1), (5, 1, 1), (6, 0, 0)])
def test_df_single_class_digestion(lx, oracle, cls):
    """One class at a time (so that a failure names the kernel): gamma and J of a two-shell-type basis whose only
    off-diagonal pair class is (la, lb), against the oracle.  Contracted shells; no screening."""
    lxa, la, lb = cls
    rng = np.random.default_rng(1000 * lxa + 100 * la + 10 * lb)
    from helpers import table
    shells = []
    for l in (la, lb, la, lb, la):
        k = int(rng.integers(1, 3))
        z = np.exp(rng.uniform(np.log(0.2), np.log(3.0), k))
        shells.append((l, rng.uniform(0, 4, 3), z, rng.uniform(0.3, 1.0, k) * gen.prim_norm(z, l)))
    prim = table(shells)
    xs = []
    for _ in range(5):
        k = int(rng.integers(1, 3))
        z = np.exp(rng.uniform(np.log(0.2), np.log(3.0), k))
        xs.append((lxa, rng.uniform(0, 4, 3), z, rng.uniform(0.3, 1.0, k) * gen.prim_norm(z, lxa)))
    aux = table(xs)
    pairs = np.array([[0, 1], [2, 3], [2, 1], [4, 3], [0, 3], [4, 1]], np.int32)    # all of class (la, lb)
    D = rng.normal(size=(prim.nbf, prim.nbf))
    D = D + D.T
    d = rng.normal(size=aux.nbf)
    g_ref, J_ref, nsets, _ = oracle.df_gamma_J(aux, prim, pairs, None, None, 0.0, D=D, d=d)
    sched, gamma, J = _gpu_df(lx, aux, prim, pairs, None, None, 0.0, D, d)
    assert sched.num_sets == nsets
    eg, eJ = _relerr(gamma, g_ref), _relerr(J, J_ref)
    assert eg <= TOL_DF and eJ <= TOL_DF, (lx.lx_kernel_family(*cls), eg, eJ)


def test_df_config4_full_screened(lx, oracle):
    """BASELINE.json configs[3] as stated: 64-atom cluster, 960 AO x 6 784 Cartesian DFAO, all 73 920 unique shell
    pairs, Schwarz screening at 1e-12 with the oracle's factors.  The oracle evaluates EVERY surviving shell-set
    (22 M sets, long double); gamma and J are compared in full."""
    c4 = gen.config4()
    aux, prim, pairs = c4["aux"], c4["prim"], c4["pair_idx"]
    assert (prim.nbf, aux.nbf, len(pairs), aux.nshell) == (960, 6784, 73920, 1344)
    qx, qp = oracle.schwarz_aux(aux), oracle.schwarz_pair(prim, pairs)
    g_ref, J_ref, nsets, nints = oracle.df_gamma_J(aux, prim, pairs, qx, qp, c4["tau"], D=c4["D"], d=c4["d"])
    sched, gamma, J = _gpu_df(lx, aux, prim, pairs, qx, qp, c4["tau"], c4["D"], c4["d"])
    assert sched.num_sets == nsets and sched.num_integrals == nints          # identical screening: bit-exact counts
    assert 0.1 < nsets / (len(pairs) * aux.nshell) < 0.5                     # the screen does remove most sets
    eg, eJ = _relerr(gamma, g_ref), _relerr(J, J_ref)
    print(f"config 4: {nsets} sets, {nints} integrals; rel. Frobenius error gamma {eg:.2e}, J {eJ:.2e}")
    assert eg <= TOL_DF and eJ <= TOL_DF, (eg, eJ)
    assert abs(gamma @ c4["d"] - np.sum(J * c4["D"])) <= 1e-10 * abs(gamma @ c4["d"])


def test_df_config5_sampled(lx, oracle):
    """BASELINE.json configs[4] as stated: 256-atom cluster, nbf 8 960, naux 54 016 (Cartesian), 3 278 080 unique
    shell pairs, Schwarz 1e-12, integral-direct.  The GPU runs the WHOLE pass (both contractions over every
    surviving shell-set); the oracle evaluates the sampled outputs SURVEY.md §8(d) names — gamma for seeded aux
    shells (of every L) summed over ALL surviving pairs, J blocks for 2 048 seeded pairs summed over ALL surviving
    aux shells — and the run-time identity sum_X gamma_X d_X = sum_ab J_ab D_ab ties the rest together."""
    c5 = gen.config5()
    aux, prim, pairs = c5["aux"], c5["prim"], c5["pair_idx"]
    assert (prim.nbf, aux.nbf, len(pairs), aux.nshell) == (8960, 54016, 3278080, 7424)
    qx, qp = oracle.schwarz_aux(aux), oracle.schwarz_pair(prim, pairs)
    tau = c5["tau"]
    rng = np.random.default_rng(55)
    # aux sample: 3 shells of every L = 0..6 (the single i shell per atom included), 21 shells
    x_sel = np.sort(np.concatenate([rng.choice(np.nonzero(aux.L == l)[0], 3, replace=False) for l in range(7)])).astype(np.int32)
    # pair sample: 2 048 pairs among those with at least one surviving aux shell, every (la, lb) class present
    alive = np.nonzero(qp * qx.max() >= tau)[0]
    p_sel = rng.choice(alive, 2048 - 64, replace=False)
    La, Lb = prim.L[pairs[alive, 0]], prim.L[pairs[alive, 1]]
    extra = [rng.choice(alive[(La == 3) & (Lb == lb)], 16, replace=False) for lb in range(4)]
    p_sel = np.unique(np.concatenate([p_sel] + extra)).astype(np.int32)
    g_ref, _, _, _ = oracle.df_gamma_J(aux, prim, pairs, qx, qp, tau, D=c5["D"], x_sel=x_sel)
    _, J_ref, _, _ = oracle.df_gamma_J(aux, prim, pairs, qx, qp, tau, d=c5["d"], p_sel=p_sel)
    nsets_ref = int(np.sum(np.outer(qp, qx) >= tau)) if len(qp) * len(qx) < 1 << 24 else \
        sum(int(np.sum(qp[i:i + 65536, None] * qx[None, :] >= tau)) for i in range(0, len(qp), 65536))
    sched, gamma, J = _gpu_df(lx, aux, prim, pairs, qx, qp, tau, c5["D"], c5["d"])
    assert sched.num_sets == nsets_ref                                       # identical screening decisions
    # the GPU-made Schwarz factors (what bench.py uses) against the oracle's, all 3.3 M pairs
    gx, gp = lx.lx_schwarz_aux_host(lx.HostShells(aux)), lx.lx_schwarz_pair_host(lx.HostShells(prim), pairs)
    big = qp >= 1e-30
    eq = max(float(np.max(np.abs(gx - qx) / qx)), float(np.max(np.abs(gp[big] - qp[big]) / qp[big])))
    nsets_g = sum(int(np.sum(gp[i:i + 65536, None] * gx[None, :] >= tau)) for i in range(0, len(gp), 65536))
    print(f"config 5: GPU Schwarz factors rel. error {eq:.2e}; surviving sets oracle {nsets_ref}, GPU factors {nsets_g}")
    assert eq <= 1e-12 and abs(nsets_g - nsets_ref) <= 1e-9 * nsets_ref
    gsel = np.concatenate([np.arange(aux.bf_off[x], aux.bf_off[x + 1]) for x in x_sel])
    eg = _relerr(gamma[gsel], g_ref[gsel])
    mask = np.zeros((prim.nbf, prim.nbf), dtype=bool)
    for a, b in pairs[p_sel]:
        mask[prim.bf_off[a]:prim.bf_off[a + 1], prim.bf_off[b]:prim.bf_off[b + 1]] = True
        mask[prim.bf_off[b]:prim.bf_off[b + 1], prim.bf_off[a]:prim.bf_off[a + 1]] = True
    eJ = _relerr(J[mask], J_ref[mask])
    print(f"config 5: {sched.num_sets} sets, {sched.num_integrals} integrals; sampled rel. Frobenius error "
          f"gamma {eg:.2e} ({len(gsel)} entries), J {eJ:.2e} ({int(mask.sum())} entries)")
    assert np.isfinite(gamma).all() and np.isfinite(J).all()
    assert eg <= TOL_DF and eJ <= TOL_DF, (eg, eJ)
    lhs, rhs = float(gamma @ c5["d"]), float(np.sum(J * c5["D"]))
    assert abs(lhs - rhs) <= 1e-10 * np.linalg.norm(gamma) * np.linalg.norm(c5["d"]), (lhs, rhs)


@pytest.mark.parametrize("cls", [(2, 1, 1), (3, 2, 1), (4, 3, 1), (5, 3, 2), (6, 3, 3), (0, 0, 0)])
def test_df_ragged_prefixes(lx, oracle, cls):
    """The prefix map of a DF launch with RAGGED, short prefixes: hand-made screening factors (any positive numbers are legal
    inputs of the schedule) leave 0..6 aux shells per pair, so that one batch of 32 sets spans a dozen and more pairs and the
    pairs at the tail of a bucket have no set at all — the warp-cooperative pair search (find_pair_warp) and the run-wise J
    reduction against the oracle, which screens with the same numbers.  Set counts are bit-exact."""
    from helpers import table
    lxa, la, lb = cls
    rng = np.random.default_rng(900 + 100 * lxa + 10 * la + lb)
    nsh = 30
    shells = []
    for i in range(2 * nsh):
        l = la if i < nsh else lb
        k = int(rng.integers(1, 3))
        z = np.exp(rng.uniform(np.log(0.3), np.log(2.5), k))
        shells.append((l, rng.uniform(0, 5, 3), z, rng.uniform(0.3, 1.0, k) * gen.prim_norm(z, l)))
    prim = table(shells)
    xs = []
    for _ in range(6):
        z = np.exp(rng.uniform(np.log(0.3), np.log(2.5), 1))
        xs.append((lxa, rng.uniform(0, 5, 3), z, gen.prim_norm(z, lxa)))
    aux = table(xs)
    # every (la-shell, lb-shell) pair: 900 pairs of one class
    pairs = np.array([[i, nsh + j] for i in range(nsh) for j in range(nsh)], np.int32)
    qx = 10.0 ** -np.arange(6, dtype=np.float64)                      # 1, 0.1, ... 1e-5
    qp = 10.0 ** -rng.uniform(0.0, 8.0, len(pairs))
    tau = 1e-6
    D = rng.normal(size=(prim.nbf, prim.nbf))
    D = D + D.T
    d = rng.normal(size=aux.nbf)
    g_ref, J_ref, nsets, nints = oracle.df_gamma_J(aux, prim, pairs, qx, qp, tau, D=D, d=d)
    sched, gamma, J = _gpu_df(lx, aux, prim, pairs, qx, qp, tau, D, d)
    assert sched.num_sets == nsets and sched.num_integrals == nints
    assert 1.5 * len(pairs) < nsets < 4.5 * len(pairs)                # a few sets per pair on average
    eg, eJ = _relerr(gamma, g_ref), _relerr(J, J_ref)
    assert eg <= TOL_DF and eJ <= TOL_DF, (lx.lx_kernel_family(*cls), eg, eJ)
