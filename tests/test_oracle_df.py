"""Pins for the oracle Schwarz factors and DF contractions (SURVEY.md §8(c) pins)."""
import numpy as np

import lx_inputs as gen
from helpers import table


def _small_cluster(seed=7, natom=4):
    rng = np.random.default_rng(seed)
    prim, aux = gen._cluster(rng, natom, 6.0, gen._PRIM4, gen._AUX4[:3])
    nbf, naux = prim.nbf, aux.nbf
    Cm = rng.normal(0, 1 / np.sqrt(nbf), size=(nbf, nbf // 4))
    return prim, aux, Cm @ Cm.T, rng.normal(size=naux)


def test_schwarz_aux_s_primitive_closed_form(oracle):
    """(X|X) for an s primitive = 2 pi^{5/2} / (q^2 sqrt(2q))."""
    for q in [0.05, 0.8, 13.0]:
        aux = table([(0, [0.1, 0.2, 0.3], [q], [1.0])])
        ex = np.sqrt(2 * np.pi ** 2.5 / (q * q * np.sqrt(2 * q)))
        assert abs(oracle.schwarz_aux(aux)[0] - ex) < 1e-15 * ex


def test_schwarz_aux_contracted_p_closed_form(oracle):
    """Contracted p shell: (p_z|p_z) for two concentric p primitives q1, q2 follows from the s-s value
    [s|s](R) = 2 pi^{5/2}/(q1 q2 sqrt(q1+q2)) F_0(alpha R^2) by p_z = (1/2q) d/dC_z:
        (p_z|p_z') = -(1/(4 q1 q2)) d^2/dR_z^2 [s|s](R) at R = 0,   F_0(T) = 1 - T/3 + ...  ->  2 alpha / 3."""
    zs, cs = [0.7, 2.5], [0.6, 0.3]
    aux = table([(1, [0, 0, 0], zs, cs)])
    tot = 0.0
    for q1, c1 in zip(zs, cs):
        for q2, c2 in zip(zs, cs):
            al = q1 * q2 / (q1 + q2)
            tot += c1 * c2 * 2 * np.pi ** 2.5 / (q1 * q2 * np.sqrt(q1 + q2)) * (2 * al / 3) / (4 * q1 * q2)
    assert abs(oracle.schwarz_aux(aux)[0] - np.sqrt(tot)) < 1e-15 * np.sqrt(tot)


def test_schwarz_pair_ss_closed_form(oracle):
    """(ss|ss) diagonal for primitives: 2 pi^{5/2}/(p^2 sqrt(2p)) exp(-2 mu |AB|^2)  (R = P - P = 0, F_0(0) = 1)."""
    A, B, za, zb = np.array([0.0, 0.3, -0.2]), np.array([0.9, -0.5, 0.4]), 1.1, 0.6
    prim = table([(0, A, [za], [1.0]), (0, B, [zb], [1.0])])
    p = za + zb
    ex = np.sqrt(2 * np.pi ** 2.5 / (p * p * np.sqrt(2 * p)) * np.exp(-2 * za * zb / p * np.sum((A - B) ** 2)))
    assert abs(oracle.schwarz_pair(prim, [[0, 1]])[0] - ex) < 1e-15 * ex


def test_cauchy_schwarz_bound_holds(oracle):
    prim, aux, D, d = _small_cluster()
    pairs = gen.unique_pairs(prim.nshell)
    qx, qp = oracle.schwarz_aux(aux), oracle.schwarz_pair(prim, pairs)
    rng = np.random.default_rng(0)
    for ip in rng.choice(len(pairs), 25, replace=False):
        a, b = pairs[ip]
        for x in rng.choice(aux.nshell, 6, replace=False):
            v = oracle.eri3_batch(int(aux.L[x]), int(prim.L[a]), int(prim.L[b]), aux, prim, [x], [[a, b]])
            assert np.max(np.abs(v)) <= qx[x] * qp[ip] * (1 + 1e-12)


def test_gamma_J_against_stored_tensor(oracle):
    """γ and J from the stored oracle tensor with numpy contractions (definition)."""
    prim, aux, D, d = _small_cluster()
    pairs = gen.unique_pairs(prim.nshell)
    qx, qp = oracle.schwarz_aux(aux), oracle.schwarz_pair(prim, pairs)
    tau = 1e-6                                    # loose enough that some sets are actually screened
    gamma, J, nsets, nints = oracle.df_gamma_J(aux, prim, pairs, qx, qp, tau, D=D, d=d)
    g_ref = np.zeros(aux.nbf)
    J_ref = np.zeros((prim.nbf, prim.nbf))
    count = 0
    for ip, (a, b) in enumerate(pairs):
        for x in range(aux.nshell):
            if qx[x] * qp[ip] < tau:
                continue
            count += 1
            v = oracle.eri3_batch(int(aux.L[x]), int(prim.L[a]), int(prim.L[b]), aux, prim, [x], [[a, b]])[0, 0]
            sa = slice(prim.bf_off[a], prim.bf_off[a + 1])
            sb = slice(prim.bf_off[b], prim.bf_off[b + 1])
            sx = slice(aux.bf_off[x], aux.bf_off[x + 1])
            f = 2.0 if a != b else 1.0
            g_ref[sx] += f * np.einsum("xab,ab->x", v, D[sa, sb])
            blk = np.einsum("xab,x->ab", v, d[sx])
            J_ref[sa, sb] += blk
            if a != b:
                J_ref[sb, sa] += blk.T
    assert 0 < count < len(pairs) * aux.nshell and count == nsets
    assert np.linalg.norm(gamma - g_ref) < 1e-13 * np.linalg.norm(g_ref)
    assert np.linalg.norm(J - J_ref) < 1e-13 * np.linalg.norm(J_ref)
    assert np.allclose(J, J.T, rtol=0, atol=1e-14 * np.abs(J).max())
    # exact cross identity: sum_X gamma_X d_X = sum_ab J_ab D_ab (same unscreened sets on both sides)
    assert abs(gamma @ d - np.sum(J * D)) < 1e-12 * abs(gamma @ d)


def test_df_selection_is_partial_sum(oracle):
    prim, aux, D, d = _small_cluster(seed=9, natom=3)
    pairs = gen.unique_pairs(prim.nshell)
    qx, qp = oracle.schwarz_aux(aux), oracle.schwarz_pair(prim, pairs)
    g_all, J_all, _, _ = oracle.df_gamma_J(aux, prim, pairs, qx, qp, 1e-12, D=D, d=d)
    half = np.arange(len(pairs))[::2]
    rest = np.arange(len(pairs))[1::2]
    g1, J1, _, _ = oracle.df_gamma_J(aux, prim, pairs, qx, qp, 1e-12, D=D, d=d, p_sel=half)
    g2, J2, _, _ = oracle.df_gamma_J(aux, prim, pairs, qx, qp, 1e-12, D=D, d=d, p_sel=rest)
    assert np.linalg.norm(g1 + g2 - g_all) < 1e-14 * np.linalg.norm(g_all)
    assert np.linalg.norm(J1 + J2 - J_all) < 1e-14 * np.linalg.norm(J_all)


def test_schwarz_pair_against_bruteforce_quadrature(oracle):
    """Q_ab for La+Lb > 0 (only the one-sided Cauchy-Schwarz bound pinned it): (ab|ab) of one (p,s) and one
    (d,p) primitive pair by plain quadrature (helpers.bruteforce_pair_diagonal: independent of Boys, of the Hermite
    coefficients and of every recurrence); Q_ab^2 must equal the largest diagonal element."""
    from helpers import bruteforce_pair_diagonal
    comps = lambda l: [(x, y, l - x - y) for x in range(l, -1, -1) for y in range(l - x, -1, -1)]
    for (la, lb, A, B, za, zb) in [(1, 0, np.array([0.2, -0.1, 0.3]), np.array([-0.4, 0.5, 0.1]), 0.9, 1.4),
                                   (2, 1, np.array([0.0, 0.3, -0.2]), np.array([0.7, -0.4, 0.5]), 1.1, 0.6)]:
        prim = table([(la, A, [za], [1.0]), (lb, B, [zb], [1.0])])
        q = oracle.schwarz_pair(prim, [[0, 1]])[0]
        diag = [bruteforce_pair_diagonal(ca, cb, A, B, za, zb) for ca in comps(la) for cb in comps(lb)]
        assert min(diag) > 0
        assert abs(q * q - max(diag)) <= 2e-11 * max(diag), (q * q, max(diag))
