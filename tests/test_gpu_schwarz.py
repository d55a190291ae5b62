"""GPU Schwarz factors (lx_schwarz_aux_host / lx_schwarz_pair_host) against the
long-double oracle: relative error <= 1e-12, and the screening decisions they lead to (integer work: compared as
integers; the products that sit within 1e-12 of tau are counted and reported)."""
import numpy as np
import pytest

import lx_inputs as gen
from helpers import table

pytestmark = pytest.mark.gpu

TOL_Q = 1e-12


@pytest.fixture(scope="module")
def lx():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2210_03192_b200 import lx as _lx
    _lx.lx_init(0)
    return _lx


def _rel(got, ref):
    nz = ref > 0
    assert np.all(got[~nz] == 0)
    return float(np.max(np.abs(got[nz] - ref[nz]) / ref[nz])) if nz.any() else 0.0


def test_schwarz_every_class_contracted(lx, oracle):
    """Every aux L <= 6 and every primary pair class up to (4,4), contracted shells, distinct and coinciding centres."""
    rng = np.random.default_rng(5)
    shells, xs = [], []
    for l in range(5):
        for _ in range(2):
            k = int(rng.integers(1, 4))
            z = np.exp(rng.uniform(np.log(0.15), np.log(4.0), k))
            shells.append((l, rng.uniform(0, 3, 3), z, rng.uniform(0.3, 1.0, k) * gen.prim_norm(z, l)))
    for l in range(7):
        for k in (1, 2):
            z = np.exp(rng.uniform(np.log(0.1), np.log(10.0), k))
            xs.append((l, rng.uniform(0, 3, 3), z, rng.uniform(0.3, 1.0, k) * gen.prim_norm(z, l)))
    prim, aux = table(shells), table(xs)
    pairs = gen.unique_pairs(prim.nshell)
    pairs = np.concatenate([pairs, pairs[::7, ::-1]])                   # both orders of a pair
    qx = lx.lx_schwarz_aux_host(lx.HostShells(aux))
    qp = lx.lx_schwarz_pair_host(lx.HostShells(prim), pairs)
    ex, ep = _rel(qx, oracle.schwarz_aux(aux)), _rel(qp, oracle.schwarz_pair(prim, pairs))
    assert ex <= TOL_Q and ep <= TOL_Q, (ex, ep)


def test_schwarz_config4_and_decisions(lx, oracle):
    """Config 4 in full: factors to 1e-12 and IDENTICAL screening decisions at tau = 1e-12 (set count as integers)."""
    c4 = gen.config4()
    aux, prim, pairs = c4["aux"], c4["prim"], c4["pair_idx"]
    qx, qp = lx.lx_schwarz_aux_host(lx.HostShells(aux)), lx.lx_schwarz_pair_host(lx.HostShells(prim), pairs)
    rx, rp = oracle.schwarz_aux(aux), oracle.schwarz_pair(prim, pairs)
    assert _rel(qx, rx) <= TOL_Q
    big = rp >= 1e-30                                                   # below: underflowing overlaps, far under any tau
    assert _rel(qp[big], rp[big]) <= TOL_Q and np.all(qp[~big] < 1e-29)
    dec_g, dec_o = np.outer(qp, qx) >= c4["tau"], np.outer(rp, rx) >= c4["tau"]
    ndiff = int(np.sum(dec_g != dec_o))
    near = int(np.sum(np.abs(np.outer(rp, rx) / c4["tau"] - 1.0) < 1e-11))
    print(f"config 4: {int(dec_o.sum())} surviving sets; decisions that differ {ndiff}; products within 1e-11 of tau {near}")
    assert ndiff <= near
    sg = lx.Schedule(lx.HostShells(aux), lx.HostShells(prim), qx, qp, pairs, c4["tau"])
    assert abs(sg.num_sets - int(dec_o.sum())) <= near


def test_schwarz_empty_and_errors(lx):
    c = gen.config1(npair=2, nx=2)
    hp = lx.HostShells(c["prim"])
    assert len(lx.lx_schwarz_pair_host(hp, np.zeros((0, 2), np.int32))) == 0
    with pytest.raises(lx.LxError) as e:
        lx.lx_schwarz_pair_host(hp, np.array([[0, 99]], np.int32))
    assert e.value.status == lx.LX_EINVAL
