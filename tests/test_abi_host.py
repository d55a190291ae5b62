"""CPU-side checks of the boundary: liblx.so loads, exports every symbol include/lx.h declares, and the entry points
that need no device behave as documented (no compute call is made here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lx():
    from paper_2210_03192_b200 import build
    build.build()
    from paper_2210_03192_b200 import lx as _lx
    return _lx


def _declared():
    src = open(os.path.join(ROOT, "include", "lx.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lx_[a-zA-Z0-9_]+)\s*\(", src)))


def test_header_symbols_exported(lx):
    names = _declared()
    assert {"lx_eri3_batch", "lx_df_gamma", "lx_df_J", "lx_schedule_create", "lx_init"} <= set(names)
    for n in names:
        assert hasattr(lx._lib, n), f"{n} declared in include/lx.h but not exported by liblx.so"
    assert set(lx.EXPORTS) == set(names), set(lx.EXPORTS) ^ set(names)


def test_not_initialised_and_strerror(lx):
    # no lx_init on this box (no device): every compute entry point must refuse, not crash
    assert lx._lib.lx_eri3_batch(2, 1, 1, None, None, None, 1, None, 1, None, None, 0, None) == lx.LX_ENOTINIT
    assert lx._lib.lx_boys(None, 1, 3, None, None) == lx.LX_ENOTINIT
    h = C.c_void_p()
    assert lx._lib.lx_schedule_create(None, None, None, None, None, 0, C.c_double(0.0), C.byref(h)) == lx.LX_ENOTINIT
    assert lx._lib.lx_metric_2c(None, None, 0) == lx.LX_ENOTINIT
    assert lx._lib.lx_fit_solve(None, 0, 0, None, 0, 0) == lx.LX_ENOTINIT
    for code in (0, -1, -2, -3, -5, -6, -7):
        assert len(lx.lx_strerror(code)) > 0 and lx.lx_strerror(code) != "unknown status"
    assert lx.lx_strerror(-99) == "unknown status"
    assert "sm_100a" in lx.lx_version()


def test_workspace_bytes_and_family(lx):
    assert lx.lx_eri3_workspace_bytes(2, 1, 1, 32, 64, 1) >= 64 * 6 * 8
    assert lx.lx_eri3_workspace_bytes(4, 2, 2, 256, 1024, 9) >= 1024 * 9 * 6 * 8
    assert lx.lx_eri3_workspace_bytes(0, 0, 0, 0, 0, 0) > 0
    assert lx.lx_kernel_family(7, 0, 0) == "" and lx.lx_kernel_family(0, 5, 0) == ""
    for lxa in range(7):
        for la in range(5):
            for lb in range(5):
                assert lx.lx_kernel_family(lxa, la, lb) in ("team", "chain", "owner", "lane", "group", "slab")
                assert lx.lx_kernel_family(lxa, la, lb) == lx.lx_kernel_family(lxa, lb, la)
                for k in (0, 1, 4, 9, 100):
                    assert lx.lx_kernel_family_k(lxa, la, lb, k) in ("team", "chain", "owner", "lane", "group", "slab")
                assert lx.lx_kernel_family_k(lxa, la, lb, 0) == lx.lx_kernel_family(lxa, la, lb)
    # K-aware dispatch: config 2 (K = 9) keeps the round-1 kernels, weakly contracted launches of the chain
    # classes and every launch of the Lx = 5, 6 classes with La+Lb >= 3 go to the owner kernel, La+Lb = 5, 6 to the slab kernel
    assert lx.lx_kernel_family_k(4, 2, 2, 9) == "chain" and lx.lx_kernel_family_k(4, 2, 2, 1) == "owner"
    assert lx.lx_kernel_family_k(2, 1, 1, 1) == "team" and lx.lx_kernel_family_k(3, 2, 1, 2) == "owner"
    assert lx.lx_kernel_family_k(6, 2, 2, 1) == "owner" and lx.lx_kernel_family_k(5, 2, 2, 25) == "owner"
    assert lx.lx_kernel_family_k(5, 1, 1, 4) == "owner" and lx.lx_kernel_family_k(5, 1, 1, 9) == "lane"
    assert lx.lx_kernel_family_k(6, 3, 3, 1) == "slab" and lx.lx_kernel_family_k(4, 4, 4, 1) == "group" and lx.lx_kernel_family_k(1, 3, 2, 1) == "owner"
    assert lx.lx_kernel_family_k(4, 3, 2, 9) == "owner" and lx.lx_kernel_family_k(0, 3, 3, 1) == "group"


def test_shard_pairs_partition():
    from paper_2210_03192_b200 import shard
    import lx_inputs as gen
    rng = np.random.default_rng(0)
    prim, _ = gen._cluster(rng, 4, 8.0, gen._PRIM4, gen._AUX4)
    pairs = gen.unique_pairs(prim.nshell)
    cost = shard.pair_cost(prim.L, prim.K, pairs)
    for world in (1, 2, 3, 8):
        for c in (None, cost):
            parts = [shard.shard_pairs(pairs, r, world, c) for r in range(world)]
            allrows = np.concatenate(parts)
            assert len(allrows) == len(pairs) and len(np.unique(allrows)) == len(pairs)
            if c is not None and world > 1:
                tot = np.array([cost[p].sum() for p in parts])
                assert tot.max() - tot.min() <= cost.max() * 1.0001 + 1e-9
    with pytest.raises(ValueError):
        shard.shard_pairs(pairs, 2, 2)


def test_solid_matrix_matches_oracle(lx):
    """Row a6: the library builds its Cartesian -> solid-harmonic matrices by the recurrences of the regular solid
    harmonics, the oracle by the closed formula; the two independent routes must agree for every l (host only)."""
    from oracle import solid
    for l in range(7):
        got = lx.lx_solid_matrix(l)
        ref = solid.solid_matrix(l)
        assert got.shape == ref.shape == (2 * l + 1, (l + 1) * (l + 2) // 2)
        assert np.max(np.abs(got - ref)) <= 1e-13 * np.max(np.abs(ref)), l
    with pytest.raises(lx.LxError):
        lx.lx_solid_matrix(7)
