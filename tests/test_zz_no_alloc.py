"""lx_eri3_batch_static — the allocation-free entry point (include/lx.h): same result as lx_eri3_batch, primitive-pair data in
the library's static device array.  Collected LAST on purpose (the suite runs with pytest -x); passes alone in a fresh
process and after the other GPU tests.  Tolerance: the one of tests/test_gpu_parity.py (max-abs <= 1e-12 x batch max)."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import lx_inputs as gen  # noqa: E402

pytestmark = pytest.mark.gpu
TOL = 1e-12


@pytest.fixture(scope="module")
def lx():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2210_03192_b200 import lx as _lx
    _lx.lx_init(0)
    return _lx


def _case(lx, cls, npair, nx, seed):
    """Inputs of one call on the device + the existing path's result (lx_eri3_batch with a caller workspace)."""
    import torch
    cfg = gen.config2(*cls, npair=npair, nx=nx, seed=seed)            # primary K = 3 -> K_a K_b = 9
    aux, prim = lx.DeviceShells(cfg["aux"]), lx.DeviceShells(cfg["prim"])
    dx = torch.from_numpy(cfg["x_idx"]).cuda()
    dp = torch.from_numpy(cfg["pair_idx"]).cuda().contiguous()
    ref = lx.lx_eri3_batch(*cls, aux, prim, dx, dp, kmax=9)
    out = torch.full_like(ref, float("nan"))
    torch.cuda.synchronize()
    return dict(cls=cls, aux=aux, prim=prim, dx=dx, dp=dp, ref=ref, out=out)


def _compare(c):
    got, ref = c["out"].cpu().numpy(), c["ref"].cpu().numpy()
    assert np.isfinite(got).all()
    scale = np.max(np.abs(ref))
    err = np.max(np.abs(got - ref))
    assert err <= TOL * scale, (c["cls"], err, scale)


def test_static_matches_existing_path_two_calls_in_a_row(lx):
    """Two calls in a row (a large contracted class, then a smaller one of another kernel family that reuses the front of the
    array with the first call's records behind it, then the first again), each against lx_eri3_batch; no device memory is
    allocated between the first and the last call."""
    import torch
    a = _case(lx, (4, 2, 2), 300, 40, seed=21)      # chain kernel, 2 700 primitive pairs = 130 KB of the scratch
    b = _case(lx, (2, 1, 0), 37, 19, seed=22)       # team kernel, ragged tail
    c = _case(lx, (5, 1, 2), 64, 24, seed=23)       # mirrored class (la < lb), owner / lane kernels
    # warm-up: loads the kernels (CUDA lazy loading) and sets their attributes, as include/lx.h asks before a capture
    for k in (a, b, c):
        lx.lx_eri3_batch_static(*k["cls"], k["aux"], k["prim"], k["dx"], k["dp"], k["out"], 9)
        k["out"].fill_(float("nan"))
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for k in (a, b, a, c, b):
        lx.lx_eri3_batch_static(*k["cls"], k["aux"], k["prim"], k["dx"], k["dp"], k["out"], 9)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    assert free1 == free0, (free0, free1)            # nothing was allocated (or freed) on the device by the calls
    assert lx.lx_async_status() == lx.LX_OK
    for k in (a, b, c):
        _compare(k)


def test_static_limit_and_errors(lx):
    """Beyond the stated maximum the call refuses with LX_ELIMIT (and launches nothing); at the maximum it runs."""
    import torch
    assert lx.lx_static_scratch_bytes() == 4 << 20
    nmax = lx.lx_static_scratch_bytes() // 48                 # primitive pairs that fit: 87 381
    cfg = gen.config1(npair=64, nx=2)
    aux, prim = lx.DeviceShells(cfg["aux"]), lx.DeviceShells(cfg["prim"])
    dx = torch.from_numpy(cfg["x_idx"]).cuda()
    pairs = np.tile(cfg["pair_idx"], (nmax // 64 + 2, 1))
    out = torch.empty((nmax + 1) * 2 * 6 * 3 * 3, dtype=torch.float64, device="cuda")
    n0 = lx.lx_launch_count()
    dp = torch.from_numpy(np.ascontiguousarray(pairs[:nmax + 1])).cuda()
    with pytest.raises(lx.LxError) as e:
        lx.lx_eri3_batch_static(2, 1, 1, aux, prim, dx, dp, out, 1)
    assert e.value.status == lx.LX_ELIMIT and "LX_STATIC_SCRATCH_BYTES" in str(e.value)
    assert lx.lx_launch_count() == n0
    with pytest.raises(lx.LxError) as e:                       # the same pairs with a K stride of 2: twice the bytes
        lx.lx_eri3_batch_static(2, 1, 1, aux, prim, dx, dp[:nmax // 2 + 1].contiguous(), out[:(nmax // 2 + 1) * 108], 2)
    assert e.value.status == lx.LX_ELIMIT
    # exactly at the limit: runs, and agrees with the existing path on the first and the last pair
    dpm = dp[:nmax].contiguous()
    o = out[:nmax * 108]
    lx.lx_eri3_batch_static(2, 1, 1, aux, prim, dx, dpm, o, 1)
    ref = lx.lx_eri3_batch(2, 1, 1, aux, prim, dx, dpm, kmax=1)
    torch.cuda.synchronize()
    got = o.view(ref.shape)
    scale = float(ref.abs().max())
    assert float((got[:64] - ref[:64]).abs().max()) <= TOL * scale
    assert float((got[-64:] - ref[-64:]).abs().max()) <= TOL * scale
    assert float((got - ref).abs().max()) <= TOL * scale
