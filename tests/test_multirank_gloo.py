"""N > 1 host logic on CPU (gloo, world_size 2): the pair-list partition of SURVEY.md §8(e) plus the one collective
of the DF path.  Each rank evaluates its shard of shell pairs — here with the oracle standing in for the device
kernels, which need a GPU — and the assembled γ / J / eri3 blocks must equal the single-rank result."""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      OMP_NUM_THREADS="2")
    import torch
    import torch.distributed as dist
    import lx_inputs as gen
    import oracle
    from paper_2210_03192_b200 import shard
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rng = np.random.default_rng(11)
        prim, aux = gen._cluster(rng, 3, 6.0, gen._PRIM4, gen._AUX4)
        pairs = gen.unique_pairs(prim.nshell)
        D = rng.normal(size=(prim.nbf, prim.nbf)); D = D + D.T
        d = rng.normal(size=aux.nbf)
        qx, qp = oracle.schwarz_aux(aux), oracle.schwarz_pair(prim, pairs)
        rows = shard.shard_pairs(pairs, rank, world, shard.pair_cost(prim.L, prim.K, pairs))
        g, J, nsets, _ = oracle.df_gamma_J(aux, prim, pairs[rows], qx, qp[rows], 1e-12, D=D, d=d)
        g_t, J_t = torch.from_numpy(g.copy()), torch.from_numpy(J.copy())
        shard.allreduce_gamma(g_t)
        shard.allreduce_J(J_t)
        n_t = torch.tensor([nsets], dtype=torch.int64)
        dist.all_reduce(n_t)
        # eri3: disjoint output rows, gathered without arithmetic
        p11 = np.array([[3, 4], [4, 3], [3, 3], [4, 4], [9, 10]], np.int32)   # (p,p) pairs of the cluster
        rows11 = shard.shard_pairs(p11, rank, world)
        xs = np.nonzero(aux.L == 2)[0][:3].astype(np.int32)
        part = oracle.eri3_batch(2, 1, 1, aux, prim, xs, p11[rows11])
        full = torch.zeros((len(p11),) + part.shape[1:], dtype=torch.float64)
        full[torch.from_numpy(rows11)] = torch.from_numpy(part)
        dist.all_reduce(full)
        if rank == 0:
            g_ref, J_ref, n_ref, _ = oracle.df_gamma_J(aux, prim, pairs, qx, qp, 1e-12, D=D, d=d)
            e_ref = oracle.eri3_batch(2, 1, 1, aux, prim, xs, p11)
            np.savez(out, g=g_t.numpy(), J=J_t.numpy(), n=n_t.numpy(), g_ref=g_ref, J_ref=J_ref, n_ref=n_ref,
                     e=full.numpy(), e_ref=e_ref)
    finally:
        dist.destroy_process_group()


def test_world2_pair_shards_reassemble(tmp_path, oracle):
    import torch.multiprocessing as mp
    out = str(tmp_path / "res.npz")
    port = _free_port()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    r = np.load(out)
    assert int(r["n"][0]) == int(r["n_ref"])                       # integer work: exact
    assert np.linalg.norm(r["g"] - r["g_ref"]) <= 1e-13 * np.linalg.norm(r["g_ref"])
    assert np.linalg.norm(r["J"] - r["J_ref"]) <= 1e-13 * np.linalg.norm(r["J_ref"])
    assert np.array_equal(r["e"], r["e_ref"])                     # disjoint blocks: bit-exact
