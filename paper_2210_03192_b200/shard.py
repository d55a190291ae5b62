"""Multi-GPU sharding of the hot path.

Every shell-set is independent, so the path shards over the shell-PAIR list with no data-path collective for
``lx_eri3_batch`` (outputs are disjoint) and for J (the J blocks of different pairs are disjoint); γ needs one
all-reduce of naux doubles (each rank holds the partial sum over its pairs).  D and d are replicated.

Host logic only: index arithmetic and ``torch.distributed`` calls; no integral arithmetic.
"""
import numpy as np


def pair_cost(L, K, pair_idx):
    """Relative cost of a shell pair: primitive pairs × Cartesian components (a proxy that balances classes)."""
    p = np.asarray(pair_idx, dtype=np.int64).reshape(-1, 2)
    L = np.asarray(L, dtype=np.int64)
    K = np.asarray(K, dtype=np.int64)
    nc = (L + 1) * (L + 2) // 2
    return (K[p[:, 0]] * K[p[:, 1]] * nc[p[:, 0]] * nc[p[:, 1]]).astype(np.float64)


def shard_pairs(pair_idx, rank, world, cost=None):
    """Rows of ``pair_idx`` owned by ``rank``: a deterministic, cost-balanced, class-interleaved partition.

    Without ``cost``: round-robin (row i → rank i % world).  With ``cost``: pairs sorted by decreasing cost are dealt
    in groups of ``world`` in serpentine order (0..w-1, w-1..0, ...), so every rank sees every class and the totals
    stay close.  Returns the sorted row indices; the union over ranks is exactly ``range(npair)`` and the shards are
    disjoint."""
    p = np.asarray(pair_idx).reshape(-1, 2)
    n = len(p)
    if world <= 1:
        return np.arange(n, dtype=np.int64)
    if not 0 <= rank < world:
        raise ValueError("rank out of range")
    if cost is None:
        return np.arange(rank, n, world, dtype=np.int64)
    cost = np.asarray(cost, dtype=np.float64)
    if cost.shape != (n,):
        raise ValueError("cost must have one entry per pair")
    order = np.argsort(-cost, kind="stable")
    # groups of `world` consecutive pairs (similar cost) are dealt in a serpentine order: O(n), deterministic
    owner = np.empty(n, dtype=np.int64)
    pos = np.arange(n)
    rnd, k = pos // world, pos % world
    owner[order] = np.where(rnd % 2 == 0, k, world - 1 - k)
    return np.nonzero(owner == rank)[0].astype(np.int64)


def allreduce_gamma(gamma):
    """Sum the per-rank partial γ in place (the one collective of the DF path; naux doubles)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(gamma, op=dist.ReduceOp.SUM)
    return gamma


def allreduce_J(J):
    """Replicate J: the per-rank J hold disjoint blocks (zeros elsewhere), so a sum assembles the matrix."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(J, op=dist.ReduceOp.SUM)
    return J
