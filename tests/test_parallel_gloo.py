"""N > 1 host logic of the path on CPU: two processes over gloo.

The bSB steps need no exchange; the only collective is the final best-replica selection across ranks.  These tests run
parallel.select_best_across_ranks with world_size 2 on CPU tensors and check the sharding helpers.
"""
from __future__ import annotations

import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2603_25762_b200 import parallel


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, cuts, n: int, out_dir: str):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    r, w, _ = parallel.init_from_env(backend="gloo")
    assert (r, w) == (rank, world) and dist.get_backend() == "gloo"
    spins = torch.full((n,), 1 if rank % 2 == 0 else -1, dtype=torch.int8)
    spins[rank] = -spins[rank]                                    # make every rank's vector distinct
    best, win_spins, winner = parallel.select_best_across_ranks(torch.tensor([cuts[rank]], dtype=torch.int64), spins)
    np.save(os.path.join(out_dir, f"r{rank}.npy"), np.concatenate([[int(best[0]), winner], win_spins.numpy().astype(np.int64)]))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("cuts,expect", [([5, 9], 1), ([9, 5], 0), ([7, 7], 0), ([-3, -8], 0)])
def test_select_best_across_two_ranks(tmp_path, cuts, expect):
    n, world = 16, 2
    mp.spawn(_worker, args=(world, _free_port(), cuts, n, str(tmp_path)), nprocs=world, join=True)
    got = [np.load(tmp_path / f"r{r}.npy") for r in range(world)]
    assert np.array_equal(got[0], got[1]), "all ranks must end with the same winner"
    assert got[0][0] == max(cuts) and got[0][1] == expect         # ties -> lowest rank (= lowest global replica index)
    exp_spins = np.full(n, 1 if expect % 2 == 0 else -1)
    exp_spins[expect] = -exp_spins[expect]
    assert np.array_equal(got[0][2:], exp_spins)


def _rank_logic_worker(rank: int, world: int, port: int, R: int, n: int, scaling: str, out_dir: str):
    """bench.py's rank logic end to end on CPU tensors: plan_rank -> (stand-in for the solve: a cut per GLOBAL replica id and
    seed, spins that encode them) -> local best (lowest index on ties) -> select_best_across_ranks."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    r, w, _ = parallel.init_from_env(backend="gloo")
    plan = parallel.plan_rank(R, 20260001, r, w, scaling)
    gids = np.arange(plan["replica_begin"], plan["replica_begin"] + plan["replicas"], dtype=np.int64)
    cuts = _fake_cuts(plan["seed"], gids)
    lb = int(np.flatnonzero(cuts == cuts.max())[0]) if len(cuts) else 0
    best = torch.tensor([int(cuts[lb]) if len(cuts) else -(1 << 60)], dtype=torch.int64)
    spins = torch.from_numpy(_fake_spins(plan["seed"], int(gids[lb]) if len(gids) else -1, n))
    cut, win_spins, winner = parallel.select_best_across_ranks(best, spins)
    np.save(os.path.join(out_dir, f"r{rank}.npy"), np.concatenate([[int(cut[0]), winner, plan["replicas"], plan["replica_begin"]],
                                                                     win_spins.numpy().astype(np.int64)]))
    dist.barrier()
    dist.destroy_process_group()


def _fake_cuts(seed: int, gids: np.ndarray) -> np.ndarray:
    return ((gids * 2654435761 + (seed % 1000003)) % 97).astype(np.int64)          # many ties on purpose


def _fake_spins(seed: int, gid: int, n: int) -> np.ndarray:
    return np.where((np.arange(n) + gid + seed % 7) % 3 == 0, 1, -1).astype(np.int8)


@pytest.mark.parametrize("scaling", ["strong", "weak"])
def test_bench_rank_logic_two_ranks(tmp_path, scaling):
    R, n, world, seed = 37, 24, 2, 20260001
    mp.spawn(_rank_logic_worker, args=(world, _free_port(), R, n, scaling, str(tmp_path)), nprocs=world, join=True)
    got = [np.load(tmp_path / f"r{r}.npy") for r in range(world)]
    assert np.array_equal(got[0][:2], got[1][:2]) and np.array_equal(got[0][4:], got[1][4:])
    if scaling == "strong":
        # the union over the ranks is the single-GPU run: same best cut, and the spins of the LOWEST global replica holding it
        assert got[0][2] + got[1][2] == R and got[0][3] == 0 and got[1][3] == got[0][2]
        cuts = _fake_cuts(seed, np.arange(R, dtype=np.int64))
        gbest = int(np.flatnonzero(cuts == cuts.max())[0])
        assert got[0][0] == cuts.max() and got[0][1] == (0 if gbest < got[0][2] else 1)
        assert np.array_equal(got[0][4:], _fake_spins(seed, gbest, n))
    else:
        assert got[0][2] == got[1][2] == R and got[0][3] == got[1][3] == 0
        per_rank = [_fake_cuts(parallel.rank_seed(seed, r), np.arange(R, dtype=np.int64)).max() for r in range(world)]
        assert got[0][0] == max(per_rank) and got[0][1] == int(np.argmax(per_rank))


def test_shards_partition_the_work():
    for total, world in [(1024, 8), (10, 3), (2, 4), (0, 2)]:
        spans = [parallel.replica_shard(total, r, world) for r in range(world)]
        assert spans[0][0] == 0 and spans[-1][1] == total
        assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
        sizes = [e - b for b, e in spans]
        assert max(sizes) - min(sizes) <= 1
    for n_blocks, world in [(47, 8), (3, 4), (0, 2)]:
        owned = sorted(b for r in range(world) for b in parallel.block_shard(n_blocks, r, world))
        assert owned == list(range(n_blocks))
    seeds = {parallel.rank_seed(20260001, r) for r in range(8)}
    assert len(seeds) == 8 and parallel.rank_seed(20260001, 0) == 20260001


def test_single_process_is_identity():
    cut, spins = torch.tensor([11], dtype=torch.int64), torch.ones(4, dtype=torch.int8)
    c, s, w = parallel.select_best_across_ranks(cut, spins)
    assert c is cut and s is spins and w == 0
