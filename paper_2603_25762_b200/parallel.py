"""Multi-GPU plumbing of the QHap hot path: one process per GPU, replicas (or blocks) sharded across ranks.

Replicas are independent trajectories of the same graph ("multiple initial configurations are sampled in
parallel"; L118 "200 parallel samples") and blocks / connected components are independent problems, so
the bSB steps need NO per-step exchange.  The only exchange of the path is the final best-replica selection: 16 bytes
per rank (best cut, rank) are all-gathered, the winner (maximal cut, lowest rank on ties -- the same tie rule as inside
one GPU: lowest global replica index) broadcasts its n spin bytes.  Works on NCCL (GPU) and gloo (CPU tests).
"""
from __future__ import annotations

import os
from typing import Optional, Tuple

import torch
import torch.distributed as dist


def init_from_env(backend: Optional[str] = None) -> Tuple[int, int, int]:
    """(rank, world_size, local_rank) from torchrun's environment; initialises the process group when world_size > 1."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1 and not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend or ("nccl" if torch.cuda.is_available() else "gloo"), rank=rank, world_size=world)
    return rank, world, local


def replica_shard(replicas_total: int, rank: int, world: int) -> Tuple[int, int]:
    """[begin, end) of the global replica indices owned by `rank` (contiguous, sizes differ by at most 1)."""
    base, rem = divmod(int(replicas_total), int(world))
    begin = rank * base + min(rank, rem)
    return begin, begin + base + (1 if rank < rem else 0)


def block_shard(n_blocks: int, rank: int, world: int) -> list:
    """Blocks b == rank (mod world) -- independent problems, no exchange at all."""
    return list(range(rank, int(n_blocks), int(world)))


def rank_seed(seed: int, rank: int) -> int:
    """Seed of a rank's replica shard under weak scaling (every rank runs its own R replicas)."""
    return (int(seed) + 0x632BE59BD9B4E019 * int(rank)) & 0xFFFFFFFFFFFFFFFF


def plan_rank(replicas: int, seed: int, rank: int, world: int, scaling: str) -> dict:
    """What one rank runs.  "weak": every rank runs `replicas` replicas of the region from its own seed (per-GPU work
    fixed).  "strong": ONE seed's `replicas` replicas are split into contiguous slices; rank r starts the
    device-side seeded state at global replica `replica_begin`, so the union over the ranks is exactly the single-GPU run
    and the lowest rank that holds the maximal cut also holds the lowest global replica index."""
    if scaling == "weak" or world == 1:
        return dict(replicas=int(replicas), replica_begin=0, seed=rank_seed(seed, rank), replicas_total=int(replicas) * int(world))
    assert scaling == "strong", scaling
    b, e = replica_shard(replicas, rank, world)
    return dict(replicas=e - b, replica_begin=b, seed=int(seed), replicas_total=int(replicas))


def spawn_under_torchrun(n_gpus: int, script: str, argv: list) -> None:
    """`bench.py --gpus N` started as a plain process: re-exec it as N ranks (one per GPU) under torch.distributed.run with
    a loopback rendezvous.  Does not return."""
    import socket
    import sys
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={int(n_gpus)}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), script] + list(argv)
    os.execv(sys.executable, cmd)


def select_best_across_ranks(best_cut: torch.Tensor, best_spins: torch.Tensor) -> Tuple[torch.Tensor, torch.Tensor, int]:
    """All ranks return (global best cut [n_inst] int64, its spins [n] int8, winning rank of instance 0).

    best_cut: [n_inst] int64 of this rank, best_spins: [n] int8 of this rank (single instance: n_inst == 1; for several
    instances the spins of instance b are taken from the rank that wins b -- callers pass inst_ptr-free single instances
    here and shard multi-instance problems by block instead)."""
    if not dist.is_initialized() or dist.get_world_size() == 1:
        return best_cut, best_spins, 0
    world, rank = dist.get_world_size(), dist.get_rank()
    assert best_cut.numel() == 1, "replica sharding is used for single instances; shard multi-instance problems by block"
    mine = best_cut.reshape(1).to(torch.int64)
    allc = torch.empty(world, dtype=torch.int64, device=mine.device)
    dist.all_gather_into_tensor(allc, mine)
    host = allc.cpu()
    winner = int(torch.argmax(host))            # argmax returns the first maximal entry = lowest rank on ties
    for r in range(world):
        if int(host[r]) == int(host[winner]):
            winner = r
            break
    spins = best_spins.clone()
    dist.broadcast(spins, src=winner)
    return allc[winner:winner + 1].clone(), spins, winner
