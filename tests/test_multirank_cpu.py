"""world_size-2 gloo test of the multi-GPU host logic (CPU only): round sharding + gather.

The data path has no collective: each rank runs its own round slice; results are
gathered once.  Here the per-slice work is done by the oracle (no GPU on this box); what is under
test is shard.round_slice / weak_slice and that slicing the round space is bit-identical to one
run over the whole range (the property bits_mc_rounds guarantees through (seed, round) addressing).
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1208_3407_b200 import shard
from paper_1208_3407_b200 import workloads as W


def test_round_slice_partitions_the_range():
    for world in (1, 2, 3, 8):
        for total in (0, 1, 7, 100, 1001):
            got = []
            for r in range(world):
                first, n = shard.round_slice(r, world, total, round_begin=5)
                got += list(range(first, first + n))
            assert got == list(range(5, 5 + total))
    assert shard.weak_slice(3, 1000) == (3000, 1000)
    with pytest.raises(ValueError):
        shard.round_slice(2, 2, 10)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, which, total_rounds, out_path):
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = W.make_config(1)
    first, n = shard.round_slice(rank, world, total_rounds)
    obs, rc = oracle.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, which, w.mc_seed, first, n)
    # pad to equal length for all_gather, then rank 0 reassembles in round order
    width = -(-total_rounds // world)
    mine = torch.zeros(width + 2, dtype=torch.int64)
    mine[0], mine[1] = first, n
    mine[2:2 + n] = torch.from_numpy(rc.astype(np.int64))
    parts = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine)
    t_obs = torch.tensor([obs], dtype=torch.int64)
    dist.all_reduce(t_obs, op=dist.ReduceOp.MAX)
    assert int(t_obs.item()) == obs                      # every rank saw the same observed count
    if rank == 0:
        full = np.zeros(total_rounds, dtype=np.uint64)
        for p in parts:
            f, k = int(p[0]), int(p[1])
            full[f:f + k] = p[2:2 + k].numpy().astype(np.uint64)
        np.save(out_path, full)
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("which", [0, 1])
def test_two_ranks_gloo_round_sharding_matches_single_run(tmp_path, oracle_mod, which):
    total = 21                                           # odd: the ranks get 11 and 10 rounds
    out = str(tmp_path / "rc.npy")
    mp.spawn(_worker, args=(2, _free_port(), which, total, out), nprocs=2, join=True)
    w = W.make_config(1)
    _, ref = oracle_mod.mc_rounds(w.a_start, w.a_end, w.b_start, w.b_end, w.chrom_offsets, which, w.mc_seed, 0, total)
    assert np.array_equal(np.load(out), ref)
