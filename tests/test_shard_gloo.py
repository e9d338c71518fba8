"""Multi-rank host logic on CPU (-m "not gpu"): world size 2 over gloo. Each rank aligns its shard of
the pair list (with the CPU oracle standing in for the per-rank aligner; tests may use it), rank 0
stitches the results, and the stitched result must equal the unsharded one."""
import os
import socket

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from oracle import OracleScoring
from paper_1302_5507_b200 import shard
from paper_1302_5507_b200 import workloads as W


def oracle_align(b):
    return oracle.align_batch(b.reads_packed, b.read_off, b.read_len, b.wins_packed, b.win_off, b.win_len, b.pairs,
                              OracleScoring(), read_nmask=b.read_nmask, win_nmask=b.win_nmask, threads=1)


def test_pair_range_covers_everything():
    for P in (0, 1, 2, 7, 1000, 1001):
        for world in (1, 2, 3, 8):
            spans = [shard.pair_range(P, world, r) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == P
            assert all(spans[r][1] == spans[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1


def _worker(rank, world, port, n_pairs, out_path):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        batch = W.make_config(5, n_pairs=n_pairs, ref_bases=300_000)       # mixed lengths, N-masked windows
        got = shard.align_sharded(batch, oracle_align)
        if rank == 0:
            np.savez(out_path, **got)
        else:
            assert got is None
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_pairs", [401, 2])
def test_two_ranks_equal_unsharded(tmp_path, n_pairs):
    oracle.build()
    W.build()
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    out = str(tmp_path / "stitched.npz")
    mp.spawn(_worker, args=(2, port, n_pairs, out), nprocs=2, join=True)
    got = np.load(out)
    exp = oracle_align(W.make_config(5, n_pairs=n_pairs, ref_bases=300_000))
    for f in shard.FIELDS:
        a, b = np.asarray(getattr(exp, f)).astype(np.int64), got[f].astype(np.int64)
        assert a.shape == b.shape and np.array_equal(a, b), f
