"""N > 1 host logic (world_size 2, gloo) on CPU, and -- marked gpu -- the same split through the library: contiguous market shards keyed by the GLOBAL
market id reproduce the single-process run, with no data-path collective (SURVEY.md S8(e),
PAPER.md:105-107).  The per-shard compute stands in for one GPU's ks_create_ex(market_base) +
ks_run; here it is the oracle, which is keyed the same way.  Only the gather of the results and
the max-over-ranks of the timing (what bench.py does) use the process group."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_21784_b200.workloads import mix3_params, shard_markets, zi_params


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, case, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import ks_oracle
        M, L, A, S, seed, params = case
        base, count = shard_markets(M, rank, world)
        ids = np.arange(base, base + count, dtype=np.uint32)
        books, recs = ks_oracle.run_markets(params, L, A, seed, ids, S)
        # what bench.py does across ranks: max of the per-rank time, nothing on the data path
        t = torch.tensor([float(rank + 1)], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert t.item() == float(world)
        # gather the shard results on rank 0 (a host gather of M x (8L+128) bytes, off the hot path)
        gathered = [None] * world
        dist.all_gather_object(gathered, (base, count, books, recs))
        if rank == 0:
            gathered.sort(key=lambda g: g[0])
            assert [g[0] for g in gathered] == [shard_markets(M, r, world)[0] for r in range(world)]
            assert sum(g[1] for g in gathered) == M
            np.save(os.path.join(out_dir, "books.npy"), np.concatenate([g[2] for g in gathered]))
            np.save(os.path.join(out_dir, "recs.npy"), np.concatenate([g[3] for g in gathered]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("case", [
    (7, 64, 100, 30, 11, zi_params(8, 10)),            # odd M: shards of 4 and 3 markets
    (4, 256, 90, 20, 4, mix3_params()),
])
def test_two_rank_shards_equal_the_global_run(oracle, tmp_path, case):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), case, str(tmp_path)), nprocs=world, join=True)
    M, L, A, S, seed, params = case
    eb, er = oracle.run_markets(params, L, A, seed, np.arange(M, dtype=np.uint32), S)
    assert np.array_equal(np.load(tmp_path / "books.npy"), eb)
    assert np.array_equal(np.load(tmp_path / "recs.npy"), er)


def test_shard_markets_partitions_the_range():
    for M in (1, 2, 7, 64, 65536, 65537):
        for world in (1, 2, 3, 8):
            parts = [shard_markets(M, r, world) for r in range(world)]
            assert parts[0][0] == 0 and sum(c for _, c in parts) == M
            for (b0, c0), (b1, _) in zip(parts, parts[1:]):
                assert b1 == b0 + c0
            assert max(c for _, c in parts) - min(c for _, c in parts) <= 1


# ---- the same split through the LIBRARY: each rank = ks_create_ex(market_base = shard start) + ks_run.
# One GPU is enough: the ranks' kernels never wait on one another (there is no data-path collective),
# so two processes sharing cuda:0 exercise exactly what two GPUs would run.
def _gpu_worker(rank, world, port, case, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2606_21784_b200 import binding as ks
        ks.load()
        M, L, A, S, seed, params = case
        base, count = shard_markets(M, rank, world)
        sim = ks.KsSim(count, L, A, params, seed, market_base=base, device="cuda:0")
        sim.ks_run(S)
        books, recs = sim.books_to_host(), sim.stats_to_host()
        sim.ks_destroy()
        gathered = [None] * world
        dist.all_gather_object(gathered, (base, count, books, recs))
        if rank == 0:
            gathered.sort(key=lambda g: g[0])
            np.save(os.path.join(out_dir, "books.npy"), np.concatenate([g[2] for g in gathered]))
            np.save(os.path.join(out_dir, "recs.npy"), np.concatenate([g[3] for g in gathered]))
    finally:
        dist.destroy_process_group()


@pytest.mark.gpu
@pytest.mark.parametrize("case", [
    (7, 64, 100, 30, 11, zi_params(8, 10)),            # shards of 4 and 3 markets
    (301, 256, 1024, 40, 1, zi_params(16, 100)),       # the C2 shape cut 151 / 150: decoupled kernel on both ranks
    (5, 512, 700, 25, 4, mix3_params()),
])
def test_two_rank_shards_through_the_library(oracle, tmp_path, case):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from ks_testlib import oracle_rows
    world = 2
    mp.spawn(_gpu_worker, args=(world, _free_port(), case, str(tmp_path)), nprocs=world, join=True)
    M, L, A, S, seed, params = case
    eb, er = oracle_rows(oracle, params, L, A, seed, np.arange(M, dtype=np.uint32), S)
    assert np.array_equal(np.load(tmp_path / "books.npy"), eb)
    assert np.array_equal(np.load(tmp_path / "recs.npy"), er)
