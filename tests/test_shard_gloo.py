"""World-size-2 gloo test (CPU) of the N>1 host logic: shard ranges tile the problem exactly, the
timing reduction is a max over ranks, and gathering per-rank column shards reproduces the full product."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import sys
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import oracle
    from paper_2606_21023_b200 import inputs
    from paper_2606_21023_b200.shard import shard_cols, shard_rows
    M, N, K = 37, 300, 96
    A = inputs.activations(M, K, seed=0)
    W = inputs.weights_f16(K, N, seed=0)
    # N-sharding: each rank owns a column range of W and of C (the oracle stands in for the GPU here)
    c0, c1 = shard_cols(N, world, rank)
    part = torch.from_numpy(oracle.gemm_f64(A, np.ascontiguousarray(W[:, c0:c1])))
    parts = [None] * world
    dist.all_gather_object(parts, (c0, c1, part))
    # M-sharding ranges
    rows = [None] * world
    dist.all_gather_object(rows, shard_rows(M, world, rank))
    # M-sharding as bench.py does it: rank r GENERATES exactly its rows of the global activation matrix (rows are regenerable from
    # (seed, row index)), runs the path on them, and the row blocks concatenate to the product over the global batch
    from paper_2606_21023_b200.shard import aggregate_throughput
    Mg = world * 16
    r0, r1 = shard_rows(Mg, world, rank)
    A_mine = inputs.activations(r1 - r0, K, seed=3, outliers=True, row0=r0)
    A_glob = inputs.activations(Mg, K, seed=3, outliers=True)
    mine_ok = np.array_equal(A_mine, A_glob[r0:r1])
    mparts = [None] * world
    dist.all_gather_object(mparts, (r0, oracle.gemm_f64(A_mine, W), mine_ok))
    if rank == 0:
        catm = np.concatenate([p[1] for p in sorted(mparts, key=lambda p: p[0])], axis=0)
        assert all(p[2] for p in mparts) and np.array_equal(catm, oracle.gemm_f64(A_glob, W))
        assert aggregate_throughput([5.0] * world, [1000.0, 2000.0][:world]) == 5.0 * world / max([1.0, 2.0][:world])
    # timing: max over ranks
    t = torch.tensor([10.0 + rank])
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    if rank == 0:
        full = oracle.gemm_f64(A, W)
        cat = np.concatenate([p[2].numpy() for p in sorted(parts, key=lambda p: p[0])], axis=1)
        q.put((np.array_equal(cat, full), [p[:2] for p in parts], rows, float(t.item())))
    dist.destroy_process_group()


def test_two_rank_sharding_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    same, cols, rows, tmax = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert same                                          # column shards concatenate to the full product, bit for bit
    assert cols == [(0, 256), (256, 300)]
    assert rows == [(0, 19), (19, 37)]
    assert tmax == 11.0


def test_shard_helpers():
    from paper_2606_21023_b200.shard import aggregate_throughput, shard_cols, shard_rows
    for M in (0, 1, 7, 2048):
        for w in (1, 2, 3, 8):
            r = [shard_rows(M, w, i) for i in range(w)]
            assert r[0][0] == 0 and r[-1][1] == M and all(r[i][1] == r[i + 1][0] for i in range(w - 1))
            assert max(e - b for b, e in r) - min(e - b for b, e in r) <= 1
    for N in (8, 128, 4096, 14336, 128256):
        for w in (1, 2, 4, 8):
            c = [shard_cols(N, w, i) for i in range(w)]
            assert c[0][0] == 0 and c[-1][1] == N and all(c[i][1] == c[i + 1][0] for i in range(w - 1))
            assert all(b % 128 == 0 or b == N for b, _ in c)
    assert aggregate_throughput([10, 10], [1000.0, 2000.0]) == 10.0
