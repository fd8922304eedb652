"""world_size-2 gloo test of the N > 1 plumbing bench.py uses (independent replicas, no
data-path collective): per-rank seeds differ, the job time is the max over ranks, the job rate is the sum of
the ranks' units over that time.  CPU only."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import workloads as wl
    from paper_2606_06742_b200 import ranks
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = wl.config0(n=40, p=3, L=2, V=2, seed=ranks.replica_seed(1001, rank))
    ms = 10.0 * (rank + 1)                      # rank 1 is the slow one
    job_ms = ranks.max_over_ranks(ms, dist)
    rate = ranks.whole_job_rate(w.B, ms, dist)
    dist.barrier()
    out.put((rank, float(w.X[0, 0]), w.B, job_ms, rate))
    dist.destroy_process_group()


def test_two_rank_replicas_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, x0, b0, ms0, rate0), (r1, x1, b1, ms1, rate1) = res
    assert (r0, r1) == (0, 1) and x0 != x1            # different data sets, same shape
    assert b0 == b1 == 2 * 3
    assert ms0 == ms1 == 20.0                         # max over ranks
    assert np.isclose(rate0, (b0 + b1) / 0.020) and rate0 == rate1


def test_single_process_is_identity():
    from paper_2606_06742_b200 import ranks
    assert ranks.max_over_ranks(3.5) == 3.5 and ranks.whole_job_rate(10, 500.0) == 20.0


def _shard_worker(rank, world, port, L, out):
    import torch.distributed as dist
    from paper_2606_06742_b200 import ranks
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    T, V = 2, 3
    full = np.arange(T * L * V, dtype=np.float64).reshape(T, L, V) * 0.5
    full_i = np.arange(T * L * V, dtype=np.int64).reshape(T, L, V)
    mine = ranks.lambda_slice(L, rank, world)
    got = ranks.gather_lambda_tables(full[:, mine], L, rank, world, dist)
    got_i = ranks.gather_lambda_tables(full_i[:, mine], L, rank, world, dist)
    out.put((rank, mine.tolist(), bool(np.array_equal(got, full)), bool(np.array_equal(got_i, full_i)),
             str(got_i.dtype)))
    dist.barrier()
    dist.destroy_process_group()


def test_column_sharding_gloo_ragged_slices():
    """lambda columns interleaved over ranks, loss tables gathered before the argmin.  L = 7 on
    two ranks: slices of 4 and 3 (padding path), every rank ends with the full table, integer table exact."""
    world, port, L = 2, _free_port(), 7
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_shard_worker, args=(r, world, port, L, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == [0, 2, 4, 6] and res[1][1] == [1, 3, 5]
    assert all(r[2] and r[3] and r[4] == "int64" for r in res)


def test_lambda_slice_partitions_the_grid():
    import pytest
    from paper_2606_06742_b200 import ranks
    for L, world in [(50, 8), (7, 2), (5, 5), (9, 1)]:
        parts = [ranks.lambda_slice(L, r, world) for r in range(world)]
        assert sorted(np.concatenate(parts).tolist()) == list(range(L))
        assert max(map(len, parts)) - min(map(len, parts)) <= 1
    with pytest.raises(ValueError):
        ranks.lambda_slice(3, 0, 4)
    one = np.ones((1, 9, 2))
    assert np.array_equal(ranks.gather_lambda_tables(one, 9, 0, 1), one)
