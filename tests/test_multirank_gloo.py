"""N>1 host logic on CPU: world_size-2 `gloo` ranks shard the packed triangle with clusco_partition_rows exactly as
the multi-GPU path does (contiguous row ranges, no data-path collective, results stay sharded).

No GPU here, so each rank fills ITS slice with the oracle's rows (tests may call the oracle); what is under test is
the library's partition arithmetic and the slice layout `clusco_crmsd_allpairs_ex` documents:
    slice r = out[idx(b[r], b[r]+1) : idx(b[r+1], b[r+1]+1)],  slices tile the triangle with no gap or overlap.
The gather at the end exists only to check that; the product path never gathers.
"""
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


def _packed_index(i, j, N):
    return i * (2 * N - i - 1) // 2 + (j - i - 1)


def _rank_main(rank, world, port, N, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        import paper_1302_4000_b200 as pkg
        from paper_1302_4000_b200 import workloads as wl

        ens = wl.make_config("C2", N=N)                         # same seeded ensemble on every rank (replicated)
        b = pkg.clusco_partition_rows(N, world)
        lo, hi = b[rank], b[rank + 1]
        P = N * (N - 1) // 2
        base = _packed_index(lo, lo + 1, N) if lo < N - 1 else P
        end = _packed_index(hi, hi + 1, N) if hi < N - 1 else P
        mine, _ = oracle.crmsd_rows(ens.coords, lo, hi) if hi > lo else (np.zeros(0), None)
        assert mine.size == end - base, (mine.size, base, end)

        # every rank learns every slice extent: they must tile [0, P) in rank order
        ext = [None] * world
        dist.all_gather_object(ext, (int(base), int(end)))
        assert ext[0][0] == 0 and ext[-1][1] == P
        assert all(a[1] == c[0] for a, c in zip(ext, ext[1:]))

        # timing plumbing of bench.py: max over ranks of a per-rank scalar
        t = torch.tensor([1.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert float(t) == float(world)

        # bench.py's own N > 1 code path (`--gpus N` = ONE ensemble, row-partitioned): the slice each rank times and
        # the per-rank record of the JSON line, driven here with gloo and host tensors
        import bench
        bounds, lo2, hi2, my_pairs = bench.rank_slice(pkg, N, world, rank)
        assert (lo2, hi2) == (lo, hi) and my_pairs == end - base
        job_ms, per_rank = bench.combine_ranks(torch, dist, world, bounds, 10.0 + rank, 9.0 + rank, my_pairs, "cpu")
        assert job_ms == 10.0 + world - 1 and sum(per_rank["pairs"]) == P
        assert per_rank["rows"][0][0] == 0 and per_rank["rows"][-1][1] == N
        assert abs(per_rank["slowest_over_fastest"] - (10.0 + world - 1) / 10.0) < 1e-12

        # check-only gather: concatenated slices == the full triangle
        parts = [None] * world
        dist.all_gather_object(parts, mine.astype(np.float64))
        if rank == 0:
            full, _ = oracle.crmsd_allpairs(ens.coords)
            got = np.concatenate(parts)
            q.put(("ok", bool(got.shape == full.shape and np.array_equal(got, full)), [int(x) for x in b]))
    except Exception as e:  # pragma: no cover - surfaced in the parent
        q.put(("error", repr(e), None))
        raise
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("N", [300, 129])
def test_two_ranks_shard_the_triangle(N):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, N, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(180)
    assert all(p.exitcode == 0 for p in procs), [p.exitcode for p in procs]
    kind, ok, b = q.get(timeout=10)
    assert kind == "ok" and ok, (kind, ok)
    assert b[0] == 0 and b[-1] == N and b[1] % 128 == 0
