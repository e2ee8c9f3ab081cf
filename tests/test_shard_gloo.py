"""N > 1 path: a batch shards by sequence with no data-path collective.  World-size-2 gloo
run on CPU of the host logic in paper_1307_7820_b200/shard.py; the per-rank "fold" is the oracle here (tests
may use it), on a GPU rank it is Rna4r.fold_batch_host."""
import os
import socket

import numpy as np
import pytest

import oracle
import workloads
from paper_1307_7820_b200 import shard


def test_shard_indices_partition_and_balance():
    rs = np.random.RandomState(7)
    lens = rs.randint(0, 900, size=101)
    for world in (1, 2, 3, 8):
        parts = [shard.shard_indices(lens, world, r) for r in range(world)]
        allidx = np.concatenate(parts)
        assert sorted(allidx.tolist()) == list(range(len(lens)))          # a partition
        assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1
        work = [float(np.sum(lens[p].astype(np.float64) ** 3)) for p in parts]
        assert max(work) <= 1.35 * (sum(work) / world) + float(lens.max()) ** 3   # near-equal n^3 work
    with pytest.raises(ValueError):
        shard.shard_indices(lens, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        seqs, lens = workloads.random_sequences(21, 37, 0, 90)
        calls = []

        def fold_fn(my_seqs, my_lens):
            calls.append(len(my_seqs))
            assert [len(s) for s in my_seqs] == [int(x) for x in my_lens]
            return np.array([oracle.nussinov(s) for s in my_seqs], dtype=np.int32)

        out = shard.fold_batch_sharded(fold_fn, seqs, lens, world, rank, dist)
        dist.barrier()
        if rank == 0:
            want = np.array([oracle.nussinov(s) for s in seqs], dtype=np.int32)
            q.put(("ok", bool((out == want).all()), calls[0], len(seqs)))
        else:
            q.put(("other", out is None, calls[0], len(seqs)))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_batch_sharding():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    res = {r[0]: r for r in res}
    assert res["ok"][1] is True            # rank 0 holds every score, in the caller's order
    assert res["other"][1] is True         # the other rank returns nothing
    assert res["ok"][2] + res["other"][2] == res["ok"][3]   # every sequence folded exactly once
