"""The N>1 path on CPU: world_size-2 `gloo` processes run the host-side sharding logic of
`paper_2606_22327_b200.sharding` (shard by instance, no data-path collective).
Each rank simulates ITS shard with the CPU oracle (the GPU is not needed to check the
partitioning and the report reductions); the gathered per-instance totals must equal the
oracle's run over the whole batch, the time reduction must be the max and the work the sum."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_22327_b200 import sharding as S  # noqa: E402
from paper_2606_22327_b200 import traces as T  # noqa: E402


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, mode, per_rank, total, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import svf_ref
        if mode == "weak":
            lo, hi = S.weak_shard(rank, per_rank)
        else:
            lo, hi = S.strong_shard(total, rank, world)
        batch = T.config3(n_instances=hi - lo, n=60, lam=4.0, M=40_000, first_instance=lo)
        res = svf_ref.simulate(batch, svf_ref.SVF)
        tel = S.gather_per_instance(torch.from_numpy(res.total_latency))
        dec = S.gather_per_instance(torch.from_numpy(res.decisions))
        times, counts = S.reduce_report([10.0 + rank, 5.0 - rank], [batch.request_steps, hi - lo])
        if rank == 0:
            q.put((tel.numpy(), dec.numpy(), times, counts))
    finally:
        dist.destroy_process_group()


def _run(mode, per_rank=0, total=0, world=2):
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, mode, per_rank, total, q)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    return q.get()


@pytest.mark.timeout(300)
def test_weak_sharding_two_ranks_matches_whole_batch(oracle):
    tel, dec, times, counts = _run("weak", per_rank=5)
    whole = T.config3(n_instances=10, n=60, lam=4.0, M=40_000)
    ref = oracle.simulate(whole, oracle.SVF)
    assert np.array_equal(tel, ref.total_latency)
    assert np.array_equal(dec, ref.decisions)
    assert times == [11.0, 5.0]                       # max over ranks
    assert counts == [float(whole.request_steps), 10.0]  # summed over ranks


@pytest.mark.timeout(300)
def test_strong_sharding_uneven_split(oracle):
    tel, dec, _, counts = _run("strong", total=7)
    whole = T.config3(n_instances=7, n=60, lam=4.0, M=40_000)
    ref = oracle.simulate(whole, oracle.SVF)
    assert np.array_equal(tel, ref.total_latency)
    assert np.array_equal(dec, ref.decisions)
    assert counts[1] == 7.0


def test_shards_are_disjoint_and_cover():
    for n in (0, 1, 5, 8, 4096, 4097):
        for w in (1, 2, 3, 8):
            r = [S.strong_shard(n, k, w) for k in range(w)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(w - 1))
            sizes = [hi - lo for lo, hi in r]
            assert max(sizes) - min(sizes) <= 1
    assert S.weak_shard(3, 4096) == (3 * 4096, 4 * 4096)
    with pytest.raises(ValueError):
        S.strong_shard(4, 2, 2)


def test_single_process_is_the_identity():
    x = torch.arange(5, dtype=torch.int64)
    assert torch.equal(S.gather_per_instance(x), x)
    assert S.reduce_report([1.5], [2.0]) == ([1.5], [2.0])
    assert S.world() == (0, 1)
