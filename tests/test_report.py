"""NEXT-4 report layer: the paper's metrics from integer schedules, on CPU tensors,
against plain numpy; and combined over two gloo ranks."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2606_22327_b200 import report as R  # noqa: E402
from paper_2606_22327_b200 import traces as T  # noqa: E402


def _metrics_numpy(tr, finish, status=None):
    ptl, thr = [], []
    for j in range(tr.n_instances):
        lo, hi = int(tr.offsets[j]), int(tr.offsets[j + 1])
        if hi == lo or (status is not None and status[j] != 0):
            continue
        lat = (finish[lo:hi].astype(np.int64) - tr.arrival[lo:hi]) / tr.output[lo:hi].astype(np.float64)
        ptl.extend(lat.tolist())
        thr.append(tr.output[lo:hi].sum() / max(1, int(finish[lo:hi].max()) - int(tr.arrival[lo:hi].min())))
    ptl = np.sort(np.array(ptl))
    k = -(-95 * len(ptl) // 100)
    return {"requests": len(ptl), "mean_per_token_latency": float(ptl.mean()), "p95_per_token_latency": float(ptl[k - 1]),
            "token_throughput": float(np.mean(thr))}


def _call(tr, finish, status=None):
    t = lambda x, dt: torch.from_numpy(np.ascontiguousarray(x)).to(dt)
    return R.paper_metrics(t(tr.arrival, torch.int32), t(tr.output, torch.int32), t(finish, torch.int32),
                           t(tr.offsets, torch.int64), None if status is None else t(status, torch.int32))


def test_paper_metrics_match_numpy(oracle):
    parts = [T.random_small(40 + i, 5 + 9 * i, 9, 11, 30, a_hi=20) for i in range(7)] + [T.random_small(1, 0, 9, 11, 30)]
    tr = T.concat(parts, "rep", 30, 2, 8)
    r = oracle.simulate(tr, oracle.SVF)
    got, want = _call(tr, r.finish, r.status), _metrics_numpy(tr, r.finish, r.status)
    assert got["requests"] == want["requests"] == tr.n_requests
    for k in ("mean_per_token_latency", "p95_per_token_latency", "token_throughput"):
        assert abs(got[k] - want[k]) <= 1e-12 * max(1.0, abs(want[k])), k
    # unbounded memory: every request finishes o steps after it arrives: per-token latency exactly 1
    free = oracle.simulate(tr, oracle.SVF, M=10 ** 9)
    m = _call(tr, free.finish)
    assert m["mean_per_token_latency"] == 1.0 and m["p95_per_token_latency"] == 1.0
    # a rejected instance is left out
    st = r.status.copy(); st[2] = 16
    assert _call(tr, r.finish, st)["requests"] == tr.n_requests - parts[2].n_requests


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import svf_ref
        tr = T.config3(n_instances=3, n=80, lam=4.0, M=30_000, first_instance=3 * rank)
        r = svf_ref.simulate(tr, svf_ref.SJF)
        m = _call(tr, r.finish, r.status)
        if rank == 0:
            q.put(m)
    finally:
        dist.destroy_process_group()


def test_paper_metrics_over_two_ranks(oracle):
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    got = q.get()
    whole = T.config3(n_instances=6, n=80, lam=4.0, M=30_000)
    want = _metrics_numpy(whole, oracle.simulate(whole, oracle.SJF).finish)
    assert got["requests"] == want["requests"]
    for k in ("mean_per_token_latency", "p95_per_token_latency", "token_throughput"):
        assert abs(got[k] - want[k]) <= 1e-12 * max(1.0, abs(want[k])), k
