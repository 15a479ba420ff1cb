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


# ---------------------------------------------------------------------------------------------
# NEXT-3: the constants of the stochastic analysis (PAPER.md 3.4, App. H) by hand values
# ---------------------------------------------------------------------------------------------
def test_stochastic_constants_hand_values():
    """mu = 1/2, theta = 2, E[s] = 3, lambda = 1, M = 100, p_max = 20 (alpha = 0.2), worked by hand:
    q^theta = 1/4, d = 2 (1/4) / (3/4) = 2/3, eps = d^2/2 = 2/9, O0 = 2 - 2/3 = 4/3, O1 = 2 + 2 = 4;
    E[vol] = 3*2 + 4 = 10 (Eq. 101); rho = 10 / (0.8 * 50) = 1/4; Thm 3.4: 1 + 2 / (0.8 * 0.5 * 0.75) = 23/3;
    Thm 3.5: 1 + 10 / (10 - 2/9) * 20/3 = 1 + (45/44)(20/3) = 86/11; W_exact = 1 * (1/2)/(1/4) * (3 + 4) = 14
    (Eq. 89), OPT >= max{2, 14/100} = 2."""
    c = R.stochastic_constants(mu=0.5, mean_s=3.0, lam=1.0, M=100.0, p_max=20.0, theta=2)
    want = {"alpha": 0.2, "E_vol": 10.0, "rho": 0.25, "thm34_bound": 23.0 / 3.0, "W_exact": 14.0, "opt_lower_bound": 2.0,
            "eps": 2.0 / 9.0, "O0": 4.0 / 3.0, "O1": 4.0, "thm35_bound": 86.0 / 11.0}
    for k, v in want.items():
        assert abs(c[k] - v) < 1e-12 * max(1.0, abs(v)), (k, c[k], v)
    # O0 and O1 ARE the conditional means of Geo(1/2) split at theta = 2: (1/2 + 2/4) / (3/4) and 2 + 2
    pk = np.array([0.5 ** k for k in range(1, 60)])
    ks = np.arange(1, 60)
    assert abs((pk[:2] * ks[:2]).sum() / pk[:2].sum() - c["O0"]) < 1e-12
    assert abs((pk[2:] * ks[2:]).sum() / pk[2:].sum() - c["O1"]) < 1e-9
    # the queueing term takes over under load: lambda = 20 -> W_exact / M = 2.8 > 1/mu; rho >= 1 -> no bound
    assert abs(R.stochastic_constants(0.5, 3.0, 20.0, 100.0, 20.0)["opt_lower_bound"] - 2.8) < 1e-12
    assert R.stochastic_constants(0.5, 3.0, 20.0, 100.0, 20.0)["thm34_bound"] == float("inf")
    # rate_for_load inverts rho; the printed proxies of the App. H calibration (1/mu = theta = 293): 123, 586
    lam = R.rate_for_load(0.6, 1.0 / 293.0, 597.0, 300_000.0, 8192.0)
    assert abs(R.stochastic_constants(1.0 / 293.0, 597.0, lam, 300_000.0, 8192.0)["rho"] - 0.6) < 1e-12
    assert T.onebit_proxies(1.0 / 293.0, 293) == (123, 586)
    # eps decays as theta grows (the Remark)
    eps = [R.stochastic_constants(1.0 / 293.0, 597.0, lam, 300_000.0, 8192.0, theta=th)["eps"] for th in (64, 147, 293, 586, 1172)]
    assert all(a > b for a, b in zip(eps[1:], eps[2:])) and eps[-1] < 0.02 * eps[1]


def test_mean_request_latency_is_total_over_requests():
    off = torch.tensor([0, 3, 3, 10], dtype=torch.int64)
    tel = torch.tensor([30, 0, 140], dtype=torch.int64)
    assert R.mean_request_latency(tel, off) == 17.0
    assert R.mean_request_latency(tel, off, torch.tensor([0, 0, 19], dtype=torch.int32)) == 10.0
