"""Report layer: the paper's evaluation metrics computed from
the integer outputs of ``svf_simulate``: per-token latency = end-to-end latency / actual output
tokens (mean and 95th percentile) and token throughput = generated tokens / duration.  One model
step stands for one engine step, so latencies are in steps per token and throughput in tokens per
step.  Floating point and outside the parity contract: it post-processes bit-exact integers.

Works on torch tensors on any device; with an initialised process group the per-rank partial
results are combined over ranks (instances shard by rank, ``sharding.py``)."""
from __future__ import annotations

from typing import Dict

import torch

from . import sharding as S


def per_token_latency(arrival: torch.Tensor, output: torch.Tensor, finish: torch.Tensor) -> torch.Tensor:
    """(finish - arrival) / output per request, float64."""
    return (finish.to(torch.int64) - arrival.to(torch.int64)).to(torch.float64) / output.to(torch.float64)


def paper_metrics(arrival: torch.Tensor, output: torch.Tensor, finish: torch.Tensor,
                  offsets: torch.Tensor, status: torch.Tensor = None) -> Dict[str, float]:
    """Metrics over every request of every accepted instance of this rank's batch and, with a
    process group, of all ranks: mean / P95 per-token latency, token throughput averaged over
    instances (tokens of an instance / its duration from first arrival to last finish)."""
    I = offsets.numel() - 1
    sizes = (offsets[1:] - offsets[:-1]).to(torch.int64)
    ok_inst = torch.ones(I, dtype=torch.bool, device=offsets.device) if status is None else (status[:I] == 0)
    ok_inst &= sizes > 0
    inst_of = torch.repeat_interleave(torch.arange(I, device=offsets.device), sizes)
    ok_req = ok_inst[inst_of]
    ptl = per_token_latency(arrival, output, finish)[ok_req]
    # per-instance throughput: segment sums / (max finish - min arrival)
    tok = torch.zeros(I, dtype=torch.float64, device=offsets.device).index_add_(0, inst_of, output.to(torch.float64))
    last = torch.zeros(I, dtype=torch.int64, device=offsets.device).scatter_reduce_(
        0, inst_of, finish.to(torch.int64), reduce="amax", include_self=False)
    first = torch.zeros(I, dtype=torch.int64, device=offsets.device).scatter_reduce_(
        0, inst_of, arrival.to(torch.int64), reduce="amin", include_self=False)
    dur = (last - first).clamp(min=1).to(torch.float64)
    thr = (tok / dur)[ok_inst]
    # combine over ranks: gather the per-request values (P95 needs them all)
    ptl = S.gather_per_instance(ptl)
    thr = S.gather_per_instance(thr)
    if ptl.numel() == 0:
        return {"requests": 0, "mean_per_token_latency": 0.0, "p95_per_token_latency": 0.0, "token_throughput": 0.0}
    k = max(1, int(-(-95 * ptl.numel() // 100)))          # nearest rank ceil(0.95 n), as R13 does for p99
    p95 = torch.kthvalue(ptl, k).values
    return {"requests": int(ptl.numel()), "mean_per_token_latency": float(ptl.mean().item()),
            "p95_per_token_latency": float(p95.item()), "token_throughput": float(thr.mean().item())}


# ---------------------------------------------------------------------------------------------
# the stochastic regime (PAPER.md 3.4 and App. H): Poisson(lambda) arrivals,
# o ~ Geo(mu).  "E[TEL]" there is the expected end-to-end latency PER REQUEST (Lemma H.1 bounds it
# below by E[o] = 1/mu).  Real-valued and outside the parity contract, like everything in this file.
# ---------------------------------------------------------------------------------------------
def stochastic_constants(mu: float, mean_s: float, lam: float, M: float, p_max: float, theta: float = None) -> Dict[str, float]:
    """The constants of Thm 3.4 / Thm 3.5 / Lemma H.1 for one operating point.
      alpha   = p_max / M, p_max the largest peak s + o (the paper's s + o <= alpha M)
      E_vol   = E[s]/mu + 1/mu^2                                          (Eq. 101)
      rho     = lambda E[vol] / ((1 - alpha) M / 2)
      thm34   = 1 + 2 / ((1 - alpha)(1 - mu)(1 - rho))                    (Eq. 7)
      W_exact = lambda (1 - mu)/mu^2 (E[s] + 2/mu);  opt_lb = max{1/mu, W_exact / M}   (Eq. 89)
    and, given a 1-bit threshold theta:
      d       = theta q^theta / (1 - q^theta), q = 1 - mu;  O0 = 1/mu - d;  O1 = theta + 1/mu
      eps     = d^2 / 2;   thm35 = 1 + E_vol / (E_vol - eps) * 2 / ((1 - alpha)(1 - mu)(1 - rho))   (Eq. 8)
    Bounds are +inf when rho >= 1 (outside the theorems' range)."""
    alpha = p_max / M
    e_vol = mean_s / mu + 1.0 / (mu * mu)
    rho = lam * e_vol / ((1.0 - alpha) * M / 2.0)
    tail = 2.0 / ((1.0 - alpha) * (1.0 - mu) * (1.0 - rho)) if rho < 1.0 else float("inf")
    w_exact = lam * (1.0 - mu) / (mu * mu) * (mean_s + 2.0 / mu)
    out = {"alpha": alpha, "E_vol": e_vol, "rho": rho, "thm34_bound": 1.0 + tail, "W_exact": w_exact,
           "opt_lower_bound": max(1.0 / mu, w_exact / M)}
    if theta is not None:
        q_t = (1.0 - mu) ** theta
        d = theta * q_t / (1.0 - q_t)
        eps = 0.5 * d * d
        out.update({"theta": theta, "O0": 1.0 / mu - d, "O1": theta + 1.0 / mu, "eps": eps,
                    "thm35_bound": 1.0 + e_vol / (e_vol - eps) * tail})
    return out


def rate_for_load(rho: float, mu: float, mean_s: float, M: float, p_max: float) -> float:
    """The Poisson rate lambda that gives the conservative load rho (inverse of the definition above)."""
    alpha = p_max / M
    return rho * (1.0 - alpha) * M / 2.0 / (mean_s / mu + 1.0 / (mu * mu))


def mean_request_latency(total_latency: torch.Tensor, offsets: torch.Tensor, status: torch.Tensor = None) -> float:
    """The sample estimate of E[TEL] per request: sum of the accepted instances' total latencies over
    the number of their requests (all ranks, with a process group)."""
    I = offsets.numel() - 1
    sizes = (offsets[1:] - offsets[:-1]).to(torch.float64)
    ok = torch.ones(I, dtype=torch.bool, device=offsets.device) if status is None else (status[:I] == 0)
    num = (total_latency[:I].to(torch.float64) * ok).sum().reshape(1)
    den = (sizes * ok).sum().reshape(1)
    both = S.gather_per_instance(torch.cat([num, den]))
    num, den = float(both[0::2].sum().item()), float(both[1::2].sum().item())
    return num / den if den > 0 else 0.0
