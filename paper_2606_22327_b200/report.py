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
