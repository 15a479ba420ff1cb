"""GPU parity (bit-exact) at the sizes BASELINE.json states for every config the north star lists,
every field, against the CPU oracle, through the C ABI.  Run on the B200 box with ``-m gpu``.
(configs[0], configs[1] and configs[2] at rate 4 are in test_gpu_admit_simulate.py.)"""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from paper_2606_22327_b200 import traces as T

pytestmark = pytest.mark.gpu

FIELDS = ("start", "finish", "total_latency", "p99_latency", "makespan", "peak_kv", "rounds",
          "decisions", "status")
THREADS = max(1, min(16, os.cpu_count() or 1))


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2606_22327_b200 import binding
    binding.lib()
    return binding


def _same(out, ref, tr, ctx):
    I, N = tr.n_instances, tr.n_requests
    for k in FIELDS:
        g = getattr(out, k).cpu().numpy()
        g = g[:N] if k in ("start", "finish") else g[:I]
        r = getattr(ref, k)
        if not np.array_equal(g, r):
            bad = np.nonzero(g != r)[0]
            raise AssertionError(f"{ctx}: field {k} differs at {bad[:8]} (gpu {g[bad[:8]]}, oracle {r[bad[:8]]}); "
                                 f"{len(bad)} of {len(r)}")


def _properties(out, tr):
    """What holds at any size (Eq. 3c, Lemma G.1), on every instance."""
    start, finish = out.start.cpu().numpy()[: tr.n_requests], out.finish.cpu().numpy()[: tr.n_requests]
    assert not out.status.cpu().numpy()[: tr.n_instances].any()
    assert np.array_equal(finish - start, tr.output) and (start >= tr.arrival).all()
    tel = out.total_latency.cpu().numpy()[: tr.n_instances]
    assert np.array_equal(tel, np.add.reduceat((finish - tr.arrival).astype(np.int64), tr.offsets[:-1]))
    assert (tel >= np.add.reduceat(tr.output.astype(np.int64), tr.offsets[:-1])).all()
    assert (out.peak_kv.cpu().numpy()[: tr.n_instances] <= tr.M).all()


@pytest.mark.parametrize("lam", [2.0, 4.0, 8.0])
def test_config3_full_size_other_rates(B, oracle, lam):
    """configs[2]: 4,096 instances x 1,000 requests at Poisson rates 2, 4 (the launch bench.py times)
    and 8, all four policies in the one-launch call, EVERY instance and field."""
    import torch
    tr = T.config3(n_instances=4096, lam=lam)
    outs = B.svf_simulate_policies(B.DeviceTrace.from_host(tr), [0, 1, 2, 3])
    torch.cuda.synchronize()
    for pol, out in enumerate(outs):
        _same(out, oracle.simulate(tr, pol, n_threads=THREADS), tr, f"cfg3 lam={lam} policy {pol}")
        _properties(out, tr)


def test_config4_full_size_all_policies(B, oracle):
    """configs[3]: ONE instance of n = 200,000 at rate 64, M = 1e6 under all four policies (SVF and
    FCFS are also in test_gpu_admit_simulate.py): every start / finish and every scalar."""
    import torch
    tr = T.config4()
    with ThreadPoolExecutor(4) as ex:                       # the oracle is one serial chain per policy
        refs = list(ex.map(lambda p: oracle.simulate(tr, p), range(4)))
    dt = B.DeviceTrace.from_host(tr)
    for pol in range(4):
        out = B.svf_simulate(dt, pol)
        torch.cuda.synchronize()
        _same(out, refs[pol], tr, f"cfg4 policy {pol}")
        _properties(out, tr)
        assert int(refs[pol].total_latency[0]) > 2 ** 31


@pytest.mark.parametrize("M", [50_000, 200_000, 800_000])
def test_config5_full_grid(B, oracle, M):
    """configs[4]: 256 instances x 5,000 requests, bimodal outputs, for every budget M and every flip
    probability p in {0, 0.05, 0.2} under SVF, 1-bit SVF and SJF: EVERY instance and field of all 27
    cells against the oracle."""
    import torch
    base_tel = {}
    for p in (0.0, 0.05, 0.2):
        tr = T.config5(n_instances=256, M=M, p_flip=p)
        assert tr.n_instances == 256 and tr.n_requests == 256 * 5000
        dt = B.DeviceTrace.from_host(tr)
        outs = B.svf_simulate_policies(dt, [0, 1, 2])
        torch.cuda.synchronize()
        for pol, out in zip((0, 1, 2), outs):
            ref = oracle.simulate(tr, pol, n_threads=THREADS)
            _same(out, ref, tr, f"cfg5 M={M} p={p} policy {pol}")
            _properties(out, tr)
            if pol != 1:                                     # only the 1-bit order looks at the bits
                assert np.array_equal(ref.total_latency, base_tel.setdefault(pol, ref.total_latency))
        # the single-policy entry point picks its kernel family from I alone (not I x P)
        one = B.svf_simulate(dt, 1)
        torch.cuda.synchronize()
        for k in FIELDS:
            assert np.array_equal(getattr(one, k).cpu().numpy(), getattr(outs[1], k).cpu().numpy()), (k, p)
