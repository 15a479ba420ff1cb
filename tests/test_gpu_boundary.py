"""GPU-side checks of the boundary (include/svf.h conventions): workspace errors with real device
buffers, the width rule of the volume lower bound, corrupt offsets, empty 1-bit calls, concurrent
calls on several streams, and the report layer on CUDA tensors.  Run with ``-m gpu``."""
import numpy as np
import pytest

from paper_2606_22327_b200 import traces as T

pytestmark = pytest.mark.gpu

FIELDS = ("start", "finish", "total_latency", "p99_latency", "makespan", "peak_kv", "rounds",
          "decisions", "status")


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2606_22327_b200 import binding
    binding.lib()
    return binding


def test_short_and_unaligned_workspace_on_the_device(B):
    """SVF_EWORKSPACE (2) with real device buffers: one byte short, and an unaligned view of a buffer
    that would be large enough were it aligned; the full size (from an unaligned base too) is OK."""
    import ctypes as C
    import torch
    tr = T.config3(n_instances=40, n=300, lam=4.0, M=60_000)
    dt = B.DeviceTrace.from_host(tr)
    out = B.SimOut.alloc(dt)
    need = B.svf_simulate_workspace_bytes(dt)
    buf = torch.empty(need + 512, dtype=torch.uint8, device="cuda")
    ctr, res = dt.c_struct(), out.c_struct()
    L = B.lib()
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    call = lambda off, nbytes: L.svf_simulate(C.byref(ctr), 0, tr.M, C.byref(res), C.c_void_p(buf.data_ptr() + off), nbytes, st)
    assert call(0, need - 257) == B.EWORKSPACE
    assert call(1, 100) == B.EWORKSPACE                  # smaller than the alignment pad: must not wrap
    assert call(1, need - 256) == B.EWORKSPACE           # the pad eats into it
    assert call(1, need) == B.OK and call(0, need) == B.OK
    torch.cuda.synchronize()
    assert not out.status.cpu().numpy()[:40].any()
    w = torch.arange(1000, dtype=torch.int64, device="cuda").flip(0).contiguous()
    o = torch.empty_like(w)
    sneed = int(L.svf_sort_workspace_bytes(1000, 0, 64))
    assert L.svf_sort_words(1000, C.c_void_p(w.data_ptr()), C.c_void_p(o.data_ptr()), 0, 64, C.c_void_p(buf.data_ptr() + 8), 200, st) == B.EWORKSPACE
    assert L.svf_sort_words(1000, C.c_void_p(w.data_ptr()), C.c_void_p(o.data_ptr()), 0, 64, C.c_void_p(buf.data_ptr() + 8), sneed, st) == B.OK
    torch.cuda.synchronize()
    assert np.array_equal(o.cpu().numpy(), np.arange(1000))
    # svf_admit: the same through the ctypes prototype of the binding
    n_wait, n_run = 50, 5
    w = torch.ones(n_wait, dtype=torch.int32, device="cuda")
    r = torch.ones(n_run, dtype=torch.int32, device="cuda")
    n_adm = torch.zeros(1, dtype=torch.int64, device="cuda")
    aneed = B.svf_admit_workspace_bytes(n_wait, n_run)
    p = lambda t: C.c_void_p(t.data_ptr())
    adm = lambda off, nbytes: L.svf_admit(B.SVF, 1000, 0, n_wait, p(w), p(w), p(w), None, 1, 1, n_run, p(r), p(r), p(n_adm),
                                          None, None, None, C.c_void_p(buf.data_ptr() + off), nbytes, st)
    assert aneed + 512 <= buf.numel() + 512 and adm(0, aneed - 257) == B.EWORKSPACE and adm(3, 2) == B.EWORKSPACE
    if aneed <= buf.numel() - 8:
        assert adm(3, aneed) == B.OK
        torch.cuda.synchronize()
        assert int(n_adm.item()) == n_wait               # 50 requests of (s 1, o 1) fit beside five (kv 1, rem 1)


def test_onebit_calls_without_requests(B, oracle):
    """(1-bit, n = 0, bit = NULL) is a valid call on both sides (svf.h conventions)."""
    import torch
    e32 = torch.zeros(0, dtype=torch.int32, device="cuda")
    words, st = B.svf_keys(B.SVF_1BIT, e32, e32, e32, None, 2, 8)
    torch.cuda.synchronize()
    assert words.numel() == 0 and int(st.item()) == 0
    one = torch.ones(3, dtype=torch.int32, device="cuda")
    res = B.svf_admit(B.SVF_1BIT, 100, 0, e32, e32, e32, None, 2, 8, one, one)
    torch.cuda.synchronize()
    assert int(res.n_admitted.item()) == 0 and int(res.status.item()) == 0
    empty = T._one("empty", *(np.zeros(0, np.int32),) * 3, np.zeros(0, np.uint8), 100, 2, 8)
    dt = B.DeviceTrace.from_host(empty)
    dt.bit = None
    out = B.svf_simulate(dt, B.SVF_1BIT)
    torch.cuda.synchronize()
    assert int(out.status[0]) == 0 and int(out.total_latency[0]) == 0
    with pytest.raises(B.SvfError) as e:
        B.svf_keys(B.SVF_1BIT, one, one, one, None, 2, 8)                 # n > 0: bit is required
    assert e.value.code == B.EINVAL


def test_volume_lower_bound_width_rule(B, oracle):
    """A KNOWN DIVERGENCE, stated in include/svf.h and DESIGN.md R19: the library's presort orders 32-bit
    keys, so an instance that holds a volume >= 2^32 is refused with SVF_EOVERFLOW (never a silently
    mis-sorted bound), while Eq. 5 sets no such width and the oracle returns the exact value.  s = o =
    60,000 (5.4e9) beside s = 30,000, o = 60,000 (3.6e9); the other instances of the call agree exactly."""
    import torch
    parts = [T._one("mixed", np.zeros(2, np.int32), np.array([60_000, 30_000]), np.array([60_000, 60_000]), np.zeros(2, np.uint8), 10 ** 9, 1, 1),
             T._one("below", np.zeros(2, np.int32), np.array([30_000, 30_000]), np.array([60_000, 60_000]), np.zeros(2, np.uint8), 10 ** 9, 1, 1),
             T.random_small(5, 40, 60, 50, 10 ** 6)]
    tr = T.concat(parts, "lb-wide", 10 ** 9, 1, 1)
    lb, st = B.svf_volume_lower_bound(B.DeviceTrace.from_host(tr))
    torch.cuda.synchronize()
    lb, st = lb.cpu().numpy(), st.cpu().numpy()
    rlb, rst = oracle.volume_lower_bound(tr)
    assert rst.tolist() == [0, 0, 0] and int(rlb[0]) == 12_600_090_000 and int(rlb[1]) == 3 * 3_600_030_000
    assert st.tolist() == [B.EOVERFLOW, 0, 0] and int(lb[0]) == 0                  # the library's limit
    assert np.array_equal(lb[1:], rlb[1:])                                         # everything it accepts is exact


def test_corrupt_offsets_are_reported_not_simulated(B):
    """Offsets that are not non-decreasing can make two 'valid' instances overlap: the whole call
    reports SVF_EINVAL per instance and returns (no hang, no write outside the buffers)."""
    import torch
    tr = T.config3(n_instances=6, n=50, lam=4.0, M=60_000)
    good = B.svf_simulate(B.DeviceTrace.from_host(tr), 0)
    torch.cuda.synchronize()
    assert not good.status.cpu().numpy()[:6].any()
    for bad_off in ([0, 100, 50, 150, 200, 250, 300],       # instance 1 runs backwards, 2 overlaps 0
                    [0, 50, 100, 150, 200, 250, 299],       # does not end at N
                    [5, 50, 100, 150, 200, 250, 300]):      # does not start at 0
        dt = B.DeviceTrace.from_host(tr)
        dt.offsets = torch.tensor(bad_off, dtype=torch.int64, device="cuda")
        dt.max_instance = 100
        for pols in ([0], [3, 1]):
            outs = B.svf_simulate_policies(dt, pols)
            torch.cuda.synchronize()
            for out in outs:
                assert (out.status.cpu().numpy()[:6] == B.EINVAL).all()
                assert not out.total_latency.cpu().numpy()[:6].any()
        lb, st = B.svf_volume_lower_bound(dt)
        torch.cuda.synchronize()
        assert (st.cpu().numpy() == B.EINVAL).all() and not lb.cpu().numpy().any()


def test_concurrent_calls_on_several_streams(B, oracle):
    """The compute calls keep no state between calls: eight svf_simulate_policies calls in flight at
    once on eight streams (the end-to-end leg of bench.py), each with its own workspace, give the
    results of the same calls made one after the other."""
    import torch
    batch = T.config3(n_instances=256, n=400, lam=4.0, M=120_000)
    chunks = [batch.subset(range(32 * c, 32 * c + 32)) for c in range(8)]
    streams = [torch.cuda.Stream() for _ in chunks]
    dts = [B.DeviceTrace.from_host(c) for c in chunks]
    wss = [torch.empty(B.svf_simulate_policies_workspace_bytes(d, 4), dtype=torch.uint8, device="cuda") for d in dts]
    torch.cuda.synchronize()
    for rep in range(3):
        outs = []
        for d, w, s in zip(dts, wss, streams):
            with torch.cuda.stream(s):
                outs.append(B.svf_simulate_policies(d, [0, 1, 2, 3], ws=w, stream=s))
        torch.cuda.synchronize()
        for c, (chunk, o4) in enumerate(zip(chunks, outs)):
            for pol, out in enumerate(o4):
                ref = oracle.simulate(chunk, pol, n_threads=8)
                for k in FIELDS:
                    g = getattr(out, k).cpu().numpy()
                    r = getattr(ref, k)
                    assert np.array_equal(g[: len(r)], r), (rep, c, pol, k)


def test_report_layer_on_cuda_tensors(B, oracle):
    """NEXT-4: paper_metrics on the CUDA tensors bench.py hands it == the same function on
    CPU copies == plain numpy on the oracle's schedule."""
    import torch
    from paper_2606_22327_b200 import report as R
    tr = T.config3(n_instances=64, n=300, lam=4.0, M=60_000)
    tr.output[tr.offsets[5] + 3] = 0                         # one rejected instance: left out of the metrics
    dt = B.DeviceTrace.from_host(tr)
    out = B.svf_simulate(dt, 0)
    torch.cuda.synchronize()
    got = R.paper_metrics(dt.arrival, dt.output, out.finish[: tr.n_requests], dt.offsets, out.status)
    cpu = R.paper_metrics(dt.arrival.cpu(), dt.output.cpu(), out.finish[: tr.n_requests].cpu(), dt.offsets.cpu(), out.status.cpu())
    ref = oracle.simulate(tr, 0)
    ptl, thr = [], []
    for j in range(tr.n_instances):
        lo, hi = int(tr.offsets[j]), int(tr.offsets[j + 1])
        if ref.status[j] != 0:
            continue
        ptl.extend(((ref.finish[lo:hi].astype(np.int64) - tr.arrival[lo:hi]) / tr.output[lo:hi].astype(np.float64)).tolist())
        thr.append(tr.output[lo:hi].sum() / max(1, int(ref.finish[lo:hi].max()) - int(tr.arrival[lo:hi].min())))
    ptl = np.sort(np.array(ptl))
    want = {"requests": len(ptl), "mean_per_token_latency": float(ptl.mean()),
            "p95_per_token_latency": float(ptl[-(-95 * len(ptl) // 100) - 1]), "token_throughput": float(np.mean(thr))}
    assert got["requests"] == cpu["requests"] == want["requests"] == 63 * 300
    for k in ("mean_per_token_latency", "p95_per_token_latency", "token_throughput"):
        assert abs(got[k] - want[k]) <= 1e-12 * max(1.0, abs(want[k])), k
        assert abs(cpu[k] - want[k]) <= 1e-12 * max(1.0, abs(want[k])), k


def test_stochastic_regime_report(B, oracle):
    """NEXT-3: on the App. H reference workload the GPU's estimate of E[TEL] per request, over Lemma
    H.1's lower bound on OPT (Eq. 89), sits below the bounds of Thm 3.4 (SVF) and Thm 3.5 (1-bit SVF) and
    not below 1 by more than sampling noise; the estimate itself equals the oracle's (integers in, one
    division)."""
    import torch
    from paper_2606_22327_b200 import report as R
    mu, M, p_max = 1.0 / 293.0, 300_000, 8192
    for rho, theta in ((0.6, 293), (0.9, 147)):
        probe = T.stochastic(n_instances=48, n=800, lam=1.0, M=M)
        mean_s = float(probe.prompt.mean())
        lam = R.rate_for_load(rho, mu, mean_s, M, p_max)
        tr = T.stochastic(n_instances=48, n=800, lam=lam, M=M, theta=theta)
        c = R.stochastic_constants(mu, mean_s, lam, M, p_max, theta=theta)
        assert abs(c["rho"] - rho) < 1e-9 and (tr.O0, tr.O1) == T.onebit_proxies(mu, theta)
        dt = B.DeviceTrace.from_host(tr)
        outs = B.svf_simulate_policies(dt, [B.SVF, B.SVF_1BIT], want=("total_latency", "status"))
        torch.cuda.synchronize()
        for pol, out, bound in ((B.SVF, outs[0], c["thm34_bound"]), (B.SVF_1BIT, outs[1], c["thm35_bound"])):
            est = R.mean_request_latency(out.total_latency, dt.offsets, out.status)
            ref = oracle.simulate(tr, pol, n_threads=8)
            assert est == float(ref.total_latency.sum()) / tr.n_requests
            ratio = est / c["opt_lower_bound"]
            assert 0.9 < ratio <= bound, (rho, theta, pol, ratio, bound)
