"""svf_admit_static: the admission decision for callers that are not allowed to allocate.

A scheduler embedded in a serving engine takes this decision every engine step, but the engine has
usually given all spare HBM to its KV-cache pool at start-up: a cudaMalloc from the step loop may
fail, and it would stall the decode stream even when it succeeds.  ``svf_admit_static`` therefore
keeps its scratch in a fixed 3 MiB array inside the library (limit: 65,536 waiting and 8,192 running
requests) and takes only inputs and outputs from the caller.

What is checked here, through the C ABI on the GPU: the answer is the same, bit for bit (the
tolerance of every admission test in this suite), as ``svf_admit`` with a caller-supplied workspace
-- on calls made back to back, so that each later call finds the array full of the previous call's
leftovers; the size limit is refused up front; and a repeated call leaves the amount of free device
memory untouched.

The file is named to be collected last: it must pass both on its own in a fresh process and after
every other GPU test has run (including those that switch the profiling aid on and off).
"""
import numpy as np
import pytest

from paper_2606_22327_b200 import traces as T

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2606_22327_b200 import binding
    binding.lib()
    binding.set_profiling(0)        # the entry point refuses to run under the timing aid (it creates events)
    return binding


def _state_on_device(seed, n_wait, n_run, M):
    import torch
    st = T.admit_state(seed, n_wait, n_run, M)
    return [torch.from_numpy(np.ascontiguousarray(x)).cuda() for x in st]


def _blank_out(B, n_wait, want_sorted=True):
    import torch
    return B.AdmitOut(torch.full((1,), -7, dtype=torch.int64, device="cuda"),
                      torch.full((max(n_wait, 1),), -1, dtype=torch.int32, device="cuda"),
                      torch.zeros(max(n_wait, 1), dtype=torch.int64, device="cuda") if want_sorted else None,
                      torch.full((1,), -7, dtype=torch.int32, device="cuda"))


def _same_as_existing_path(B, policy, M, st, O0=179, O1=887):
    """One decision through both entry points; every output compared exactly.  Returns k."""
    import torch
    w_s, w_o, w_a, w_bit, r_kv, r_rem = st
    n_wait = int(w_s.numel())
    ref = B.svf_admit(policy, M, 5, w_s, w_o, w_a, w_bit, O0, O1, r_kv, r_rem)      # caller-supplied workspace
    torch.cuda.synchronize()
    out = B.svf_admit_static(policy, M, 5, w_s, w_o, w_a, w_bit, O0, O1, r_kv, r_rem, _blank_out(B, n_wait))
    torch.cuda.synchronize()
    assert int(out.status.item()) == int(ref.status.item())
    k = int(ref.n_admitted.item())
    assert int(out.n_admitted.item()) == k
    assert torch.equal(out.admitted_idx[:k], ref.admitted_idx[:k])
    if int(ref.status.item()) == 0:
        assert torch.equal(out.sorted_words[:n_wait], ref.sorted_words[:n_wait])
    return k


def test_static_scratch_gives_the_same_decisions_call_after_call(B):
    import torch
    # (n_wait, n_run, M, policy): deep queues first -- these are the ones that use the scratch (keys,
    # onesweep sort, bisection, serial hand-over) -- each with another shape and policy, so that the
    # array is dirty in a different way every time; then a queue small enough for the one-launch form
    calls = [(40_000, 1_000, 4_000_000, 0),
             (65_536, 8_192, 30_000_000, 1),        # the stated maximum; n_run > 4096 sorts the running set too
             (20_000, 100, 10_000_000, 0),          # window exhausted, handed over to the serial kernels
             (9_000, 700, 1_500_000, 2),
             (30_000, 4_096, 8_000_000, 3),
             (3_000, 500, 1_000_000, 0)]
    ks = []
    for i, (n_wait, n_run, M, policy) in enumerate(calls):
        ks.append(_same_as_existing_path(B, policy, M, _state_on_device(300 + i, n_wait, n_run, M)))
    assert min(ks) >= 0 and max(ks) > 0
    # the first call again, after all that: same decision as at the start
    n_wait, n_run, M, policy = calls[0]
    assert _same_as_existing_path(B, policy, M, _state_on_device(300, n_wait, n_run, M)) == ks[0]
    # a data error travels through status_out exactly as with svf_admit
    st = _state_on_device(7, 12_000, 50, 1_000_000)
    st[1][77] = 0                                                                    # o < 1
    assert _same_as_existing_path(B, 0, 1_000_000, st) == 0
    torch.cuda.synchronize()


def test_sizes_beyond_the_array_are_refused_and_nothing_is_written(B):
    import torch
    for n_wait, n_run in ((65_537, 0), (10, 8_193)):
        st = _state_on_device(1, n_wait, n_run, 10 ** 9)
        out = _blank_out(B, n_wait, want_sorted=False)
        with pytest.raises(B.SvfError) as e:
            B.svf_admit_static(0, 10 ** 9, 0, *st[:4], 1, 1, *st[4:], out)
        assert e.value.code == B.EWORKSPACE
        torch.cuda.synchronize()
        assert int(out.n_admitted.item()) == -7 and int(out.status.item()) == -7


def test_a_repeated_call_takes_no_device_memory(B):
    """Not a proof, but what a caller would see: once the kernels of a given shape have been loaded by a
    first call, further calls leave cudaMemGetInfo's free figure where it was."""
    import torch
    n_wait, n_run, M = 50_000, 2_000, 6_000_000
    st = _state_on_device(9, n_wait, n_run, M)
    out = _blank_out(B, n_wait)
    B.svf_admit_static(0, M, 1, *st[:4], 179, 887, *st[4:], out)
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        B.svf_admit_static(0, M, 1, *st[:4], 179, 887, *st[4:], out)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before
    assert int(out.status.item()) == 0 and int(out.n_admitted.item()) > 0
