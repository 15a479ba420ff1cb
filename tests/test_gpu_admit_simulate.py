"""GPU parity (bit-exact): svf_admit and svf_simulate against the CPU oracle, through the C ABI.
Run on the B200 box with ``-m gpu``."""
import os

import numpy as np
import pytest

from paper_2606_22327_b200 import traces as T

pytestmark = pytest.mark.gpu

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
POL = {"svf": 0, "svf_1bit": 1, "sjf": 2, "fcfs": 3}
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


def _dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def run_gpu(B, trace, policy, M=None, want=FIELDS):
    import torch
    dt = B.DeviceTrace.from_host(trace)
    out = B.svf_simulate(dt, policy, M, want=want)
    torch.cuda.synchronize()
    return {k: getattr(out, k).cpu().numpy() for k in want}


def assert_same(got, ref, trace, ctx=""):
    I, N = trace.n_instances, trace.n_requests
    for k in got:
        g = got[k][:N] if k in ("start", "finish") else got[k][:I]
        r = getattr(ref, k)
        if not np.array_equal(g, r):
            bad = np.nonzero(g != r)[0]
            raise AssertionError(f"{ctx}: field {k} differs at {bad[:8]} (gpu {g[bad[:8]]}, oracle {r[bad[:8]]}); "
                                 f"{len(bad)} of {len(r)}")


def check(B, oracle, trace, policy, M=None, ctx="", threads=8):
    ref = oracle.simulate(trace, policy, M=M, n_threads=threads)
    got = run_gpu(B, trace, policy, M)
    assert_same(got, ref, trace, ctx or f"{trace.name} policy {policy}")
    return ref, got


# ---------------------------------------------------------------------------------------------
# svf_simulate
# ---------------------------------------------------------------------------------------------
def _golden_examples():
    ex, cur = [], None
    for line in open(os.path.join(GOLDEN, "hand_examples.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        tok = line.split()
        if tok[0] == "example":
            cur = {"name": tok[1], "M": int(tok[2].split("=")[1]), "policy": tok[3].split("=")[1], "req": []}
            ex.append(cur)
        elif tok[0] == "req":
            cur["req"].append(tuple(int(x) for x in tok[1:4]))
        elif tok[0] == "start":
            cur["start"] = [int(x) for x in tok[1:]]
        elif tok[0] == "tel":
            cur["tel"] = int(tok[1])
    return ex


def test_hand_examples_from_the_paper_model(B):
    """Values derived by hand from Eq. 3c (tests/golden/hand_examples.txt), not from any code."""
    for ex in _golden_examples():
        a, s, o = (np.array(x, np.int32) for x in zip(*ex["req"]))
        tr = T._one(ex["name"], a, s, o, np.zeros(len(a), np.uint8), ex["M"], 1, 1)
        got = run_gpu(B, tr, POL[ex["policy"]])
        assert list(got["start"][: len(a)]) == ex["start"], ex["name"]
        assert int(got["total_latency"][0]) == ex["tel"], ex["name"]
        assert int(got["status"][0]) == 0


def test_config1_tiny_offline_batch(B, oracle):
    """configs[0]: n=8 at t=0, M=32, all four policies, 512 seeds batched as instances."""
    parts = [T.config1(i) for i in range(512)]
    tr = T.concat(parts, "cfg1x512", 32, 2, 8)
    for policy in range(4):
        check(B, oracle, tr, policy)


def test_config2_single_online_trace(B, oracle):
    """configs[1]: n=2000, lambda=4, M=300k: one instance, one CTA."""
    for inst in range(2):
        tr = T.config2(inst)
        for policy in range(4):
            ref, _ = check(B, oracle, tr, policy)
            assert ref.status[0] == 0 and ref.peak_kv[0] <= tr.M


@pytest.mark.parametrize("lam", [2.0, 4.0, 8.0])
def test_config3_batched_subset(B, oracle, lam):
    """configs[2] shape, 96 instances x 1000 requests (several waves of the warp-per-instance
    kernel would need 4096; the full size is covered by test_config3_full_size_sampled)."""
    tr = T.config3(n_instances=96, lam=lam)
    for policy in range(4):
        check(B, oracle, tr, policy)


def test_config3_full_size_sampled(B, oracle):
    """configs[2] at full size (4096 x 1000, the launch bench.py times): every instance's scalar
    outputs against the oracle for SVF; start/finish on all requests."""
    tr = T.config3(n_instances=4096, lam=4.0)
    check(B, oracle, tr, 0)
    got = run_gpu(B, tr, 3, want=("total_latency", "status", "peak_kv"))
    sub = np.arange(0, 4096, 64)
    ref = oracle.simulate(tr.subset(sub), 3, n_threads=8)
    assert np.array_equal(got["total_latency"][sub], ref.total_latency)
    assert np.array_equal(got["peak_kv"][sub], ref.peak_kv)
    assert not got["status"][:4096].any()


def test_bench_launch_configuration_sampled(B, oracle):
    """The exact call bench.py times: configs[2] at full size, all four policies in ONE
    svf_simulate_policies launch, every output; 96 sampled instances per policy against the
    oracle, every field, plus properties that hold at any size for all instances."""
    import torch
    tr = T.config3(n_instances=4096, lam=4.0)
    dt = B.DeviceTrace.from_host(tr)
    outs = B.svf_simulate_policies(dt, [0, 1, 2, 3])
    torch.cuda.synchronize()
    sub = np.arange(5, 4096, 43)
    subtr = tr.subset(sub)
    rows = np.concatenate([np.arange(tr.offsets[j], tr.offsets[j + 1]) for j in sub])
    sum_o = np.add.reduceat(tr.output.astype(np.int64), tr.offsets[:-1])
    for pol, out in zip(range(4), outs):
        ref = oracle.simulate(subtr, pol, n_threads=8)
        for k in FIELDS:
            g = getattr(out, k).cpu().numpy()
            g = g[rows] if k in ("start", "finish") else g[sub]
            assert np.array_equal(g, getattr(ref, k)), f"policy {pol} field {k}"
        start, finish = out.start.cpu().numpy(), out.finish.cpu().numpy()
        assert not out.status.cpu().numpy().any()
        assert np.array_equal(finish - start, tr.output)                     # non-preemptive, o steps each
        assert (start >= tr.arrival).all()
        tel = out.total_latency.cpu().numpy()
        assert np.array_equal(tel, np.add.reduceat((finish - tr.arrival).astype(np.int64), tr.offsets[:-1]))
        assert (tel >= sum_o).all()                                          # Lemma G.1
        assert (out.peak_kv.cpu().numpy() <= tr.M).all()                     # Eq. 3c
        assert np.array_equal(out.makespan.cpu().numpy(), np.maximum.reduceat(finish, tr.offsets[:-1]))


def test_config4_high_concurrency_reduced(B, oracle):
    """configs[3] laws at n=20,000 (state in the global-memory slot: > 16k entries)."""
    tr = T.config4(n=20_000, M=1_000_000)
    for policy in range(4):
        check(B, oracle, tr, policy)


def test_config4_full_size(B, oracle):
    """configs[3]: n=200,000, lambda=64, M=1e6; total latency exceeds 2^32 (int64 path)."""
    tr = T.config4()
    for policy in (0, 3):
        ref, _ = check(B, oracle, tr, policy)
        assert ref.total_latency[0] > (2 ** 31 if policy == 0 else 2 ** 32)


@pytest.mark.parametrize("M", [50_000, 200_000, 800_000])
def test_config5_onebit_sweep_subset(B, oracle, M):
    """configs[4] shape: 24 instances x 5000, bimodal outputs, flipped bits."""
    for p in (0.0, 0.2):
        tr = T.config5(n_instances=24, M=M, p_flip=p)
        for policy in (0, 1, 2):
            check(B, oracle, tr, policy)


def test_ragged_batch_with_empty_and_rejected_instances(B, oracle):
    """Instances of different sizes, empty ones, and every data error; a bad instance must not
    disturb its neighbours."""
    M = 40
    parts = []
    parts.append(T.random_small(1, 17, 10, 12, M, a_hi=30))
    parts.append(T._one("empty", *(np.zeros(0, np.int32),) * 3, np.zeros(0, np.uint8), M, 2, 8))
    bad_range = T.random_small(2, 9, 10, 12, M, a_hi=5); bad_range.output[3] = 0
    parts.append(bad_range)
    unsorted = T.random_small(3, 9, 10, 12, M, a_hi=50); unsorted.arrival[5] = 0; unsorted.arrival[4] = 7
    parts.append(unsorted)
    infeasible = T.random_small(4, 9, 10, 12, M, a_hi=5); infeasible.prompt[0] = 35; infeasible.output[0] = 6
    parts.append(infeasible)
    overflow = T.random_small(5, 5, 10, 12, M, a_hi=5); overflow.arrival[-1] = 2 ** 31 - 5
    parts.append(overflow)
    parts.append(T.random_small(6, 33, 10, 12, M, a_hi=3))
    parts.append(T.random_small(7, 1, 10, 12, M))
    neg = T.random_small(8, 6, 10, 12, M, a_hi=5); neg.prompt[2] = -1
    parts.append(neg)
    parts.append(T.random_small(9, 64, 10, 12, M, a_hi=100))
    tr = T.concat(parts, "ragged", M, 2, 8)
    for policy in range(4):
        ref, got = check(B, oracle, tr, policy)
        assert set(ref.status.tolist()) >= {0, 16, 17, 18, 19}


def test_random_small_instances_all_policies(B, oracle):
    """Many tiny random online instances (tight budgets: M hit exactly, blocked heads, event-free
    admissions) in one batch."""
    parts = [T.random_small(100 + i, 3 + i % 40, 9, 11, 24, a_hi=(i % 7) * 5) for i in range(600)]
    tr = T.concat(parts, "small600", 24, 3, 9)
    for policy in range(4):
        check(B, oracle, tr, policy)
    # the same batch under a loose budget: everything starts on arrival, TEL = sum o (Lemma G.1)
    ref, got = check(B, oracle, tr, 0, M=10 ** 9)
    assert int(got["total_latency"][: tr.n_instances].sum()) == tr.request_steps


def test_group_widths_and_state_placement(B, oracle):
    """Shapes that select each form of the one-warp kernel (M = 60,000: few requests run at once); the
    CTA-wide kernels and the 32-slot warp kernel are in the crowd test, configs[3] and configs[4]."""
    shapes = [(200, 1300, 4.0),        # one warp each, two bitmap words per lane (more than 1024 requests)
              (100, 2500, 8.0),        # one warp each, register queue of eight words per lane, packed records (2,049 .. 8,192 requests)
              (4096 // 8, 40, 2.0),     # many small instances -> one warp each
              (100, 600, 4.0),         # register queue, one bitmap word per lane
              (1, 2000, 4.0),          # a single instance: register queue, two words per lane
              (2, 9000, 8.0)]          # shared-memory bitmap, ext slots in the global slot
    for I, n, lam in shapes:
        tr = T.config3(n_instances=I, n=n, lam=lam, M=60_000)
        for policy in (0, 3):
            check(B, oracle, tr, policy, ctx=f"I={I} n={n}")


def test_policies_in_one_call(B, oracle):
    """svf_simulate_policies: one launch over n_policies x I work items == separate calls == oracle,
    for each kernel family (warp + register bitmap, CTA + shared bitmap, wide kernel for M >= 2^30)."""
    import torch
    cases = [(T.config3(n_instances=300, n=200, lam=4.0, M=60_000), None, [0, 1, 2, 3]),
             (T.config3(n_instances=6, n=1500, lam=8.0, M=60_000), None, [3, 0, 2]),
             (T.config5(n_instances=3, n=5000, M=200_000, p_flip=0.2), None, [1, 0]),
             (T.config3(n_instances=20, n=100, lam=4.0), 1 << 30, [0, 3]),
             (T.config3(n_instances=70, n=150, lam=8.0, M=40_000), None, [0, 1, 2, 3, 3, 2, 1, 0])]   # the maximum of 8
    for tr, M, pols in cases:
        dt = B.DeviceTrace.from_host(tr)
        outs = B.svf_simulate_policies(dt, pols, M)
        torch.cuda.synchronize()
        for pol, out in zip(pols, outs):
            ref = oracle.simulate(tr, pol, M=M, n_threads=8)
            got = {k: getattr(out, k).cpu().numpy() for k in FIELDS}
            assert_same(got, ref, tr, f"{tr.name} policies={pols} policy {pol}")


def test_policies_call_with_rejected_and_empty_instances(B, oracle):
    import torch
    parts = [T.random_small(7, 12, 9, 11, 24, a_hi=10), T.random_small(8, 0, 9, 11, 24),
             T.random_small(9, 30, 9, 11, 24, a_hi=3)]
    parts[2].output[4] = 0                              # ERANGE in instance 2
    tr = T.concat(parts, "mixed", 24, 3, 9)
    dt = B.DeviceTrace.from_host(tr)
    outs = B.svf_simulate_policies(dt, [2, 1])
    torch.cuda.synchronize()
    for pol, out in zip([2, 1], outs):
        ref = oracle.simulate(tr, pol)
        assert_same({k: getattr(out, k).cpu().numpy() for k in FIELDS}, ref, tr, f"mixed policy {pol}")
    assert int(outs[0].status[2]) != 0


@pytest.mark.parametrize("sigma", [0.3, 1.0])
def test_predicted_length_keys(B, oracle, sigma):
    """NEXT-1: `output_key` (predicted lengths) orders SVF / SJF, the true lengths drive the model
    (R7).  Every presort path: shared-memory segment sort (warp kernel and CTA
    kernel), device-wide onesweep (instances > 4096), wide kernel (M >= 2^30)."""
    cases = [(T.config3(n_instances=64, n=300, lam=4.0, M=60_000), None),
             (T.config3(n_instances=5, n=1500, lam=8.0, M=60_000), None),
             (T.config3(n_instances=2, n=6000, lam=8.0, M=60_000), None),
             (T.config3(n_instances=12, n=100, lam=4.0), 1 << 30)]
    for base_tr, M in cases:
        tr = T.with_predicted_lengths(base_tr, sigma=sigma, seed=3, hi=4096)
        assert not np.array_equal(tr.output_key, tr.output)
        for policy in range(4):
            check(B, oracle, tr, policy, M=M, ctx=f"{tr.name} policy {policy}")
    # predictions change the SVF schedule, but not FCFS
    tr = T.with_predicted_lengths(cases[0][0], sigma=1.0, seed=3, hi=4096)
    assert not np.array_equal(run_gpu(B, tr, 0)["start"], run_gpu(B, cases[0][0], 0)["start"])
    assert np.array_equal(run_gpu(B, tr, 3)["start"], run_gpu(B, cases[0][0], 3)["start"])
    # a prediction < 1 is a range error of that instance only
    tr.output_key[tr.offsets[2] + 5] = 0
    ref, got = check(B, oracle, tr, 0)
    assert got["status"][2] == oracle.ERANGE and not got["status"][:2].any()


def test_outputs_are_optional(B, oracle):
    tr = T.config3(n_instances=8, lam=4.0)
    ref = oracle.simulate(tr, 0)
    got = run_gpu(B, tr, 0, want=("total_latency",))
    assert np.array_equal(got["total_latency"][:8], ref.total_latency)
    got = run_gpu(B, tr, 0, want=("p99_latency", "finish"))
    assert np.array_equal(got["p99_latency"][:8], ref.p99_latency)
    assert np.array_equal(got["finish"][: tr.n_requests], ref.finish)


def test_schedule_passes_the_independent_validator(B):
    """The GPU schedule itself (not via the oracle simulator) against the paper's definitions:
    capacity, area conservation, no bypass, blocked heads really blocked (oracle/validator.py)."""
    from oracle import validator
    tr = T.config2(3, n=600, M=120_000)
    for policy in range(4):
        got = run_gpu(B, tr, policy)
        facts = validator.validate(tr, policy, got["start"][: tr.n_requests], finish=got["finish"][: tr.n_requests],
                                   check_blocked=200)
        assert facts["total_latency"] == int(got["total_latency"][0])
        assert facts["rounds"] == int(got["rounds"][0]) and facts["decisions"] == int(got["decisions"][0])
        assert facts["peak_kv"] == int(got["peak_kv"][0]) and facts["p99_latency"] == int(got["p99_latency"][0])


# ---------------------------------------------------------------------------------------------
# svf_admit
# ---------------------------------------------------------------------------------------------
def _admit_state(seed, n_wait, n_run, M):
    sd = T.instance_seed(88, seed)
    w_s = T.lognormal_int(sd, 2, 3, n_wait, 1000.0, 0.8, 16, 8192)
    w_o = T.lognormal_int(sd, 4, 5, n_wait, 400.0, 1.0, 1, 4096)
    w_a = np.sort(T.uniform_int(sd, 1, n_wait, 0, 5000))
    w_bit = (w_o > 400).astype(np.uint8)
    r_rem = T.uniform_int(sd, 6, n_run, 1, 3000)
    # running set scaled to sit just under the budget at its worst completion time
    r_kv = T.lognormal_int(sd, 7, 8, n_run, 1200.0, 0.8, 16, 12000)
    if n_run:
        order = np.argsort(-r_rem, kind="stable")
        cum = np.cumsum(r_kv[order].astype(np.int64)).astype(np.float64)
        remterm = (r_rem[order].astype(np.int64) * np.arange(1, n_run + 1)).astype(np.float64)
        target = (0.97 if seed % 2 else 0.8) * M
        scale = float(np.clip(((target - remterm) / cum).min(), 0.0, 1.0))
        r_kv = np.maximum((r_kv * scale).astype(np.int32), 0)
    return w_s, w_o, w_a, w_bit, r_kv, r_rem


def _admit_both(B, oracle, policy, M, st, O0=179, O1=887):
    import torch
    w_s, w_o, w_a, w_bit, r_kv, r_rem = st
    rc, idx, words = oracle.admit(policy, M, 5, w_s, w_o, w_a, w_bit, O0, O1, r_kv, r_rem)
    out = B.svf_admit(policy, M, 5, _dev(w_s), _dev(w_o), _dev(w_a), _dev(w_bit), O0, O1, _dev(r_kv), _dev(r_rem))
    torch.cuda.synchronize()
    assert int(out.status.item()) == rc
    k = int(out.n_admitted.item())
    assert k == len(idx)
    assert np.array_equal(out.admitted_idx.cpu().numpy()[:k], idx)
    if rc == 0:
        assert np.array_equal(out.sorted_words.cpu().numpy().view(np.uint64)[: len(w_s)], words)
    return k


@pytest.mark.parametrize("n_wait,n_run", [(0, 0), (0, 50), (1, 0), (37, 0), (1024, 256), (5000, 1024),
                                           (5001, 1024), (70_000, 4096), (1 << 18, 300), (3000, 6000),
                                           (2049, 0), (3000, 1000), (4096, 0)])     # 2049..4096 entries: the 512-thread one-launch form
def test_admit_matches_oracle(B, oracle, n_wait, n_run):
    M = 1_000_000 if n_run <= 4096 else 6_000_000        # (3000, 6000): beyond the 4096 register slots
    if n_wait + n_run in (2049, 4096):
        M = 90_000                                       # tight: the bisection's answer lies inside the window
    st = _admit_state(n_wait + n_run, n_wait, n_run, M)
    ks = [_admit_both(B, oracle, policy, M, st) for policy in range(4)]
    if n_wait >= 1024 and n_run <= 1024:
        assert max(ks) > 0


def test_admit_512_thread_form_with_tied_remaining_steps(B, oracle):
    """2049..4096 entries take k_admit_prefix<true, 512> (its second scan level and shared-memory opt-in);
    here with a running set whose remaining steps are heavily tied (10 distinct values)."""
    w_s, w_o, w_a, w_bit, r_kv, r_rem = _admit_state(41, 2600, 900, 1_000_000)
    r_rem = (r_rem % 10 + 1).astype(np.int32) * 100
    for M in (700_000, 1_000_000, 1_400_000):
        ks = [_admit_both(B, oracle, policy, M, (w_s, w_o, w_a, w_bit, r_kv, r_rem)) for policy in range(4)]
    assert max(ks) > 0


def test_admit_wide_budget_takes_the_sorted_array_kernel(B, oracle):
    """M >= 2^30: the 32-bit slot passes are not exact any more; the 64-bit sorted-array path runs."""
    st = _admit_state(77, 4000, 500, 1_000_000)
    for M in ((1 << 30) - 1, 1 << 30, 5 << 30):
        k = _admit_both(B, oracle, 0, M, st)
        assert k == 4000                                  # everything fits


def test_admit_prefix_bisection_and_its_handover(B, oracle):
    """The bisection kernel holds running + the first (8192 - n_run) candidates.  Cases: the answer
    inside that window (tight budgets, every policy); the window exhausted with more waiting ->
    the serial kernels take over from the running order it wrote (32-bit slots and 64-bit path);
    n_run above 4096 -> the device-wide sort of the running set + the serial kernels; a running
    set that is infeasible on its own admits nobody."""
    for n_wait, n_run, M in ((9000, 0, 150_000), (9000, 700, 1_500_000), (30_000, 4096, 8_000_000),
                             (8192, 0, 60_000), (8193, 0, 10 ** 7), (5000, 3192, 6_000_000)):
        st = _admit_state(n_wait * 7 + n_run, n_wait, n_run, M)
        ks = [_admit_both(B, oracle, policy, M, st) for policy in range(4)]
        assert max(ks) > 0
    st = _admit_state(5, 20_000, 100, 1_000_000)
    assert _admit_both(B, oracle, 0, (1 << 30) - 1, st) == 20_000      # window exhausted: slot kernels finish
    assert _admit_both(B, oracle, 3, 1 << 40, st) == 20_000            # ... and the 64-bit kernel
    k = _admit_both(B, oracle, 0, 10_000_000, st)                      # handed over AND then blocked
    assert 8092 < k < 20_000
    st = _admit_state(6, 3000, 4097, 8_000_000)
    assert _admit_both(B, oracle, 0, 8_000_000, st) > 0                # n_run > 4096: serial path
    # the probe's 32-bit form needs M < 2^26 AND rem * count < 2^30; very long remaining times take the 64-bit form
    w_s, w_o, w_a, w_bit, r_kv, r_rem = _admit_state(8, 6000, 40, 1_000_000)
    long_rem = (r_rem.astype(np.int64) * 4000).astype(np.int32)        # up to 12,000,000 steps left
    for M in (60_000_000, 700_000_000, 2_000_000_000):
        assert _admit_both(B, oracle, 2, M, (w_s, w_o, w_a, w_bit, r_kv, long_rem)) >= 0
    w_s, w_o, w_a, w_bit, r_kv, r_rem = _admit_state(7, 500, 50, 1_000_000)
    r_kv = r_kv.copy(); r_kv[0] = 999_990                              # running set alone already over M at its first completion
    assert _admit_both(B, oracle, 0, 1_000_000, (w_s, w_o, w_a, w_bit, r_kv, r_rem)) == 0


def test_admit_everything_fits_and_nothing_fits(B, oracle):
    st = _admit_state(1, 300, 40, 10 ** 6)
    assert _admit_both(B, oracle, 0, 10 ** 12, st) == 300           # whole queue admitted
    assert _admit_both(B, oracle, 0, 10, st) == 0                   # running set already over M
    w_s, w_o, w_a, w_bit, r_kv, r_rem = st
    assert _admit_both(B, oracle, 2, int(r_kv.sum()) + int(r_rem.max()) * 40 + 1, st) >= 0


def test_admit_data_errors(B, oracle):
    base = _admit_state(2, 50, 10, 10 ** 6)
    def variant(f):
        st = [x.copy() for x in base]; f(st); return st
    cases = [variant(lambda st: st[1].__setitem__(7, 0)),            # o < 1 -> ERANGE
             variant(lambda st: st[2].__setitem__(9, 0)),            # arrivals decrease -> EUNSORTED
             variant(lambda st: (st[2].__setitem__(9, 0), st[0].__setitem__(30, -4))),  # first offender wins
             variant(lambda st: st[5].__setitem__(3, 0)),            # rem < 1 -> ERANGE
             variant(lambda st: (st[0].__setitem__(4, 2 ** 30), st[1].__setitem__(4, 2 ** 20)))]  # key overflow
    codes = []
    for st in cases:
        rc, _, _ = oracle.admit(0, 10 ** 6, 0, *st[:4], 2, 8, st[4], st[5])
        codes.append(rc)
        _admit_both(B, oracle, 0, 10 ** 6, st, 2, 8)
    assert codes == [16, 17, 17, 16, 19]


def test_admit_agrees_with_simulator_states(B, oracle):
    """Replay admission decisions at states taken from an oracle run of configs[1]: running set
    as (kv, rem), the waiting queue in arrival order."""
    tr = T.config2(1)
    ref = oracle.simulate(tr, 0)
    a, s, o = tr.arrival.astype(np.int64), tr.prompt.astype(np.int64), tr.output.astype(np.int64)
    k = ref.start.astype(np.int64)
    for t in (100, 300, 450, 520, 700):
        run = np.nonzero((k < t) & (k + o > t))[0]
        wait = np.nonzero((a <= t) & (k >= t))[0]
        st = (s[wait].astype(np.int32), o[wait].astype(np.int32), a[wait].astype(np.int32), tr.bit[wait],
              (s[run] + t - k[run]).astype(np.int32), (k[run] + o[run] - t).astype(np.int32))
        n_adm = _admit_both(B, oracle, 0, tr.M, st)
        assert n_adm == int((k[wait] == t).sum())


# ---------------------------------------------------------------------------------------------
# NEXT-2: the volume lower bound of Prop. 3.1
# ---------------------------------------------------------------------------------------------
def test_volume_lower_bound_matches_oracle(B, oracle):
    import torch
    parts = [T.random_small(700 + i, (i * 37) % 300, 60, 50, 10 ** 6) for i in range(40)]
    parts[7].output[3] = 0                                   # ERANGE
    cases = [T.concat(parts, "lb-ragged", 10 ** 6, 2, 8), T.config3(n_instances=50, n=1000, lam=4.0),
             T.config4(n=30_000), T.config5(n_instances=3)]
    for tr in cases:
        lb, st = B.svf_volume_lower_bound(B.DeviceTrace.from_host(tr))
        torch.cuda.synchronize()
        rlb, rst = oracle.volume_lower_bound(tr)
        assert np.array_equal(lb.cpu().numpy(), rlb), tr.name
        assert np.array_equal(st.cpu().numpy(), rst), tr.name
    # overflow is reported, not wrapped: 100,000 requests of volume 2.25e9 each -> 1.1e19 >= 2^63
    n = 100_000
    big = T._one("big", np.zeros(n, np.int32), np.full(n, 60_000), np.full(n, 30_000), np.zeros(n, np.uint8), 10 ** 9, 1, 1)
    lb, st = B.svf_volume_lower_bound(B.DeviceTrace.from_host(big))
    rlb, rst = oracle.volume_lower_bound(big)
    assert int(st[0]) == oracle.EOVERFLOW == int(rst[0]) and int(lb[0]) == 0 == int(rlb[0])


def test_ratio_to_lower_bound_at_scale(B, oracle):
    """Burst version of configs[2] at full size: M * TEL >= LB for every policy and instance
    (Prop. 3.1), and the SVF certificate of Thm 3.2's proof (TEL - sum o)(M - p_max) <= 2 LB
    (Lemma G.2 summed) -- properties that hold at any size, on GPU outputs only."""
    import torch
    tr = T.config3(n_instances=4096, lam=4.0)
    tr.arrival[:] = 0
    dt = B.DeviceTrace.from_host(tr)
    lb, st = B.svf_volume_lower_bound(dt)
    outs = B.svf_simulate_policies(dt, [0, 1, 2, 3], want=("total_latency", "status"))
    torch.cuda.synchronize()
    lb = lb.cpu().numpy()
    assert not st.cpu().numpy().any()
    sum_o = np.add.reduceat(tr.output.astype(np.int64), tr.offsets[:-1])
    pmax = np.maximum.reduceat(tr.prompt.astype(np.int64) + tr.output, tr.offsets[:-1])
    for pol, out in enumerate(outs):
        tel = out.total_latency.cpu().numpy()
        assert (tr.M * tel >= lb).all(), pol
    tel_svf = outs[0].total_latency.cpu().numpy()
    assert ((tel_svf - sum_o) * (tr.M - pmax) <= 2 * lb).all()
    sub = np.arange(0, 4096, 128)
    assert np.array_equal(lb[sub], oracle.volume_lower_bound(tr.subset(sub))[0])


def test_stochastic_reference_workload(B, oracle):
    """NEXT-3: Poisson arrivals, geometric outputs (App. H reference model), light and heavy load."""
    for lam, M in ((0.05, 300_000), (1.0, 300_000), (2.0, 120_000)):
        tr = T.stochastic(n_instances=48, n=600, lam=lam, M=M)
        for policy in range(4):
            check(B, oracle, tr, policy, ctx=f"{tr.name} M={M} policy {policy}")


def test_packed_waiting_records_and_their_fallback(B, oracle):
    """Instances of 2,049 .. 8,192 requests take the register queue with (s, o) packed into ONE word per
    rank, the split chosen per instance from the widths of its largest s and o; an instance whose
    widths do not fit 32 bits together (here 18 + 17) reads its records from global memory instead.
    Both in one call, under 16 (M = 200k) and 32 (M = 600k) register slots per thread."""
    def inst(j, n, wide):
        tr = T.config2(instance=300 + j, n=n, lam=6.0)
        s, o = tr.prompt.copy(), tr.output.copy()
        if wide:
            s[7], o[7] = 1 << 17, 3
            s[11], o[11] = 5, 1 << 16
        return T._one("", tr.arrival, s, o, (o > 256).astype(np.uint8), 0, 113, 572)
    for M in (200_000, 600_000):
        tr = T.concat([inst(0, 2100, False), inst(1, 3000, True), inst(2, 2049, True), inst(3, 5000, False)],
                      f"packed M={M}", M, 113, 572)
        for policy in (0, 1, 2, 3):
            ref, _ = check(B, oracle, tr, policy, ctx=f"{tr.name} policy {policy}")
            assert not ref.status.any()


def test_more_running_requests_than_register_slots(B, oracle):
    """Running sets far beyond the register slots of a group (512 per warp, 2048 / 4096 per CTA):
    the ext slots (global memory under the warp kernel, shared / global under the CTA kernels) hold
    the overflow.  Long outputs, small prompts, a budget that fits almost everything at once."""
    def crowd(I, n, seed):
        parts = []
        for j in range(I):
            sd = T.instance_seed(88, seed * 1000 + j)
            a = np.sort(T.uniform_int(sd, 1, n, 0, 40))
            s = T.uniform_int(sd, 2, n, 0, 6)
            o = T.uniform_int(sd, 3, n, 150, 400)
            parts.append(T._one("", a, s, o, (o > 250).astype(np.uint8), 0, 200, 300))
        return parts
    # (40 x 1500 at M = 800k: the one-warp kernel with 32 slots per thread, 1,024 register slots, the rest in ext slots)
    for I, n, M in ((40, 1000, 330_000), (600, 900, 200_000), (40, 1500, 800_000), (3, 5000, 1_500_000), (1, 9000, 2_500_000)):
        tr = T.concat(crowd(I, n, n), f"crowd{I}x{n}", M, 200, 300)
        for policy in (0, 1, 3):
            ref, got = check(B, oracle, tr, policy, ctx=f"{tr.name} policy {policy}")
        # the point of the case: most of an instance runs at once
        started_early = (ref.start[: tr.offsets[1]] < 150).sum()
        assert started_early > 0.6 * n


@pytest.mark.parametrize("rnd", range(8))
def test_fuzz_random_batches(B, oracle, rnd):
    """Seeded random batches over the whole parameter space of the kernels: instance sizes 0..2500
    (warp kernel, CTA kernels), arrival spreads 0..300, budgets from barely one request to hundreds
    of requests (blocked heads, ext slots), predicted keys on odd rounds, 1..4 policies per call."""
    sd = T.instance_seed(55, rnd)
    u = lambda stream, lo, hi: int(T.uniform_int(sd, stream, 1, lo, hi)[0])
    sc = (1, 10, 3)[rnd % 3]
    s_hi, o_hi = u(1, 1, 40 * sc), u(2, 1, 60 * sc)
    M = u(3, s_hi + o_hi, (6 if sc == 1 else 400) * (s_hi + o_hi) + 5)
    nmax = (12, 60, 300, 1100, 2500)[u(4, 0, 4)]
    I = 40 if nmax > 300 else u(5, 200, 1500)
    parts = []
    for i in range(I):
        si = T.instance_seed(56, rnd * 100_000 + i)
        n = int(T.uniform_int(si, 1, 1, 0, nmax)[0])
        a_hi = (0, 3, 30, 300)[int(T.uniform_int(si, 2, 1, 0, 3)[0])]
        parts.append(T.random_small(rnd * 100_000 + i, n, s_hi, o_hi, M, a_hi=a_hi, O0=1 + rnd, O1=7 + 5 * rnd))
    tr = T.concat(parts, f"fuzz{rnd}", M, 1 + rnd, 7 + 5 * rnd)
    if rnd % 2:
        tr = T.with_predicted_lengths(tr, sigma=0.7, seed=rnd, hi=max(2, 3 * o_hi))
    pols = [(rnd + k) % 4 for k in range(1 + rnd % 4)]
    import torch
    outs = B.svf_simulate_policies(B.DeviceTrace.from_host(tr), pols)
    torch.cuda.synchronize()
    for pol, out in zip(pols, outs):
        ref = oracle.simulate(tr, pol, n_threads=8)
        assert_same({k: getattr(out, k).cpu().numpy() for k in FIELDS}, ref, tr, f"fuzz {rnd} policy {pol}")


@pytest.mark.parametrize("rnd", range(3))
def test_fuzz_packed_register_queue(B, oracle, rnd):
    """The same over the sizes of the packed register queue (instances up to 8,192 requests): ragged
    sizes, budgets from a handful to hundreds of running requests (16 and 32 slots per thread, ext
    slots), bursts and spread arrivals, two policies per call."""
    sd = T.instance_seed(57, rnd)
    u = lambda stream, lo, hi: int(T.uniform_int(sd, stream, 1, lo, hi)[0])
    s_hi, o_hi = u(1, 20, 400), u(2, 20, 600)
    M = u(3, 4 * (s_hi + o_hi), (20, 300, 900)[rnd] * (s_hi + o_hi))
    parts = []
    for i in range(10):
        si = T.instance_seed(58, rnd * 1000 + i)
        n = int(T.uniform_int(si, 1, 1, 0, 8192)[0]) if i else 8192
        a_hi = (0, 30, 3000)[int(T.uniform_int(si, 2, 1, 0, 2)[0])]
        parts.append(T.random_small(rnd * 1000 + i + 77, n, s_hi, o_hi, M, a_hi=a_hi, O0=3, O1=40))
    tr = T.concat(parts, f"fuzz-packed{rnd}", M, 3, 40)
    pols = [rnd % 4, (rnd + 1) % 4]
    import torch
    outs = B.svf_simulate_policies(B.DeviceTrace.from_host(tr), pols)
    torch.cuda.synchronize()
    for pol, out in zip(pols, outs):
        ref = oracle.simulate(tr, pol, n_threads=8)
        assert_same({k: getattr(out, k).cpu().numpy() for k in FIELDS}, ref, tr, f"fuzz-packed {rnd} policy {pol}")
