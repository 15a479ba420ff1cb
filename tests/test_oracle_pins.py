"""Pins for the CPU oracle (oracle/svf_ref.c): things the paper and the mathematics fix, none of
them produced by the oracle itself or by the CUDA path.  CPU only (-m "not gpu")."""
import itertools
import os

import numpy as np
import pytest

from paper_2606_22327_b200 import traces as T

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
POL = {"svf": 0, "svf_1bit": 1, "sjf": 2, "fcfs": 3}


# --------------------------------------------------------------------------------------------
# P1: keys -- closed form Eq. 1 against the per-step memory of Eq. 3c
# --------------------------------------------------------------------------------------------
def test_volume_closed_form_equals_staircase_sum(oracle):
    ss, oo = np.meshgrid(np.arange(0, 65), np.arange(1, 65), indexing="ij")
    s, o = ss.ravel().astype(np.int32), oo.ravel().astype(np.int32)
    rc, words = oracle.keys(oracle.SVF, s, o)
    assert rc == 0
    # the area a request occupies: s + j tokens at its j-th step, j = 1..o
    expect = np.array([sum(int(si) + j for j in range(1, int(oi) + 1)) for si, oi in zip(s, o)],
                      dtype=np.uint64)
    assert np.array_equal(words >> np.uint64(32), expect)
    assert np.array_equal(words & np.uint64(0xFFFFFFFF), np.arange(len(s), dtype=np.uint64))


def test_proxy_volume_and_comparator_keys(oracle):
    s = np.array([5, 0, 7, 7], dtype=np.int32)
    o = np.array([3, 9, 1, 2], dtype=np.int32)
    a = np.array([0, 2, 2, 11], dtype=np.int32)
    bit = np.array([0, 1, 1, 0], dtype=np.uint8)
    rc, w = oracle.keys(oracle.SVF_1BIT, s, o, a, bit, 2, 8)
    # Eq. 2: s*O_m + (O_m^2+O_m)/2 with O_0=2 -> s*2+3, O_1=8 -> s*8+36
    assert rc == 0 and list(w >> np.uint64(32)) == [5 * 2 + 3, 0 * 8 + 36, 7 * 8 + 36, 7 * 2 + 3]
    rc, w = oracle.keys(oracle.SJF, s, o, a, bit, 2, 8)
    assert list(w >> np.uint64(32)) == [3, 9, 1, 2]
    rc, w = oracle.keys(oracle.FCFS, s, o, a, bit, 2, 8)
    assert list(w >> np.uint64(32)) == [0, 2, 2, 11]
    # key >= 2^32 is reported, not wrapped silently
    rc, _ = oracle.keys(oracle.SVF, np.array([65536], np.int32), np.array([65536], np.int32))
    assert rc == oracle.EOVERFLOW
    # 1-bit needs the bit array and proxies >= 1
    assert oracle.keys(oracle.SVF_1BIT, s, o, a, None, 2, 8)[0] == oracle.EINVAL
    assert oracle.keys(oracle.SVF_1BIT, s, o, a, bit, 0, 8)[0] == oracle.EINVAL
    # ... but an array nobody would read may be missing: n = 0 (include/svf.h conventions)
    e = np.zeros(0, np.int32)
    assert oracle.keys(oracle.SVF_1BIT, e, e, e, None, 2, 8)[0] == oracle.OK
    assert oracle.keys(oracle.SVF_1BIT, e, e, e, None, 0, 8)[0] == oracle.EINVAL
    rc, idx, _ = oracle.admit(oracle.SVF_1BIT, 100, 0, e, e, e, None, 2, 8, [5], [3])
    assert rc == oracle.OK and len(idx) == 0
    empty = T._one("empty", e, e, e, np.zeros(0, np.uint8), 100, 2, 8)
    empty.bit = None
    assert int(oracle.simulate(empty, oracle.SVF_1BIT).status[0]) == oracle.OK


@pytest.mark.parametrize("T_, b", [(16, 2), (81, 3), (256, 4)])
def test_eq35_sandwich_under_thm33_recipe(oracle, T_, b):
    """Eq. 35: v_hat / b^2 <= vol <= b^2 v_hat with theta = sqrt(T), O_0 = T^(1/4),
    O_1 = T^(3/4) (Thm 3.3), for every (s, o) with s + o <= T."""
    theta, O0, O1 = b * b, b, b ** 3
    so = [(s, o) for s in range(0, T_) for o in range(1, T_ + 1 - s)]
    s = np.array([x[0] for x in so], np.int32)
    o = np.array([x[1] for x in so], np.int32)
    bit = (o > theta).astype(np.uint8)
    vol = oracle.keys(oracle.SVF, s, o)[1] >> np.uint64(32)
    vhat = oracle.keys(oracle.SVF_1BIT, s, o, None, bit, O0, O1)[1] >> np.uint64(32)
    b2 = np.uint64(b * b)
    assert np.all(vhat <= b2 * vol) and np.all(vol <= b2 * vhat)


def test_table1_constants():
    """Table 1: 1 + 2/(1-alpha) = 5.00, 3.67, 3.22, 3.11, 3.02."""
    golden = {}
    for line in open(os.path.join(GOLDEN, "table1.txt")):
        if line.strip() and not line.startswith("#"):
            den, val = line.split()
            golden[int(den)] = float(val)
    assert set(golden) == {2, 4, 10, 20, 100}
    for den, val in golden.items():
        assert round(1 + 2 / (1 - 1 / den), 2) == val


# --------------------------------------------------------------------------------------------
# P2: literal FEASIBLE (Eq. 3c at every future step) == completion-time form
# --------------------------------------------------------------------------------------------
def test_feasible_literal_equals_completion_form(oracle):
    rng = np.random.default_rng(12345)
    n_true = 0
    for _ in range(20000):
        m = int(rng.integers(0, 9))
        kv = rng.integers(0, 12, size=m)
        rem = rng.integers(1, 10, size=m)
        # M near the peak so that both outcomes occur
        peak_guess = int((kv + rem).sum()) if m else 0
        M = int(rng.integers(max(0, peak_guess // 2), peak_guess + 2))
        lit = oracle.feasible(kv, rem, M, oracle.FEAS_LITERAL)
        com = oracle.feasible(kv, rem, M, oracle.FEAS_COMPLETION)
        assert lit == com
        # and against a third, direct statement in Python
        direct = all(sum(int(kv[i]) + d for i in range(m) if rem[i] >= d) <= M
                     for d in range(1, (int(rem.max()) if m else 0) + 1))
        assert lit == direct
        n_true += lit
    assert 2000 < n_true < 18000   # both outcomes exercised


def test_feasible_boundary_is_inclusive(oracle):
    # one request (kv=3, rem=4) peaks at 3+4=7 at its last step: feasible iff M >= 7 ("<=", Eq. 3c)
    assert oracle.feasible([3], [4], 7) and not oracle.feasible([3], [4], 6)
    assert oracle.feasible([3], [4], 7, oracle.FEAS_LITERAL)
    assert not oracle.feasible([3], [4], 6, oracle.FEAS_LITERAL)
    assert oracle.feasible([], [], 0)


# --------------------------------------------------------------------------------------------
# P4: hand-derived micro-examples (tests/golden/hand_examples.txt)
# --------------------------------------------------------------------------------------------
def _load_examples():
    ex, cur = [], None
    for line in open(os.path.join(GOLDEN, "hand_examples.txt")):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        tok = line.split()
        if tok[0] == "example":
            cur = {"name": tok[1], "M": int(tok[2].split("=")[1]),
                   "policy": POL[tok[3].split("=")[1]], "req": []}
            ex.append(cur)
        elif tok[0] == "req":
            cur["req"].append(tuple(int(x) for x in tok[1:4]))
        elif tok[0] == "start":
            cur["start"] = [int(x) for x in tok[1:]]
        elif tok[0] == "tel":
            cur["tel"] = int(tok[1])
    return ex


@pytest.mark.parametrize("ex", _load_examples(), ids=lambda e: e["name"])
@pytest.mark.parametrize("mode", [0, 1])
def test_hand_examples(oracle, ex, mode):
    a, s, o = (np.array(x, np.int32) for x in zip(*ex["req"]))
    tr = T._one(ex["name"], a, s, o, np.zeros(len(a), np.uint8), ex["M"], 1, 1)
    r = oracle.simulate(tr, ex["policy"], mode=mode)
    assert r.status[0] == 0
    assert list(r.start) == ex["start"]
    assert list(r.finish) == [k + int(oi) for k, oi in zip(ex["start"], o)]
    assert int(r.total_latency[0]) == ex["tel"]


# --------------------------------------------------------------------------------------------
# P5: degenerate reductions
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("policy", [0, 1, 2, 3])
def test_unbounded_memory_starts_everything_on_arrival(oracle, policy):
    tr = T.random_small(7, 60, 20, 15, M=10 ** 6, a_hi=25)
    r = oracle.simulate(tr, policy)
    assert np.array_equal(r.start, tr.arrival)
    assert int(r.total_latency[0]) == int(tr.output.sum())          # Lemma G.1 tight
    assert int(r.rounds[0]) == len(np.unique(tr.arrival))
    assert int(r.decisions[0]) == tr.n_requests


@pytest.mark.parametrize("s,o,m,r_", [(3, 4, 2, 0), (3, 4, 2, 3), (0, 5, 3, 0), (5, 1, 4, 2)])
def test_identical_requests_run_in_pure_batches(oracle, s, o, m, r_):
    """n identical (s, o), burst, M = m(s+o) + r, 0 <= r <= s: exactly m fit (each peaks at s+o
    in lockstep), so batch b (0-based) has latency (b+1) o."""
    n = 3 * m + 1
    M = m * (s + o) + r_
    tr = T._one("ident", np.zeros(n, np.int32), np.full(n, s, np.int32), np.full(n, o, np.int32),
                np.zeros(n, np.uint8), M, 1, 1)
    for policy in range(4):
        r = oracle.simulate(tr, policy)
        assert list(r.start) == [(i // m) * o for i in range(n)]
        assert int(r.total_latency[0]) == sum(((i // m) + 1) * o for i in range(n))
        assert int(r.peak_kv[0]) == m * (s + o)


def test_unit_outputs_reduce_to_prefix_packing(oracle):
    """all o_i = 1: each step admits the longest sorted prefix with sum (s_i + 1) <= M."""
    tr = T.random_small(11, 40, 9, 1, M=23)
    r = oracle.simulate(tr, oracle.SVF)
    order = np.lexsort((np.arange(40), tr.prompt.astype(np.int64) + 1))   # vol = s + 1
    t, i, expect = 0, 0, np.zeros(40, np.int64)
    while i < 40:
        load = 0
        while i < 40 and load + tr.prompt[order[i]] + 1 <= 23:
            load += tr.prompt[order[i]] + 1
            expect[order[i]] = t
            i += 1
        t += 1
    assert np.array_equal(r.start, expect)


def test_policy_coincidences(oracle):
    # equal prompts: volume is increasing in o, so SVF == SJF
    tr = T.random_small(3, 50, 0, 12, M=40)
    tr.prompt[:] = 6
    assert np.array_equal(oracle.simulate(tr, oracle.SVF).start, oracle.simulate(tr, oracle.SJF).start)
    # all keys equal: every policy is FCFS (ties broken by arrival then id)
    tr = T.random_small(4, 50, 0, 1, M=30, a_hi=10)
    tr.prompt[:] = 4
    tr.output[:] = 5
    tr.bit[:] = 1
    ref = oracle.simulate(tr, oracle.FCFS).start
    for p in (oracle.SVF, oracle.SVF_1BIT, oracle.SJF):
        assert np.array_equal(oracle.simulate(tr, p).start, ref)
    # all bits equal: 1-bit SVF orders by prompt size
    tr = T.random_small(5, 30, 10, 6, M=40)
    tr.bit[:] = 0
    r = oracle.simulate(tr, oracle.SVF_1BIT)
    order = np.lexsort((np.arange(30), tr.prompt))
    assert np.all(np.diff(r.start[order]) >= 0)


# --------------------------------------------------------------------------------------------
# literal and completion-time simulators agree; invalid inputs are rejected
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed", range(12))
def test_simulator_literal_equals_completion(oracle, seed):
    tr = T.random_small(100 + seed, 40, 10, 9, M=45, a_hi=(0 if seed % 2 else 30))
    for policy in range(4):
        r0 = oracle.simulate(tr, policy, mode=0)
        r1 = oracle.simulate(tr, policy, mode=1)
        for f in ("start", "finish", "total_latency", "p99_latency", "makespan", "peak_kv",
                  "rounds", "decisions", "status"):
            assert np.array_equal(getattr(r0, f), getattr(r1, f)), f


def test_invalid_instances_get_status_codes(oracle):
    def run(a, s, o, M=100, policy=0):
        tr = T._one("bad", np.array(a, np.int32), np.array(s, np.int32), np.array(o, np.int32),
                    np.zeros(len(a), np.uint8), M, 1, 1)
        return int(oracle.simulate(tr, policy).status[0])
    assert run([0, 1], [1, 1], [1, 1]) == oracle.OK
    assert run([0, 1], [1, 1], [0, 1]) == oracle.ERANGE
    assert run([0, 1], [-1, 1], [1, 1]) == oracle.ERANGE
    assert run([2, 1], [1, 1], [1, 1]) == oracle.EUNSORTED
    assert run([0, 1], [60, 1], [41, 1]) == oracle.EINFEASIBLE
    assert run([0, 2 ** 31 - 5], [1, 1], [3, 3], M=10) == oracle.EOVERFLOW
    assert run([0], [70000], [70000], M=10 ** 9) == oracle.EOVERFLOW
    # lowest-numbered failing check wins
    assert run([2, 1], [1, 1], [0, 1]) == oracle.ERANGE
    # a failing instance does not disturb its neighbours
    good = T.random_small(1, 10, 5, 5, M=30)
    bad = T._one("bad", np.array([3, 1], np.int32), np.array([1, 1], np.int32),
                 np.array([1, 1], np.int32), np.zeros(2, np.uint8), 30, 1, 1)
    both = T.concat([good, bad, good], "mix", 30, 2, 8)
    r = oracle.simulate(both, 0)
    assert list(r.status) == [0, oracle.EUNSORTED, 0]
    assert np.array_equal(r.start[:10], r.start[12:]) and np.all(r.start[10:12] == -1)
    assert r.total_latency[0] == r.total_latency[2] > 0 and r.total_latency[1] == 0


# --------------------------------------------------------------------------------------------
# stateless admit == what the simulator does at a step
# --------------------------------------------------------------------------------------------
def test_admit_matches_simulator_first_step(oracle):
    for seed in range(20):
        tr = T.random_small(200 + seed, 30, 10, 9, M=60)
        for policy in range(4):
            sim = oracle.simulate(tr, policy)
            rc, idx, words = oracle.admit(policy, tr.M, 0, tr.prompt, tr.output, tr.arrival,
                                          tr.bit, tr.O0, tr.O1, [], [])
            assert rc == 0
            assert sorted(idx.tolist()) == np.nonzero(sim.start == 0)[0].tolist()
            assert np.all(np.diff(words.astype(object)) > 0)
            assert np.array_equal(words[: len(idx)] & np.uint64(0xFFFFFFFF), idx.astype(np.uint64))
            rc2, idx2, _ = oracle.admit(policy, tr.M, 0, tr.prompt, tr.output, tr.arrival,
                                        tr.bit, tr.O0, tr.O1, [], [], mode=0)
            assert np.array_equal(idx, idx2)


def test_admit_with_a_running_set_hand_states(oracle):
    """svf_ref_admit with a NON-EMPTY running set, values derived by hand from Eq. 3c:
    a running member (kv, rem) holds kv + d tokens d steps from now, d = 1..rem; a request
    admitted now holds s + d for d = 1..o.
    State 1: running (kv 6, rem 1), head (s 2, o 3), M = 9: d=1 holds 7 + 3 = 10 > 9 -> blocked.
    State 2: running (kv 1, rem 6), same head: d=1..6 hold 2+3, 3+4, 4+5, 5, 6, 7 -> max 9 <= 9 ->
    admitted.  The two states are each other with kv and rem swapped, so a swap anywhere in the
    oracle's loading of the running set fails one of them.
    State 3: running A (3, 2), B (1, 4); waiting x (s 2, o 1; vol 3), y (s 1, o 3; vol 9), SVF order
    x, y.  With x: d=1 holds 4 + 2 + 3 = 9, d=2 holds 5 + 3 = 8.  With x and y: d=1 holds
    4 + 2 + 3 + 2 = 11, d=2 holds 5 + 3 + 3 = 11, d=3 holds 4 + 4 = 8, d=4 holds 5.  So M = 8 admits
    nobody, M = 9 and 10 admit x only, M = 11 admits both."""
    z = np.zeros(1, np.int32)
    for mode in (oracle.FEAS_LITERAL, oracle.FEAS_COMPLETION):
        rc, idx, _ = oracle.admit(oracle.SVF, 9, 0, [2], [3], z, None, 1, 1, [6], [1], mode=mode)
        assert rc == 0 and idx.tolist() == []
        rc, idx, _ = oracle.admit(oracle.SVF, 9, 0, [2], [3], z, None, 1, 1, [1], [6], mode=mode)
        assert rc == 0 and idx.tolist() == [0]
        rc, idx, _ = oracle.admit(oracle.SVF, 8, 0, [2], [3], z, None, 1, 1, [1], [6], mode=mode)
        assert rc == 0 and idx.tolist() == []                       # the boundary is inclusive: 9 > 8
        for M, want in ((8, []), (9, [1]), (10, [1]), (11, [1, 0]), (50, [1, 0])):
            # input order y, x (ids 0, 1): the priority order x, y is ids 1, 0
            rc, idx, _ = oracle.admit(oracle.SVF, M, 7, [1, 2], [3, 1], [0, 0], None, 1, 1, [3, 1], [2, 4], mode=mode)
            assert rc == 0 and idx.tolist() == want, (M, mode)


@pytest.mark.parametrize("policy", [0, 2, 3])
def test_admit_replays_simulator_states_with_running_sets(oracle, policy):
    """The stateless call on states taken from a simulation of configs[1] (n = 2000): at step t
    the running set is {i : k_i < t < k_i + o_i} with kv_i = s_i + t - k_i and rem_i = k_i + o_i - t
    computed HERE from the definition (Eq. 3c), the waiting queue is {i : a_i <= t <=
    k_i} in arrival order; the call must admit exactly the requests the simulator started at t, in
    priority order, under both statements of FEASIBLE."""
    tr = T.config2(1)
    ref = oracle.simulate(tr, policy)
    a, s, o = tr.arrival.astype(np.int64), tr.prompt.astype(np.int64), tr.output.astype(np.int64)
    k = ref.start.astype(np.int64)
    busy = np.unique(k[k > a])                         # steps that start somebody who had to wait
    times = [int(busy[i]) for i in np.linspace(0, len(busy) - 1, 7).astype(int)] + [int(a[50]), 100, 450]
    nonempty = 0
    for t in times:
        run = np.nonzero((k < t) & (k + o > t))[0]
        wait = np.nonzero((a <= t) & (k >= t))[0]
        kv, rem = s[run] + (t - k[run]), k[run] + o[run] - t
        started = wait[k[wait] == t]
        for mode in (oracle.FEAS_LITERAL, oracle.FEAS_COMPLETION):
            rc, idx, words = oracle.admit(policy, tr.M, t, s[wait], o[wait], a[wait], tr.bit[wait], tr.O0, tr.O1,
                                          kv, rem, mode=mode)
            assert rc == 0
            assert sorted(wait[idx].tolist()) == started.tolist(), (t, mode)
            # admitted = a PREFIX of the priority order (no bypass)
            assert np.array_equal(words[: len(idx)] & np.uint64(0xFFFFFFFF), idx.astype(np.uint64))
        nonempty += len(run) > 0 and len(started) > 0
    assert nonempty >= 5


def test_p99_is_the_nearest_rank_hand_values(oracle):
    """Reading R13: p99 = the ceil(0.99 n)-th smallest latency.  With a budget that admits everybody
    on arrival a request's latency is its o (Lemma G.1's equality case), so outputs 1..n in any order
    give latencies 1..n and p99 = ceil(0.99 n): 1, 8, 99, 100 and 1980 for n = 2000."""
    for n, want in ((1, 1), (8, 8), (100, 99), (101, 100), (199, 198), (200, 198), (2000, 1980)):
        o = np.arange(1, n + 1, dtype=np.int32)
        o = o[np.argsort(T.uniform(11, 3, n), kind="stable")]            # any order
        tr = T._one("p99", np.zeros(n, np.int32), np.ones(n, np.int32), o, np.zeros(n, np.uint8), 10 ** 9, 1, 1)
        r = oracle.simulate(tr, oracle.FCFS)
        assert int(r.total_latency[0]) == n * (n + 1) // 2
        assert int(r.p99_latency[0]) == want, n


# ---------------------------------------------------------------------------------------------
# NEXT-1: predicted output lengths order the queue, true lengths drive the model
# (deployable SVF / SJF vs Oracle-SVF / Oracle-SJF; reading R7)
# ---------------------------------------------------------------------------------------------
def test_predicted_keys_equal_to_true_lengths_change_nothing(oracle):
    tr = T.config3(n_instances=6, n=150, lam=4.0, M=40_000)
    same = T.with_predicted_lengths(tr, sigma=0.0)
    assert np.array_equal(same.output_key, tr.output)
    for policy in range(4):
        a, b = oracle.simulate(tr, policy), oracle.simulate(same, policy)
        assert np.array_equal(a.start, b.start) and np.array_equal(a.total_latency, b.total_latency)


def test_predicted_keys_hand_example(oracle):
    """Hand example A (tests/golden/hand_examples.txt: M=8, (s,o) = (2,3), (1,2), (3,1), burst).
    True SJF admits r2, r1 first: TEL 7.  With predictions (1, 2, 3) SJF's order is r0, r1, r2, the
    FCFS order, so by Eq. 3c: r0, r1 start at 0; r2 is blocked at t=0,1,2 (mem 9, 11, 9 > 8) and
    starts at 3: TEL = 3 + 2 + 4 = 9 -- the schedule derived by hand for FCFS."""
    tr = T._one("exA", np.zeros(3, np.int32), np.array([2, 1, 3]), np.array([3, 2, 1]), np.zeros(3, np.uint8), 8, 1, 1)
    true_sjf = oracle.simulate(tr, oracle.SJF)
    assert list(true_sjf.start) == [1, 0, 0] and int(true_sjf.total_latency[0]) == 7
    tr.output_key = np.array([1, 2, 3], np.int32)
    for mode in (oracle.FEAS_LITERAL, oracle.FEAS_COMPLETION):
        r = oracle.simulate(tr, oracle.SJF, mode=mode)
        assert list(r.start) == [0, 0, 3] and list(r.finish) == [3, 2, 4] and int(r.total_latency[0]) == 9
    # the true lengths still drive the dynamics: finish - start is the TRUE o
    assert np.array_equal(r.finish - r.start, tr.output)


def test_constant_prediction_orders_svf_by_prompt_like_equal_bits(oracle):
    """If every prediction is the same length c, Eq. 1 with o := c is s*c + c(c+1)/2: the order is
    by s, exactly what 1-bit SVF (Eq. 2) gives when every bit is 0 and O_0 = c -- a different key
    routine of the oracle reaching the same schedule."""
    for seed in range(6):
        tr = T.random_small(400 + seed, 40, 9, 11, 30, a_hi=25, O0=5, O1=9)
        tr.bit[:] = 0
        one_bit = oracle.simulate(tr, oracle.SVF_1BIT)
        tr.output_key = np.full(tr.n_requests, 5, np.int32)
        pred = oracle.simulate(tr, oracle.SVF)
        assert np.array_equal(pred.start, one_bit.start)
        # FCFS and 1-bit SVF never look at the predictions
        for policy in (oracle.SVF_1BIT, oracle.FCFS):
            assert np.array_equal(oracle.simulate(tr, policy).start, oracle.simulate(tr, policy, output_key=None).start)


@pytest.mark.parametrize("policy", [0, 2])
def test_predicted_keys_schedules_pass_the_validator(oracle, policy):
    """Noisy predictions: the schedule is still feasible, non-preemptive, greedy in the PREDICTED
    order with no bypass (validator (i)-(iv)), and latency >= true o."""
    from oracle import validator
    for seed in range(4):
        tr = T.with_predicted_lengths(T.random_small(500 + seed, 50, 9, 11, 26, a_hi=30), sigma=0.9, seed=seed, hi=40)
        r = oracle.simulate(tr, policy)
        facts = validator.validate(tr, policy, r.start, finish=r.finish)
        assert facts["peak_kv"] <= tr.M and facts["total_latency"] == int(r.total_latency[0])
    bad = T.with_predicted_lengths(T.random_small(1, 10, 9, 11, 26), sigma=0.5)
    bad.output_key[3] = 0
    assert int(oracle.simulate(bad, policy).status[0]) == oracle.ERANGE


# ---------------------------------------------------------------------------------------------
# NEXT-3: the stochastic reference workload of App. H -- generator facts the paper
# prints, and the oracle on it
# ---------------------------------------------------------------------------------------------
def test_geometric_reference_model_constants():
    """1/mu = 293 and a 4,096-token budget give Pr(o > 4096) ~ 8.29e-7;
    PAPER.md:953 (Eq. 101): E[o] = 1/mu, E[o^2] = (2-mu)/mu^2, E[vol] = E[s]/mu + 1/mu^2."""
    mu = 1.0 / 293.0
    assert abs((1.0 - mu) ** 4096 - 8.29e-7) < 0.005e-7
    o = T.geometric_int(T.instance_seed(6, 0), 4, 2_000_000, mu, 1 << 30).astype(np.float64)
    assert abs(o.mean() * mu - 1.0) < 0.005
    assert abs((o * o).mean() * mu * mu / (2.0 - mu) - 1.0) < 0.01
    assert o.min() == 1
    # the share of draws above the budget matches the geometric tail (1-mu)^k at a visible k
    assert abs((o > 1000).mean() / (1.0 - mu) ** 1000 - 1.0) < 0.03
    tr = T.stochastic(n_instances=200, n=1000, lam=1.0)
    vol = tr.prompt.astype(np.float64) * tr.output + (tr.output.astype(np.float64) ** 2 + tr.output) / 2
    assert abs(vol.mean() / (tr.prompt.mean() / mu + 1.0 / mu ** 2) - 1.0) < 0.03
    assert tr.O0 == 123 and tr.O1 == 586           # Thm 3.5 recipe at theta = 293


def test_oracle_on_the_stochastic_workload(oracle):
    """Under light load (rho << 1) nobody waits: TEL = sum o; the validator accepts the schedules
    under load; more load never helps (same requests, denser arrivals cannot lower SVF's TEL below
    sum o)."""
    from oracle import validator
    light = T.stochastic(n_instances=3, n=300, lam=0.05, M=300_000)
    r = oracle.simulate(light, oracle.SVF)
    assert int(r.total_latency.sum()) == light.request_steps
    heavy = T.stochastic(n_instances=2, n=300, lam=2.0, M=60_000)
    for policy in range(4):
        rr = oracle.simulate(heavy, policy)
        assert (rr.total_latency >= np.add.reduceat(heavy.output.astype(np.int64), heavy.offsets[:-1])).all()
        one = heavy.instance(0)
        r1 = oracle.simulate(one, policy)
        validator.validate(one, policy, r1.start, finish=r1.finish)
