"""Oracle pins II: brute-force hindsight optimum on tiny burst instances (config 1), the paper's
bounds (Thm 3.2, Prop. 3.1, Lemma G.1, Lemma G.2, Thm 3.3) and the independent validator."""
import itertools

import numpy as np
import pytest

from oracle import validator as V
from paper_2606_22327_b200 import traces as T


def _enumerate_opt(s, o, M):
    """Plain enumeration of all start-time vectors (no search tricks) for n <= 4."""
    n = len(s)
    H = int(sum(o))                      # a left-shifted schedule never starts later than this
    best = None
    for ks in itertools.product(range(H + 1), repeat=n):
        cost = sum(k + oi for k, oi in zip(ks, o))
        if best is not None and cost >= best:
            continue
        ok = True
        for t in range(1, H + max(o) + 1):
            mem = sum(si + t - k for si, oi, k in zip(s, o, ks) if k < t <= k + oi)
            if mem > M:
                ok = False
                break
        if ok:
            best = cost
    return best


def test_bruteforce_dfs_equals_plain_enumeration(oracle):
    rng = np.random.default_rng(5)
    for _ in range(25):
        n = int(rng.integers(2, 5))
        s = rng.integers(0, 5, size=n)
        o = rng.integers(1, 4, size=n)
        M = int(max(s + o) + rng.integers(0, 6))
        opt, start, _ = oracle.bruteforce_opt(s, o, M)
        assert opt == _enumerate_opt(list(map(int, s)), list(map(int, o)), M)
        tr = T._one("x", np.zeros(n, np.int32), s, o, np.zeros(n, np.uint8), M, 1, 1)
        info = V.validate(tr, 0, start, check_greedy=False)   # OPT need not be greedy
        assert info["total_latency"] == opt


N_SEEDS = 400


def test_config1_policies_vs_optimum_and_paper_bounds(oracle):
    """BASELINE.json configs[0]: n=8, burst, s,o ~ U{1..8}, M=32 (alpha <= 1/2)."""
    worst = 0.0
    n_opt_hit = 0
    for inst in range(N_SEEDS):
        tr = T.config1(inst)
        s, o = tr.prompt.astype(np.int64), tr.output.astype(np.int64)
        M = tr.M
        opt, _, nodes = oracle.bruteforce_opt(s, o, M)
        assert nodes < 5_000_000
        vol = s * o + o * (o + 1) // 2
        pmax = int((s + o).max())
        # Lemma G.1 and Prop. 3.1 hold for OPT itself
        assert opt >= int(o.sum())
        assert M * opt >= int(np.cumsum(np.sort(vol)).sum())
        tel = {}
        for policy in range(4):
            r = oracle.simulate(tr, policy)
            assert r.status[0] == 0
            tel[policy] = int(r.total_latency[0])
            assert tel[policy] >= opt                                    # OPT is a lower bound
            assert tel[policy] >= int(o.sum())                           # Lemma G.1
            assert M * tel[policy] >= int(np.cumsum(np.sort(vol)).sum())  # Prop. 3.1
            info = V.validate(tr, policy, r.start, finish=r.finish)
            for f in ("total_latency", "peak_kv", "makespan", "p99_latency", "rounds", "decisions"):
                assert info[f] == int(getattr(r, f)[0]), f
        # Thm 3.2: TEL(SVF) <= (1 + 2/(1-alpha)) OPT, alpha = pmax/M, in integers
        assert tel[0] * (M - pmax) <= opt * (3 * M - pmax)
        # Thm 3.3: 1-bit SVF <= (9T+1) OPT with T = 16 >= max(s+o); loose
        assert tel[1] <= (9 * 16 + 1) * opt
        worst = max(worst, tel[0] / opt)
        n_opt_hit += tel[0] == opt
        # Lemma G.2, integer form: W_j == 0 or W_j (M - pmax) < 2 sum_{i in P_j} vol_i
        r = oracle.simulate(tr, 0)
        order = np.lexsort((np.arange(len(s)), vol))
        pre = np.concatenate([[0], np.cumsum(vol[order])[:-1]])
        W = r.start[order].astype(np.int64)
        assert np.all((W == 0) | (W * (M - pmax) < 2 * pre))
    assert worst <= 5.0 and n_opt_hit > N_SEEDS // 10


@pytest.mark.parametrize("policy", [0, 1, 2, 3])
@pytest.mark.parametrize("seed", range(6))
def test_validator_accepts_oracle_on_random_online_instances(oracle, policy, seed):
    tr = T.random_small(300 + seed, 60, 12, 10, M=50, a_hi=(0 if seed % 3 == 0 else 40))
    r = oracle.simulate(tr, policy)
    info = V.validate(tr, policy, r.start, finish=r.finish)
    for f in ("total_latency", "peak_kv", "makespan", "p99_latency", "rounds", "decisions"):
        assert info[f] == int(getattr(r, f)[0]), f
    assert info["peak_kv"] <= tr.M


def test_validator_rejects_wrong_schedules(oracle):
    tr = T.random_small(42, 30, 10, 8, M=40)
    r = oracle.simulate(tr, 0)
    waited = np.nonzero(r.start > 0)[0]
    assert len(waited) > 3
    bad = r.start.copy()
    bad[waited[-1]] = 0                     # start a blocked request early -> over capacity
    with pytest.raises(AssertionError):
        V.validate(tr, 0, bad)
    late = r.start.copy()
    late[np.argmin(r.start)] += 50          # delay the first request: bypass / idle head
    with pytest.raises(AssertionError):
        V.validate(tr, 0, late)
    with pytest.raises(AssertionError):     # SVF schedule is not an FCFS-greedy schedule
        V.validate(tr, 3, r.start)


def test_config2_oracle_against_validator(oracle):
    """BASELINE.json configs[1]: n=2000 online trace, M=300k; SVF vs SJF vs FCFS (+1-bit)."""
    tr = T.config2()
    tel = {}
    for policy in range(4):
        r = oracle.simulate(tr, policy)
        assert r.status[0] == 0
        info = V.validate(tr, policy, r.start, finish=r.finish, check_blocked=40)
        for f in ("total_latency", "peak_kv", "makespan", "p99_latency", "rounds", "decisions"):
            assert info[f] == int(getattr(r, f)[0]), f
        tel[policy] = info["total_latency"]
        assert info["blocked_checked"] > 0
    assert tel[0] >= int(tr.output.astype(np.int64).sum())


# ---------------------------------------------------------------------------------------------
# NEXT-2: the volume lower bound of Prop. 3.1 as an output of its own
# ---------------------------------------------------------------------------------------------
def _burst(tr):
    tr.arrival[:] = 0
    return tr


def test_volume_lower_bound_closed_forms(oracle):
    """Eq. 5 against the weighted form Eq. 12: sum_i (N - i + 1) vol_(i), computed
    here in Python integers from the staircase definition of the volume (Eq. 3c), and against a
    value worked out by hand."""
    # by hand: (s, o) = (2,3), (1,2), (3,1): volumes 12, 5, 4 -> sorted 4, 5, 12 -> 4 + 9 + 21 = 34
    tr = T._one("exA", np.zeros(3, np.int32), np.array([2, 1, 3]), np.array([3, 2, 1]), np.zeros(3, np.uint8), 8, 1, 1)
    lb, st = oracle.volume_lower_bound(tr)
    assert int(lb[0]) == 34 and int(st[0]) == 0
    parts = [T.random_small(900 + i, 1 + 7 * i, 40, 30, 10 ** 6) for i in range(12)]
    tr = T.concat(parts, "lb", 10 ** 6, 2, 8)
    lb, st = oracle.volume_lower_bound(tr)
    for j, p_ in enumerate(parts):
        vol = sorted(sum(int(s) + k for k in range(1, int(o) + 1)) for s, o in zip(p_.prompt, p_.output))
        n = len(vol)
        assert int(lb[j]) == sum((n - i) * v for i, v in enumerate(vol)) and int(st[j]) == 0
    # identical requests: LB = vol * N (N + 1) / 2; empty instance: 0
    tr = T._one("same", np.zeros(50, np.int32), np.full(50, 7), np.full(50, 4), np.zeros(50, np.uint8), 100, 1, 1)
    assert int(oracle.volume_lower_bound(tr)[0][0]) == (7 * 4 + 10) * 50 * 51 // 2
    bad = T.random_small(3, 5, 9, 9, 50)
    bad.output[2] = 0
    assert int(oracle.volume_lower_bound(bad)[1][0]) == oracle.ERANGE
    # Eq. 5 sets no width on a volume: the bound is exact also where a volume passes 2^32 (a width the
    # CUDA library's 32-bit presort keys refuse, R19 -- its limit, tested on the GPU side).  By hand:
    # s = o = 60,000: 60000^2 + 60000*60001/2 = 5,400,030,000 >= 2^32 = 4,294,967,296;
    # s = 30,000, o = 60,000: 3,600,030,000;  LB = 2 * 3,600,030,000 + 5,400,030,000 = 12,600,090,000
    below = T._one("below", np.zeros(2, np.int32), np.array([30_000, 30_000]), np.array([60_000, 60_000]), np.zeros(2, np.uint8), 10 ** 9, 1, 1)
    lb, st = oracle.volume_lower_bound(below)
    assert int(st[0]) == 0 and int(lb[0]) == 3 * 3_600_030_000
    mixed = T._one("mixed", np.zeros(2, np.int32), np.array([60_000, 30_000]), np.array([60_000, 60_000]), np.zeros(2, np.uint8), 10 ** 9, 1, 1)
    lb, st = oracle.volume_lower_bound(mixed)
    assert int(st[0]) == 0 and int(lb[0]) == 12_600_090_000
    assert oracle.keys(oracle.SVF, mixed.prompt, mixed.output)[0] == oracle.EOVERFLOW       # as a KEY it is still refused (R11)
    # the largest requests the arrays can hold: volumes near 2^62.6, two of them still fit, five do not
    big = lambda n: T._one("big", np.zeros(n, np.int32), np.full(n, 2 ** 31 - 1), np.full(n, 2 ** 31 - 1), np.zeros(n, np.uint8), 10 ** 9, 1, 1)
    v = (2 ** 31 - 1) ** 2 + ((2 ** 31 - 1) ** 2 + (2 ** 31 - 1)) // 2
    lb, st = oracle.volume_lower_bound(big(1))
    assert int(st[0]) == 0 and int(lb[0]) == v
    lb, st = oracle.volume_lower_bound(big(5))                                          # 15 v >= 2^63
    assert 15 * v >= 2 ** 63 and int(st[0]) == oracle.EOVERFLOW and int(lb[0]) == 0


def test_volume_lower_bound_bounds_every_schedule_and_the_optimum(oracle):
    """M * TEL >= LB for the brute-force optimum and for all four policies on burst input
    (Prop. 3.1); and the SVF certificate of Thm 3.2's proof (Lemma G.2 summed over requests,
    P:L503-505): (TEL(SVF) - sum o) (M - p_max) <= 2 LB."""
    for seed in range(40):
        tr = T.config1(seed)
        lb = int(oracle.volume_lower_bound(tr)[0][0])
        opt, _, _ = oracle.bruteforce_opt(tr.prompt, tr.output, tr.M)
        assert tr.M * opt >= lb
        for policy in range(4):
            assert tr.M * int(oracle.simulate(tr, policy).total_latency[0]) >= lb
    for seed in range(10):
        tr = _burst(T.config3(n_instances=1, n=400, lam=4.0, M=60_000, first_instance=seed))
        lb = int(oracle.volume_lower_bound(tr)[0][0])
        tel = int(oracle.simulate(tr, oracle.SVF).total_latency[0])
        pmax = int((tr.prompt.astype(np.int64) + tr.output).max())
        assert tr.M * tel >= lb
        assert (tel - tr.request_steps) * (tr.M - pmax) <= 2 * lb
