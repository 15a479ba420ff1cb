"""Independent schedule validator (ORACLE side, test infrastructure only).

Takes a single-instance trace, ``M``, a policy and the ``start[]`` some simulator produced and
checks it against the paper's model *by the definitions*, sharing no code with
``oracle/svf_ref.c`` or with the CUDA path (numpy only):

 (i)   capacity: mem(t) = sum_{i: k_i < t <= f_i} (s_i + t - k_i) <= M for every t   (Eq. 3c)
 (ii)  area conservation: sum_t mem(t) == sum_i vol_i, vol_i = sum_{j=1..o_i} (s_i + j) (Eq. 1,
       P:L65, is the closed form of this sum)
 (iii) every request starts once at k_i >= a_i, finishes at k_i + o_i, latency >= o_i (Eq. 3b,
       P:L102, Lemma G.1)
 (iv)  greedy / no bypass: whenever j starts, every request ahead of j in the
       (key, arrival, id) order that had arrived by then has already started (the started set
       is a prefix of the sorted queue); and a request left at the head of a non-empty queue
       after the admissions at t would break the literal check if started at t.
"""
from __future__ import annotations

import numpy as np

SVF, SVF_1BIT, SJF, FCFS = 0, 1, 2, 3


def priority_keys(policy, a, s, o, bit, O0, O1):
    a, s, o = (np.asarray(x, dtype=np.int64) for x in (a, s, o))
    if policy == SVF:
        # area under the KV staircase: o rows of s tokens plus the triangle 1 + 2 + ... + o
        return s * o + (o * (o + 1)) // 2
    if policy == SVF_1BIT:
        Om = np.where(np.asarray(bit) != 0, np.int64(O1), np.int64(O0))
        return s * Om + (Om * (Om + 1)) // 2
    if policy == SJF:
        return o.copy()
    if policy == FCFS:
        return a.copy()
    raise ValueError(policy)


def memory_profile(a, s, o, start):
    """mem(t) for t = 0..T (T = last finish), by the definition, via difference arrays."""
    s, o, k = (np.asarray(x, dtype=np.int64) for x in (s, o, start))
    f = k + o
    T = int(f.max()) if len(f) else 0
    dA = np.zeros(T + 3, dtype=np.int64)   # sum of (s_i - k_i) over requests alive at t
    dB = np.zeros(T + 3, dtype=np.int64)   # number of requests alive at t
    np.add.at(dA, k + 1, s - k)
    np.add.at(dA, f + 1, -(s - k))
    np.add.at(dB, k + 1, 1)
    np.add.at(dB, f + 1, -1)
    A, B = np.cumsum(dA)[: T + 1], np.cumsum(dB)[: T + 1]
    t = np.arange(T + 1, dtype=np.int64)
    return A + B * t


def validate(trace, policy, start, M=None, finish=None, check_blocked="all", max_pairs=4_000_000,
             rng_seed=0, check_greedy=True):
    """Return a dict of facts about the schedule; raises AssertionError on any violation."""
    assert trace.n_instances == 1
    M = trace.M if M is None else M
    a, s, o = (np.asarray(x, dtype=np.int64) for x in (trace.arrival, trace.prompt, trace.output))
    k = np.asarray(start, dtype=np.int64)
    n = len(a)
    f = k + o
    # (iii)
    assert np.all(k >= a), "a request started before it arrived"
    if finish is not None:
        assert np.array_equal(np.asarray(finish, dtype=np.int64), f), "finish != start + o"
    lat = f - a
    assert np.all(lat >= o)
    # (i)
    mem = memory_profile(a, s, o, k)
    assert mem.max(initial=0) <= M, f"capacity exceeded: {mem.max()} > {M}"
    # (ii)
    vol = s * o + (o * (o + 1)) // 2
    assert int(mem.sum()) == int(vol.sum()), "area conservation violated"
    # (iv) prefix property
    # the ORDER may come from predicted lengths (trace.output_key); dynamics use the true o
    okey = getattr(trace, "output_key", None)
    o_for_key = o if okey is None else np.asarray(okey, dtype=np.int64)
    key = priority_keys(policy, a, s, o_for_key, trace.bit, trace.O0, trace.O1)
    order = np.lexsort((np.arange(n), a, key))          # ascending (key, arrival, id)
    pos = np.empty(n, dtype=np.int64)
    pos[order] = np.arange(n)
    if not check_greedy:                                 # model constraints only (e.g. OPT)
        check_blocked = 0
    elif n * n <= max_pairs:
        ahead = pos[:, None] < pos[None, :]              # i ahead of j
        present = a[:, None] <= k[None, :]               # i had arrived when j started
        bad = ahead & present & (k[:, None] > k[None, :])
        assert not bad.any(), "a request bypassed a higher-priority waiting request"
    else:
        rng = np.random.default_rng(rng_seed)
        js = rng.integers(0, n, size=max(1, max_pairs // n))
        for j in js:
            bad = (pos < pos[j]) & (a <= k[j]) & (k > k[j])
            assert not bad.any(), "a request bypassed a higher-priority waiting request"
    # (iv) blocked head: at each checked time t with a non-empty queue after admissions, the
    # head must fail the literal forward-looking check
    waited = np.nonzero(k > a)[0]
    times = np.unique(np.concatenate([np.arange(a[j], k[j]) for j in waited])) if len(waited) else np.zeros(0, np.int64)
    if check_blocked != "all" and int(check_blocked) == 0:
        times = times[:0]
    elif check_blocked != "all" and len(times) > int(check_blocked):
        rng = np.random.default_rng(rng_seed + 1)
        times = np.sort(rng.choice(times, size=int(check_blocked), replace=False))
    n_blocked_checked = 0
    for t in times:
        q = np.nonzero((a <= t) & (k > t))[0]            # waiting after the admissions at t
        if len(q) == 0:
            continue
        h = q[np.argmin(pos[q])]
        run = np.nonzero((k <= t) & (f > t))[0]
        horizon = int(max(f[run].max(initial=t), t + o[h]))
        tp = np.arange(t + 1, horizon + 1, dtype=np.int64)
        prof = np.zeros(len(tp), dtype=np.int64)
        for i in run:
            alive = tp <= f[i]
            prof += np.where(alive, s[i] + tp - k[i], 0)
        alive = tp <= t + o[h]
        prof += np.where(alive, s[h] + tp - t, 0)
        assert prof.max() > M, f"head {h} was left waiting at t={t} although it fits"
        n_blocked_checked += 1
    # rounds / decisions by their definitions (reading R16): a step t counts as a round iff some
    # request has arrived and not started before t; its decisions are the admissions at t plus
    # one blocked-head evaluation if somebody is still waiting afterwards
    T = int(f.max(initial=0))
    q_in = np.zeros(T + 2, dtype=np.int64)      # requests in the queue at t after ARRIVE: a<=t<=k
    np.add.at(q_in, a, 1)
    np.add.at(q_in, k + 1, -1)
    q_after = np.zeros(T + 2, dtype=np.int64)   # still waiting after ADMIT: a<=t<k
    np.add.at(q_after, a, 1)
    np.add.at(q_after, k, -1)
    q_in, q_after = np.cumsum(q_in)[: T + 1], np.cumsum(q_after)[: T + 1]
    rounds = int((q_in > 0).sum())
    decisions = int(n + (q_after > 0).sum())
    return {"rounds": rounds, "decisions": decisions, "total_latency": int(lat.sum()), "peak_kv": int(mem.max(initial=0)),
            "makespan": int(f.max(initial=0)), "blocked_checked": n_blocked_checked,
            "p99_latency": int(np.sort(lat)[(99 * n + 99) // 100 - 1]) if n else 0}
