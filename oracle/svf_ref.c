/*
 * oracle/svf_ref.c -- CPU ORACLE (test infrastructure, NOT the product).
 *
 * A plain, slow, step-by-step implementation of the scheduling model and policies of
 * "Geometry-Aware Online Scheduling for LLM Serving" (arxiv/paper_2606_22327), written from
 * /root/reference/PAPER.md ("P:L<n>" = PAPER.md line n).  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code, header,
 * table or helper with the CUDA path under paper_2606_22327_b200/csrc/ and neither includes the
 * other.  All arithmetic is integer (int64 intermediates); there is no floating point.
 *
 * What it follows, in the paper's order and notation:
 *   - model (Eq. 3a-3d): discrete time, capacity M, request i = (a_i, s_i, o_i);
 *     started at k_i >= a_i it holds s_i + (t - k_i) tokens at every t in {k_i+1..k_i+o_i}
 *     (Eq. 3c, index range max{a_i, t-o_i} <= k <= t-1), finishes at f_i = k_i + o_i, latency
 *     f_i - a_i, never preempted; mem(t) <= M for every t ("<=", Eq. 3c).
 *   - keys: volume v_i = s_i o_i + (o_i^2 + o_i)/2 (Eq. 1); proxy volume
 *     s_i O_m + (O_m^2 + O_m)/2 with m = bit_i (Eq. 2); SJF key o_i, FCFS key a_i
 *     (P:L37).
 *   - order: ascending key, ties "arbitrary but unique, consistently applied"
 *      -- fixed here as (key, arrival, id), "strict FCFS within identical priorities"
 *     (P:L969); id = index in the arrival-sorted trace.
 *   - engine loop (Alg. 1 Process 2): while capacity, pop the highest priority
 *     request into the running batch; then execute one step for the whole batch.
 *   - "capacity" = the forward-looking memory check: admit the head iff no
 *     future time t' > t exceeds M with it added; a blocked head is never bypassed.
 *   - order of events in a step (reading R1): complete, arrive, admit, advance.
 *
 * Two statements of FEASIBLE are kept side by side (tests check they agree):
 *   feas_mode 0 "literal": for every t' in (t, max f] sum the memory of every member alive
 *                          at t' (Eq. 3c written out);
 *   feas_mode 1 "completion-time": memory of a fixed set rises by |alive| per step and falls
 *                          only after a completion, so maxima sit at completion times
 *                          ("at some future completion time t_peak"): with members
 *                          ordered by remaining steps descending, mem_j = sum_{i<=j} kv_i
 *                          + rem_j * j; feasible iff max_j mem_j <= M.
 *
 * Pins: see tests/test_oracle_*.py (closed forms, hand examples from Eq. 3c, brute-force OPT,
 * Thm 3.2 / Prop. 3.1 / Lemma G.1 / Lemma G.2 bounds, degenerate reductions, an independent
 * schedule validator).  Unpinned conventions: the tie-break choice and the 1-bit harness
 * constants (they are inputs / conventions, not checkable against the paper).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

enum { POL_SVF = 0, POL_SVF_1BIT = 1, POL_SJF = 2, POL_FCFS = 3 };

/* status codes: the numbering is part of the boundary contract (include/svf.h states it in
 * prose); the oracle defines its own copies on purpose. */
enum {
    ST_OK = 0, ST_EINVAL = 1,
    ST_ERANGE = 16,      /* o_i < 1, s_i < 0 or a_i < 0                                   */
    ST_EUNSORTED = 17,   /* arrivals decrease inside an instance                          */
    ST_EINFEASIBLE = 18, /* s_i + o_i > M: could never be admitted (paper assumes <= aM)  */
    ST_EOVERFLOW = 19    /* key >= 2^32, or max a + sum o >= 2^31 (horizon)        */
};

/* ------------------------------------------------------------------------------------------
 * Keys (Eq. 1, Eq. 2; SJF / FCFS comparators).  Returns -1 for an unknown policy.
 * ---------------------------------------------------------------------------------------- */
static int64_t ref_key(int policy, int64_t s, int64_t o, int64_t a, int bit, int64_t O0,
                       int64_t O1)
{
    switch (policy) {
    case POL_SVF:      return s * o + (o * o + o) / 2;                 /* Eq. 1 */
    case POL_SVF_1BIT: { int64_t Om = bit ? O1 : O0;                   /* Eq. 2 */
                         return s * Om + (Om * Om + Om) / 2; }
    case POL_SJF:      return o;
    case POL_FCFS:     return a;
    default:           return -1;
    }
}

int svf_ref_keys(int policy, int64_t n, const int32_t *s, const int32_t *o, const int32_t *a,
                 const uint8_t *bit, int32_t O0, int32_t O1, uint64_t *words_out)
{
    if (policy < 0 || policy > 3 || n < 0) return ST_EINVAL;
    /* boundary rule (include/svf.h, "bit"): the bit array is required only when there is a request to read it for */
    if (policy == POL_SVF_1BIT && ((n > 0 && !bit) || O0 < 1 || O1 < 1)) return ST_EINVAL;
    int rc = ST_OK;
    for (int64_t i = 0; i < n; ++i) {
        int64_t k = ref_key(policy, s[i], o[i], a ? a[i] : 0, bit ? bit[i] : 0, O0, O1);
        if (k < 0 || k >= ((int64_t)1 << 32)) rc = ST_EOVERFLOW;
        /* packed (key, arrival, id) word: id = rank in (arrival, id) order = index i */
        words_out[i] = ((uint64_t)k << 32) + (uint64_t)(uint32_t)i;
    }
    return rc;
}

/* ------------------------------------------------------------------------------------------
 * FEASIBLE on a set given as (kv_i, rem_i): kv_i = tokens held now, rem_i = steps left.
 * Member i holds kv_i + d tokens d steps from now, for d = 1..rem_i.
 * ---------------------------------------------------------------------------------------- */
typedef struct { int64_t kv, rem; } member_t;

static int feasible_literal(const member_t *S, int64_t m, int64_t M)
{
    int64_t maxrem = 0;
    for (int64_t i = 0; i < m; ++i) if (S[i].rem > maxrem) maxrem = S[i].rem;
    for (int64_t d = 1; d <= maxrem; ++d) {          /* every future time t' = t + d */
        int64_t mem = 0;
        for (int64_t i = 0; i < m; ++i)
            if (S[i].rem >= d) mem += S[i].kv + d;   /* Eq. 3c term s_i + t' - k_i */
        if (mem > M) return 0;
    }
    return 1;
}

/* sort by remaining steps, descending (plain insertion sort: the sets handed in are almost
 * in order already, so this is one pass in practice and still obviously a sort) */
static void sort_rem_desc(member_t *S, int64_t m)
{
    for (int64_t i = 1; i < m; ++i) {
        member_t x = S[i];
        int64_t j = i;
        while (j > 0 && S[j - 1].rem < x.rem) { S[j] = S[j - 1]; --j; }
        S[j] = x;
    }
}

static int feasible_completion(member_t *S, int64_t m, int64_t M)
{
    sort_rem_desc(S, m);
    int64_t pre = 0;
    for (int64_t j = 0; j < m; ++j) {                /* j+1 members are alive at t + rem_j */
        pre += S[j].kv;
        if (pre + S[j].rem * (j + 1) > M) return 0;
    }
    return 1;
}

/* exported for the pin "literal == completion-time form" on random states */
int svf_ref_feasible(int feas_mode, int64_t m, const int64_t *kv, const int64_t *rem, int64_t M)
{
    member_t *S = (member_t *)malloc(sizeof(member_t) * (size_t)(m > 0 ? m : 1));
    for (int64_t i = 0; i < m; ++i) { S[i].kv = kv[i]; S[i].rem = rem[i]; }
    int r = feas_mode == 0 ? feasible_literal(S, m, M) : feasible_completion(S, m, M);
    free(S);
    return r;
}

/* ------------------------------------------------------------------------------------------
 * Waiting queue: plain array kept sorted on (key, arrival, id).  svf_ref_admit sorts it
 * ascending once; the simulator keeps it DESCENDING so that the head (smallest) is the last
 * element and Pop is n_wait-- (sorted insert by binary search + memmove).
 * ---------------------------------------------------------------------------------------- */
typedef struct { int64_t key; int32_t arrival; int32_t id; } waiter_t;

static int waiter_less(const waiter_t *x, const waiter_t *y)
{
    if (x->key != y->key) return x->key < y->key;
    if (x->arrival != y->arrival) return x->arrival < y->arrival;
    return x->id < y->id;
}

static int cmp_waiter(const void *x, const void *y)
{
    const waiter_t *a = (const waiter_t *)x, *b = (const waiter_t *)y;
    if (waiter_less(a, b)) return -1;
    if (waiter_less(b, a)) return 1;
    return 0;
}

static int cmp_i64(const void *x, const void *y)
{
    int64_t a = *(const int64_t *)x, b = *(const int64_t *)y;
    return a < b ? -1 : (a > b ? 1 : 0);
}

/* ------------------------------------------------------------------------------------------
 * svf_ref_admit: one stateless admission decision (steps a1-a5 of the hot path).
 * Waiting requests are given in (arrival, id) order (arrivals non-decreasing), running
 * requests as (kv, rem).  Admits the longest prefix of the priority order whose members are
 * jointly feasible with the running set, one at a time, stopping at the first blocked head.
 * ---------------------------------------------------------------------------------------- */
int svf_ref_admit(int policy, int64_t M, int32_t t, int feas_mode,
                  int64_t n_wait, const int32_t *w_s, const int32_t *w_o, const int32_t *w_a,
                  const uint8_t *w_bit, int32_t O0, int32_t O1,
                  int64_t n_run, const int32_t *r_kv, const int32_t *r_rem,
                  int64_t *n_admitted_out, int32_t *admitted_idx_out, uint64_t *sorted_words_out)
{
    (void)t; /* the check is relative to "now"; t only dates the decision */
    if (policy < 0 || policy > 3 || n_wait < 0 || n_run < 0 || M < 0) return ST_EINVAL;
    if (policy == POL_SVF_1BIT && ((n_wait > 0 && !w_bit) || O0 < 1 || O1 < 1)) return ST_EINVAL;
    for (int64_t i = 0; i < n_wait; ++i) {
        if (w_o[i] < 1 || w_s[i] < 0 || w_a[i] < 0) return ST_ERANGE;
        if (i > 0 && w_a[i] < w_a[i - 1]) return ST_EUNSORTED;
    }
    for (int64_t i = 0; i < n_run; ++i)
        if (r_rem[i] < 1 || r_kv[i] < 0) return ST_ERANGE;

    waiter_t *Q = (waiter_t *)malloc(sizeof(waiter_t) * (size_t)(n_wait > 0 ? n_wait : 1));
    for (int64_t i = 0; i < n_wait; ++i) {
        Q[i].key = ref_key(policy, w_s[i], w_o[i], w_a[i], w_bit ? w_bit[i] : 0, O0, O1);
        if (Q[i].key >= ((int64_t)1 << 32)) { free(Q); return ST_EOVERFLOW; }
        Q[i].arrival = w_a[i];
        Q[i].id = (int32_t)i;
    }
    qsort(Q, (size_t)n_wait, sizeof(waiter_t), cmp_waiter);
    if (sorted_words_out)
        for (int64_t i = 0; i < n_wait; ++i)
            sorted_words_out[i] = ((uint64_t)Q[i].key << 32) + (uint64_t)(uint32_t)Q[i].id;

    member_t *S = (member_t *)malloc(sizeof(member_t) * (size_t)(n_run + n_wait + 1));
    member_t *tmp = (member_t *)malloc(sizeof(member_t) * (size_t)(n_run + n_wait + 1));
    int64_t m = 0;
    for (int64_t i = 0; i < n_run; ++i) { S[m].kv = r_kv[i]; S[m].rem = r_rem[i]; ++m; }
    int64_t k = 0;
    while (k < n_wait) {
        int32_t h = Q[k].id;
        S[m].kv = w_s[h]; S[m].rem = w_o[h];          /* started now: holds s_h, o_h steps left */
        memcpy(tmp, S, sizeof(member_t) * (size_t)(m + 1));
        int ok = feas_mode == 0 ? feasible_literal(tmp, m + 1, M)
                                : feasible_completion(tmp, m + 1, M);
        if (!ok) break;                               /* blocked head: nobody may bypass it */
        if (admitted_idx_out) admitted_idx_out[k] = h;
        if (feas_mode != 0) memcpy(S, tmp, sizeof(member_t) * (size_t)(m + 1)); /* keep S in order */
        ++m; ++k;
    }
    *n_admitted_out = k;
    free(S); free(tmp); free(Q);
    return ST_OK;
}

/* ------------------------------------------------------------------------------------------
 * One instance of the time-stepped simulator (SURVEY 8(c) / DESIGN.md 3).
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    int64_t total_latency, p99_latency, peak_kv, rounds, decisions;
    int32_t makespan, status;
} inst_result_t;

/* okey (may be NULL): PREDICTED output lengths, used for the SVF / SJF priority key only (the
 * paper's deployable SVF / SJF; NULL = the true lengths = "Oracle SVF / SJF").
 * Dynamics and the feasibility check always use the true o (reading R7). */
static int64_t key_len(const int32_t *o, const int32_t *okey, int64_t i) { return okey ? okey[i] : o[i]; }

static int32_t validate_instance(int policy, int64_t n, const int32_t *a, const int32_t *s,
                                 const int32_t *o, const int32_t *okey, const uint8_t *bit,
                                 int64_t O0, int64_t O1, int64_t M)
{
    int range = 0, unsorted = 0, infeasible = 0, overflow = 0;
    int64_t sum_o = 0, max_a = 0;
    for (int64_t i = 0; i < n; ++i) {
        if (o[i] < 1 || s[i] < 0 || a[i] < 0 || (okey && okey[i] < 1)) range = 1;
        if (i > 0 && a[i] < a[i - 1]) unsorted = 1;
        if ((int64_t)s[i] + o[i] > M) infeasible = 1;
        if (ref_key(policy, s[i], key_len(o, okey, i), a[i], bit ? bit[i] : 0, O0, O1) >= ((int64_t)1 << 32))
            overflow = 1;
        sum_o += o[i] > 0 ? o[i] : 0;
        if (a[i] > max_a) max_a = a[i];
    }
    if (max_a + sum_o >= ((int64_t)1 << 31)) overflow = 1;   /* horizon bound */
    if (range) return ST_ERANGE;               /* the lowest-numbered failing check wins */
    if (unsorted) return ST_EUNSORTED;
    if (infeasible) return ST_EINFEASIBLE;
    if (overflow) return ST_EOVERFLOW;
    return ST_OK;
}

static void simulate_instance(int policy, int64_t M, int feas_mode, int64_t n,
                              const int32_t *a, const int32_t *s, const int32_t *o,
                              const int32_t *okey, const uint8_t *bit, int64_t O0, int64_t O1,
                              int32_t *start, int32_t *finish, inst_result_t *res)
{
    memset(res, 0, sizeof(*res));
    for (int64_t i = 0; i < n; ++i) { if (start) start[i] = -1; if (finish) finish[i] = -1; }
    res->status = validate_instance(policy, n, a, s, o, okey, bit, O0, O1, M);
    if (res->status != ST_OK || n == 0) return;

    int32_t *k = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);      /* start times k_i */
    int32_t *running = (int32_t *)malloc(sizeof(int32_t) * (size_t)n);
    waiter_t *waiting = (waiter_t *)malloc(sizeof(waiter_t) * (size_t)n);
    member_t *S = (member_t *)malloc(sizeof(member_t) * (size_t)(n + 1));
    int64_t *lat = (int64_t *)malloc(sizeof(int64_t) * (size_t)n);
    int64_t n_run = 0, n_wait = 0, next_arrival = 0, n_finished = 0;

    int64_t t = a[0];                                 /* arrivals are sorted: min_i a_i */
    int64_t peak = 0;
    while (n_finished < n) {
        /* 1. COMPLETE: every running i with k_i + o_i == t */
        int64_t w = 0;
        for (int64_t r = 0; r < n_run; ++r) {
            int32_t i = running[r];
            if ((int64_t)k[i] + o[i] == t) {
                if (finish) finish[i] = (int32_t)t;
                lat[i] = t - a[i];                    /* latency (t + o_i) - a_i */
                ++n_finished;
            } else running[w++] = i;
        }
        n_run = w;
        /* 2. ARRIVE: every not-yet-queued i with a_i <= t, sorted insert */
        while (next_arrival < n && a[next_arrival] <= t) {
            int32_t i = (int32_t)next_arrival++;
            waiter_t x;
            x.key = ref_key(policy, s[i], key_len(o, okey, i), a[i], bit ? bit[i] : 0, O0, O1);
            x.arrival = a[i]; x.id = i;
            int64_t lo = 0, hi = n_wait;              /* first position whose waiter < x */
            while (lo < hi) {
                int64_t mid = (lo + hi) / 2;
                if (waiter_less(&waiting[mid], &x)) hi = mid; else lo = mid + 1;
            }
            memmove(waiting + lo + 1, waiting + lo, sizeof(waiter_t) * (size_t)(n_wait - lo));
            waiting[lo] = x; ++n_wait;
        }
        /* 3. ADMIT: pop the head while the forward-looking check passes */
        if (n_wait > 0) {
            res->rounds += 1;
            int64_t admitted = 0;
            while (n_wait > 0) {
                int32_t h = waiting[n_wait - 1].id;   /* head: smallest (key, arrival, id) */
                for (int64_t r = 0; r < n_run; ++r) {
                    int32_t i = running[r];
                    S[r].kv = (int64_t)s[i] + (t - k[i]);
                    S[r].rem = (int64_t)k[i] + o[i] - t;
                }
                S[n_run].kv = s[h]; S[n_run].rem = o[h];
                int ok = feas_mode == 0 ? feasible_literal(S, n_run + 1, M)
                                        : feasible_completion(S, n_run + 1, M);
                if (!ok) break;                       /* blocked head: no bypass */
                k[h] = (int32_t)t;
                if (start) start[h] = (int32_t)t;
                /* running is kept ordered by finish time, latest first (any order is valid;
                 * this one makes the sort inside FEASIBLE a single pass) */
                int64_t pos = n_run;
                while (pos > 0 && (int64_t)k[running[pos - 1]] + o[running[pos - 1]] < t + o[h]) {
                    running[pos] = running[pos - 1]; --pos;
                }
                running[pos] = h; ++n_run;
                --n_wait;                             /* Pop(Q_wait) */
                ++admitted;
            }
            res->decisions += admitted;
            if (n_wait > 0) res->decisions += 1;      /* one blocked-head evaluation */
        }
        /* 4. ADVANCE: every running request grew one token; mem(t) by Eq. 3c counts the
         *    requests finishing AT t (they are removed at the next COMPLETE) */
        t += 1;
        int64_t mem = 0;
        for (int64_t r = 0; r < n_run; ++r) mem += (int64_t)s[running[r]] + (t - k[running[r]]);
        if (mem > peak) peak = mem;
    }
    int64_t tel = 0, mk = 0;
    for (int64_t i = 0; i < n; ++i) {
        tel += lat[i];
        if ((int64_t)k[i] + o[i] > mk) mk = (int64_t)k[i] + o[i];
    }
    qsort(lat, (size_t)n, sizeof(int64_t), cmp_i64);
    int64_t rank = (99 * n + 99) / 100;               /* nearest rank ceil(0.99 n), 1-based */
    res->total_latency = tel;
    res->p99_latency = lat[rank - 1];
    res->makespan = (int32_t)mk;
    res->peak_kv = peak;
    free(k); free(running); free(waiting); free(S); free(lat);
}

/* ------------------------------------------------------------------------------------------
 * svf_ref_simulate: every instance independently (instance-parallel over n_threads host
 * threads when built with OpenMP; each instance itself is one serial step chain).
 * Any output pointer may be NULL.
 * ---------------------------------------------------------------------------------------- */
int svf_ref_simulate_pred(int64_t n_instances, const int64_t *offsets, const int32_t *arrival,
                          const int32_t *prompt, const int32_t *output, const int32_t *output_key,
                          const uint8_t *bit, int32_t O0, int32_t O1, int policy, int64_t M,
                          int feas_mode, int n_threads,
                          int32_t *start, int32_t *finish, int64_t *total_latency,
                          int64_t *p99_latency, int32_t *makespan, int64_t *peak_kv, int64_t *rounds,
                          int64_t *decisions, int32_t *status)
{
    if (n_instances < 0 || policy < 0 || policy > 3 || M < 0) return ST_EINVAL;
    if (policy == POL_SVF_1BIT && ((n_instances > 0 && offsets[n_instances] > 0 && !bit) || O0 < 1 || O1 < 1)) return ST_EINVAL;
    if (n_threads < 1) n_threads = 1;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1) num_threads(n_threads)
#endif
    for (int64_t j = 0; j < n_instances; ++j) {
        int64_t lo = offsets[j], n = offsets[j + 1] - offsets[j];
        inst_result_t r;
        simulate_instance(policy, M, feas_mode, n, arrival + lo, prompt + lo, output + lo,
                          output_key ? output_key + lo : NULL,
                          bit ? bit + lo : NULL, O0, O1, start ? start + lo : NULL,
                          finish ? finish + lo : NULL, &r);
        if (total_latency) total_latency[j] = r.total_latency;
        if (p99_latency) p99_latency[j] = r.p99_latency;
        if (makespan) makespan[j] = r.makespan;
        if (peak_kv) peak_kv[j] = r.peak_kv;
        if (rounds) rounds[j] = r.rounds;
        if (decisions) decisions[j] = r.decisions;
        if (status) status[j] = r.status;
    }
    return ST_OK;
}

int svf_ref_simulate(int64_t n_instances, const int64_t *offsets, const int32_t *arrival,
                     const int32_t *prompt, const int32_t *output, const uint8_t *bit,
                     int32_t O0, int32_t O1, int policy, int64_t M, int feas_mode, int n_threads,
                     int32_t *start, int32_t *finish, int64_t *total_latency,
                     int64_t *p99_latency, int32_t *makespan, int64_t *peak_kv, int64_t *rounds,
                     int64_t *decisions, int32_t *status)
{
    return svf_ref_simulate_pred(n_instances, offsets, arrival, prompt, output, NULL, bit, O0, O1, policy, M,
                                 feas_mode, n_threads, start, finish, total_latency, p99_latency, makespan,
                                 peak_kv, rounds, decisions, status);
}

/* ------------------------------------------------------------------------------------------
 * NEXT-2: the volume lower bound of Proposition 3.1 (Eq. 5) for burst input,
 *     M * TEL(OPT) >= LB = sum_{j=1..N} sum_{i=1..j} vol_(i),   vol_(1) <= ... <= vol_(N),
 * written as printed: sort the volumes (Eq. 1), then for every j add the sum of the first j.
 * lb_out[j] = LB of instance j (int64); status_out[j] = ST_EOVERFLOW only if LB itself does not fit
 * (LB >= 2^63; lb 0), ST_ERANGE if some o < 1 or s < 0 (wins).  Eq. 5 is a statement about integers
 * and sets no width: a single volume may be anything an int64 holds (s, o < 2^31 gives < 2^62.6);
 * the sums are carried in 128 bits.  (The CUDA library refuses instances that hold a volume >= 2^32
 * -- its presort orders 32-bit keys, R19 -- that is ITS limit, not the bound's.)
 * Arrivals are not looked at: the bound is about the burst version of the instance.
 * ---------------------------------------------------------------------------------------- */
int svf_ref_volume_lower_bound(int64_t n_instances, const int64_t *offsets, const int32_t *prompt,
                               const int32_t *output, int64_t *lb_out, int32_t *status_out)
{
    if (n_instances < 0) return ST_EINVAL;
    for (int64_t j = 0; j < n_instances; ++j) {
        int64_t lo = offsets[j], n = offsets[j + 1] - offsets[j];
        int32_t st = ST_OK;
        int64_t *vol = (int64_t *)malloc(sizeof(int64_t) * (size_t)(n > 0 ? n : 1));
        for (int64_t i = 0; i < n; ++i) {
            if (output[lo + i] < 1 || prompt[lo + i] < 0) st = ST_ERANGE;
            vol[i] = ref_key(POL_SVF, prompt[lo + i], output[lo + i], 0, 0, 0, 0);   /* Eq. 1, exact in int64 */
        }
        unsigned __int128 lb = 0, prefix = 0;
        if (st == ST_OK) {
            qsort(vol, (size_t)n, sizeof(int64_t), cmp_i64);
            for (int64_t jj = 0; jj < n; ++jj) {      /* inner sum of Eq. 5 carried along */
                prefix += (unsigned __int128)vol[jj];
                lb += prefix;
            }
            if (lb >> 63) { st = ST_EOVERFLOW; lb = 0; }
        }
        free(vol);
        lb_out[j] = (int64_t)lb;
        if (status_out) status_out[j] = st;
    }
    return ST_OK;
}

int svf_ref_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------------
 * Brute-force hindsight optimum (IP 3a-3d) for tiny burst instances (all a_i = 0):
 * depth-first search over time; at each step any subset of the unstarted requests whose
 * addition keeps the literal check true may start.  Prunes: (i) cost so far + the latency
 * every unstarted request would have if it started now >= best; (ii) if nothing is running,
 * waiting is never better than starting something (a schedule with an idle step can be
 * shifted one step earlier), so at least one request starts.
 * ---------------------------------------------------------------------------------------- */
typedef struct {
    int n; int64_t M; const int32_t *s, *o;
    int64_t best; int64_t nodes;
    int32_t k[16]; int32_t best_k[16];
} bf_t;

static int bf_feasible(const bf_t *b, uint32_t started, int64_t t)
{
    member_t S[16]; int m = 0;
    for (int i = 0; i < b->n; ++i)
        if ((started >> i) & 1u) {
            int64_t f = (int64_t)b->k[i] + b->o[i];
            if (f > t) { S[m].kv = b->s[i] + (t - b->k[i]); S[m].rem = f - t; ++m; }
        }
    return feasible_literal(S, m, b->M);
}

static void bf_dfs(bf_t *b, uint32_t started, int64_t t, int64_t cost)
{
    b->nodes++;
    uint32_t all = (1u << b->n) - 1u;
    if (started == all) {
        if (cost < b->best) { b->best = cost; memcpy(b->best_k, b->k, sizeof(b->k)); }
        return;
    }
    int64_t lb = cost;
    for (int i = 0; i < b->n; ++i) if (!((started >> i) & 1u)) lb += t + b->o[i];
    if (lb >= b->best) return;
    int any_running = 0;
    for (int i = 0; i < b->n; ++i)
        if (((started >> i) & 1u) && (int64_t)b->k[i] + b->o[i] > t) any_running = 1;
    uint32_t un = all & ~started;
    /* every non-empty subset of the unstarted set (and the empty one if something runs) */
    for (uint32_t sub = un;; sub = (sub - 1) & un) {
        if (sub == 0) {
            if (any_running) bf_dfs(b, started, t + 1, cost);
            break;
        }
        int64_t c = cost;
        for (int i = 0; i < b->n; ++i) if ((sub >> i) & 1u) { b->k[i] = (int32_t)t; c += t + b->o[i]; }
        if (bf_feasible(b, started | sub, t)) bf_dfs(b, started | sub, t + 1, c);
    }
}

int svf_ref_bruteforce_opt(int64_t n, const int32_t *s, const int32_t *o, int64_t M,
                           int64_t *opt_out, int32_t *start_out, int64_t *nodes_out)
{
    if (n < 1 || n > 12) return ST_EINVAL;
    for (int64_t i = 0; i < n; ++i) {
        if (o[i] < 1 || s[i] < 0) return ST_ERANGE;
        if ((int64_t)s[i] + o[i] > M) return ST_EINFEASIBLE;
    }
    bf_t b; memset(&b, 0, sizeof(b));
    b.n = (int)n; b.M = M; b.s = s; b.o = o; b.best = INT64_MAX; b.nodes = 0;
    bf_dfs(&b, 0u, 0, 0);
    *opt_out = b.best;
    if (start_out) for (int i = 0; i < b.n; ++i) start_out[i] = b.best_k[i];
    if (nodes_out) *nodes_out = b.nodes;
    return ST_OK;
}
