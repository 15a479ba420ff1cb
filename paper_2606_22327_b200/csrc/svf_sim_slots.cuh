// The register-resident simulator kernel (a4-a7), included by svf_simulate.cu only.
//
// RUNNING SET as unordered SLOTS.  Slot j of an instance holds, for one request in flight,
//     f_j   absolute finish step (int32); the slot is DEAD (free) once f_j <= t
//     B_j   A_j + f_j  (mod 2^32), A_j = mem(f_j) of Eq. 3c for the current running set
//     c_j   s_j - k_j  (mod 2^32)
// The memory of a fixed set peaks at completion times only, so the set is feasible iff
// every live A_j <= M.  Admitting h = (s_h, o_h) at time t, f_h = t + o_h:
//     (1)  A_h = s_h + o_h + sum_{f_i >= f_h} (c_i + t) + #{f_i >= f_h} o_h        <= M
//     (2)  for every live j with f_j <= f_h:   A_j + s_h + (f_j - t)                <= M
// and on admission every such j gets A_j += s_h + f_j - t.  Nothing depends on the ORDER of
// the slots: no sorted array, no shifting; a pass is a flat loop over slots, the first
// THREADS*K of which live in REGISTERS (slot k*THREADS + tid is register k of thread tid); the
// rest (only when more than THREADS*K requests run at once) sit in an `ext` array that is
// only ever touched by the owning thread.  One reduction (and, for a multi-warp group, one
// barrier) per evaluation.
//
// Arithmetic is 32 bit, wrapping: every TRUE value that is compared lies in [-M, 2M] and the
// host takes this kernel only when M < 2^30, so the wrapped result read as int32 is exact.
// peak_kv = max over all A values ever produced (each entry's final A_j is mem(f_j)).
//
// WAITING QUEUE: two-level bitmap over ranks (keys are time-invariant, so the presort fixes
// the order); the two lowest waiting ranks with their (s, o, id, a) are cached in registers:
// `head` and `second` (second's record is fetched one admission ahead, hiding the L2 latency).
// ARRIVALS come from a 32-wide register window over (a, s, o, rank), refilled once per 32
// arrivals; an arrival that becomes head/second takes its record from the window.
#pragma once

#include <limits.h>

#include "svf_internal.cuh"
#include "svf_state.cuh"

namespace svf {

struct Rec { int r, s, o, id, a; };      // rank (INT_MAX = none), prompt, output, local id, arrival

// smallest set bit >= q of the two-level bitmap, INT_MAX if none.  Tolerates a stale L1 bit
// whose L0 word is already empty.  Uniform over the warp (every warp computes it redundantly).
__device__ __forceinline__ int queue_first_ge(const uint32_t* L0, const uint32_t* L1, int n, int nL1, int q)
{
    if (q >= n) return INT_MAX;
    const int lane = threadIdx.x & 31;
    const int w0 = q >> 5;
    uint32_t m = L0[w0] & (~0u << (q & 31));
    if (m) return w0 * 32 + (__ffs(m) - 1);
    int w1 = w0 >> 5;
    uint32_t m1 = L1[w1] & ~((2u << (w0 & 31)) - 1u);
    while (true) {
        while (m1) {
            const int i0 = w1 * 32 + (__ffs(m1) - 1);
            const uint32_t x = L0[i0];
            if (x) return i0 * 32 + (__ffs(x) - 1);
            m1 &= m1 - 1u;
        }
        ++w1;
        bool found = false;
        for (; w1 < nL1; w1 += 32) {
            const int idx = w1 + lane;
            const uint32_t v = idx < nL1 ? L1[idx] : 0u;
            const uint32_t b = __ballot_sync(FULL, v != 0u);
            if (b) {
                const int l = __ffs(b) - 1;
                w1 += l;
                m1 = __shfl_sync(FULL, v, l);
                found = true;
                break;
            }
        }
        if (!found) return INT_MAX;
    }
}

struct SlotArgs {
    int64_t I, N, M, max_instance;
    int policy; int32_t O0, O1;
    const int64_t* off;
    const int32_t *a, *s, *o;
    const uint8_t* bit;
    const int4* req;                 // [N] (s, o, id, a) at (instance offset + rank)
    const uint32_t* rank;            // [N] rank of (instance offset + local id)
    int32_t *start, *finish;
    int64_t *tel, *peak, *rounds, *decisions;
    int32_t *makespan, *status;
    uint64_t* latw;
    unsigned long long* work_ctr;
    unsigned long long* work_counts; // [2] E, U (only written by the COUNT variant)
    char* gstate; size_t slot_bytes; // per-CTA state when it does not fit in shared memory
    int ecap;                        // ext slots per instance
    int qcap;                        // bitmap capacity (ranks)
};

__host__ __device__ inline size_t slot_state_bytes(int qcap, int ecap)
{
    const int nL0 = (qcap + 31) / 32, nL1 = (nL0 + 31) / 32;
    return align_up((size_t)nL0 * 4, 16) + align_up((size_t)nL1 * 4, 16) + 3 * align_up((size_t)ecap * 4, 16);
}


// the five results of one evaluation pass, reduced over the group (uniform afterwards)
struct EvalRed { int cnt; uint32_t csum; int viol; int minf; int fidx; };

template <int THREADS>
__device__ __forceinline__ void reduce_eval(EvalRed& r, int (*red)[THREADS / 32][5], int& parity)
{
    r.cnt = __reduce_add_sync(FULL, r.cnt);
    r.csum = __reduce_add_sync(FULL, r.csum);
    r.viol = __reduce_max_sync(FULL, r.viol);
    r.minf = __reduce_min_sync(FULL, r.minf);
    r.fidx = __reduce_min_sync(FULL, r.fidx);
    if (THREADS > 32) {
        constexpr int WARPS = THREADS / 32;
        const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
        int (*sc)[5] = red[parity];
        parity ^= 1;
        if (lane == 0) { sc[wrp][0] = r.cnt; sc[wrp][1] = (int)r.csum; sc[wrp][2] = r.viol; sc[wrp][3] = r.minf; sc[wrp][4] = r.fidx; }
        __syncthreads();
        const bool in = lane < WARPS;
        const int l = in ? lane : 0;
        r.cnt = __reduce_add_sync(FULL, in ? sc[l][0] : 0);
        r.csum = __reduce_add_sync(FULL, in ? (uint32_t)sc[l][1] : 0u);
        r.viol = __reduce_max_sync(FULL, in ? sc[l][2] : INT_MIN);
        r.minf = __reduce_min_sync(FULL, in ? sc[l][3] : INT_MAX);
        r.fidx = __reduce_min_sync(FULL, in ? sc[l][4] : INT_MAX);
    }
}

// min over the group of one value (the next completion time when no evaluation ran this step)
template <int THREADS>
__device__ __forceinline__ int reduce_min1(int v, int (*red)[THREADS / 32][5], int& parity)
{
    v = __reduce_min_sync(FULL, v);
    if (THREADS > 32) {
        constexpr int WARPS = THREADS / 32;
        const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
        int (*sc)[5] = red[parity];
        parity ^= 1;
        if (lane == 0) sc[wrp][0] = v;
        __syncthreads();
        v = __reduce_min_sync(FULL, lane < WARPS ? sc[lane][0] : INT_MAX);
    }
    return v;
}


template <int THREADS, int K, bool SMEM, bool COUNT>
__global__ void __launch_bounds__(THREADS) k_sim_slots(SlotArgs g)
{
    using G = Group<THREADS>;
    constexpr int WARPS = THREADS / 32;
    constexpr int REGCAP = THREADS * K;
    extern __shared__ __align__(16) char dyn_smem[];
    __shared__ int scratch[2][64];
    __shared__ int red[2][WARPS][5];
    __shared__ long long inst_s;
    int parity = 0, rparity = 0;
    const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;

    char* sbase = SMEM ? dyn_smem : g.gstate + (size_t)blockIdx.x * g.slot_bytes;
    const int capL0 = (g.qcap + 31) / 32, capL1 = (capL0 + 31) / 32;
    uint32_t* L0 = reinterpret_cast<uint32_t*>(sbase);
    uint32_t* L1 = reinterpret_cast<uint32_t*>(sbase + align_up((size_t)capL0 * 4, 16));
    char* ebase = reinterpret_cast<char*>(L1) + align_up((size_t)capL1 * 4, 16);
    const size_t estride = align_up((size_t)g.ecap * 4, 16);
    int32_t* ef = reinterpret_cast<int32_t*>(ebase);
    uint32_t* eB = reinterpret_cast<uint32_t*>(ebase + estride);
    uint32_t* ec = reinterpret_cast<uint32_t*>(ebase + 2 * estride);
    const uint32_t Mu = (uint32_t)g.M;

    while (true) {
        if (tid == 0) inst_s = (long long)atomicAdd(g.work_ctr, 1ull);
        __syncthreads();
        const int64_t j = inst_s;
        __syncthreads();
        if (j >= g.I) break;

        const int64_t base = g.off[j];
        const int64_t n64 = g.off[j + 1] - base;
        uint32_t flags = 0;
        if (n64 < 0 || n64 > g.max_instance || base < 0 || base + (n64 > 0 ? n64 : 0) > g.N ||
            g.off[0] != 0 || g.off[g.I] != g.N)
            flags |= F_LAYOUT;
        const int n = (flags & F_LAYOUT) ? 0 : (int)n64;
        const int32_t* __restrict__ a = g.a + base;
        const int32_t* __restrict__ s = g.s + base;
        const int32_t* __restrict__ o = g.o + base;

        // ---- validation (data errors -> status[j], never UB) --------------------------------
        int64_t sum_o = 0;
        int max_a = 0;
        for (int i = tid; i < n; i += THREADS) {
            const int32_t ai = a[i], si = s[i], oi = o[i];
            if (oi < 1 || si < 0 || ai < 0) flags |= F_RANGE;
            if (i > 0 && ai < a[i - 1]) flags |= F_UNSORTED;
            if ((int64_t)si + oi > g.M) flags |= F_INFEASIBLE;
            const uint32_t b = g.policy == SVF_SVF_1BIT ? (uint32_t)g.bit[base + i] : 0u;
            if (oi >= 1 && si >= 0 && ai >= 0 && (priority_key(g.policy, si, oi, ai, b, g.O0, g.O1) >> 32)) flags |= F_OVERFLOW;
            sum_o += oi > 0 ? oi : 0;
            max_a = ai > max_a ? ai : max_a;
        }
        flags = G::or_u32(flags, scratch, parity);
        sum_o = G::sum_i64(sum_o, scratch, parity);
        { int z = 0; G::sum_max(z, max_a, scratch, parity); }
        if ((int64_t)max_a + sum_o >= ((int64_t)1 << 31)) flags |= F_OVERFLOW;   // horizon
        const int32_t status = status_from_flags(flags);

        int64_t tel = 0, peak = 0, rounds = 0, decisions = 0;
        int32_t mk = 0;
        long long cntE = 0, cntU = 0;

        if (status != SVF_OK || n == 0) {
            for (int i = tid; i < n; i += THREADS) {
                if (g.start) g.start[base + i] = -1;
                if (g.finish) g.finish[base + i] = -1;
                if (g.latw) g.latw[base + i] = (uint64_t)j << 32;
            }
        } else {
            const uint32_t* __restrict__ rnk = g.rank + base;
            const int4* __restrict__ req = g.req + base;
            const int nL0 = (n + 31) / 32, nL1 = (nL0 + 31) / 32;
            for (int i = tid; i < nL0; i += THREADS) L0[i] = 0;
            for (int i = tid; i < nL1; i += THREADS) L1[i] = 0;

            int f[K]; uint32_t B[K], c[K];
#pragma unroll
            for (int k = 0; k < K; ++k) { f[k] = INT_MIN; B[k] = 0; c[k] = 0; }

            // arrival window: lane l holds request wb + l
            int wb = 0, aw, sw, ow, rw;
            auto load_window = [&]() {
                const int idx = wb + lane;
                const bool in = idx < n;
                aw = in ? a[idx] : INT_MAX; sw = in ? s[idx] : 0; ow = in ? o[idx] : 0;
                rw = in ? (int)rnk[idx] : INT_MAX;
            };
            load_window();
            auto win_rec = [&](int l, int r) {
                Rec x; x.r = r; x.s = __shfl_sync(FULL, sw, l); x.o = __shfl_sync(FULL, ow, l);
                x.a = __shfl_sync(FULL, aw, l); x.id = wb + l; return x;
            };
            G::sync();

            Rec head, second;
            head.r = INT_MAX; head.s = head.o = head.id = head.a = 0;
            second = head;
            int next = 0, started = 0, hw = 0, minf = INT_MAX;
            int32_t t = a[0];

            while (started < n) {
                // 2. ARRIVE (1. COMPLETE is implicit: a slot is dead once f <= t)
                bool arrived = false;
                while (next < n) {
                    if (next >= wb + 32) { wb = next; load_window(); }
                    const int idx = wb + lane;
                    const bool v = idx >= next && aw <= t;
                    const uint32_t m = __ballot_sync(FULL, v);
                    if (!m) break;
                    // nobody may still be reading the bitmap for the previous step
                    if (!arrived) G::sync();
                    arrived = true;
                    if (wrp == 0 && v) queue_set(L0, L1, rw);
                    const int r1 = __reduce_min_sync(FULL, v ? rw : INT_MAX);
                    const int l1 = __ffs(__ballot_sync(FULL, v && rw == r1)) - 1;
                    const int r2 = __reduce_min_sync(FULL, (v && lane != l1) ? rw : INT_MAX);
                    const uint32_t b2 = __ballot_sync(FULL, v && lane != l1 && rw == r2);
                    const int l2 = b2 ? __ffs(b2) - 1 : 0;
                    if (r1 < head.r) {
                        const Rec n1 = win_rec(l1, r1);
                        if (r2 < head.r) second = win_rec(l2, r2); else second = head;
                        head = n1;
                    } else if (r1 < second.r) {
                        second = win_rec(l1, r1);
                    }
                    next += __popc(m);
                    if (next < wb + 32) break;
                }
                if (arrived && THREADS == 32) __syncwarp();

                // 3. ADMIT
                int64_t wait = 1;
                if (head.r != INT_MAX) {
                    rounds += 1;
                    while (head.r != INT_MAX) {
                        const int fh = t + head.o;
                        const uint32_t Kc = (uint32_t)head.s - (uint32_t)t - Mu;
                        EvalRed e; e.cnt = 0; e.csum = 0; e.viol = INT_MIN; e.minf = INT_MAX; e.fidx = INT_MAX;
                        int kmax = (hw + THREADS - 1) / THREADS; kmax = kmax < K ? kmax : K;
                        int fr = INT_MAX;
#pragma unroll
                        for (int k = 0; k < K; ++k) {
                            if (k >= kmax) break;
                            const int fk = f[k];
                            const bool live = fk > t, ge = fk >= fh;
                            if (ge) { e.cnt += 1; e.csum += c[k]; }
                            const int v = (int)(B[k] + Kc);
                            if (live && fk <= fh) e.viol = v > e.viol ? v : e.viol;
                            if (live) e.minf = fk < e.minf ? fk : e.minf;
                            else fr = fr < k ? fr : k;
                            if (COUNT) cntE += live;
                        }
                        if (fr != INT_MAX) e.fidx = fr * THREADS + tid;
                        for (int q = REGCAP + tid; q < hw; q += THREADS) {
                            const int x = q - REGCAP;
                            const int fk = ef[x];
                            const bool live = fk > t, ge = fk >= fh;
                            if (ge) { e.cnt += 1; e.csum += ec[x]; }
                            const int v = (int)(eB[x] + Kc);
                            if (live && fk <= fh) e.viol = v > e.viol ? v : e.viol;
                            if (live) e.minf = fk < e.minf ? fk : e.minf;
                            else e.fidx = e.fidx < q ? e.fidx : q;
                            if (COUNT) cntE += live;
                        }
                        reduce_eval<THREADS>(e, red, rparity);
                        minf = e.minf;
                        const int S = (int)(e.csum + (uint32_t)e.cnt * (uint32_t)t);
                        const int64_t Ah = (int64_t)head.s + head.o + S + (int64_t)e.cnt * head.o;
                        const bool ok2 = e.viol <= 0;
                        if (!(ok2 && Ah <= g.M)) { wait = ok2 ? 1 : e.viol; break; }   // blocked: no bypass

                        // admit the head into slot idx
                        const int idx = e.fidx == INT_MAX ? hw : e.fidx;
                        hw = idx + 1 > hw ? idx + 1 : hw;
                        const uint32_t add = (uint32_t)head.s - (uint32_t)t;
                        const uint32_t Bh = (uint32_t)Ah + (uint32_t)fh;
                        kmax = (hw + THREADS - 1) / THREADS; kmax = kmax < K ? kmax : K;
                        const int myk = (idx < REGCAP && (idx % THREADS) == tid) ? idx / THREADS : -1;
#pragma unroll
                        for (int k = 0; k < K; ++k) {
                            if (k >= kmax) break;
                            const int fk = f[k];
                            if (fk > t && fk <= fh) { B[k] += add + (uint32_t)fk; if (COUNT) cntU += 1; }
                            if (k == myk) { f[k] = fh; B[k] = Bh; c[k] = add; }
                        }
                        for (int q = REGCAP + tid; q < hw; q += THREADS) {
                            const int x = q - REGCAP;
                            const int fk = ef[x];
                            if (fk > t && fk <= fh) { eB[x] += add + (uint32_t)fk; if (COUNT) cntU += 1; }
                            if (q == idx) { ef[x] = fh; eB[x] = Bh; ec[x] = add; }
                        }
                        minf = fh < minf ? fh : minf;
                        peak = Ah > peak ? Ah : peak;
                        if (e.viol != INT_MIN) { const int64_t pj = g.M + e.viol; peak = pj > peak ? pj : peak; }
                        if (tid == 0) {
                            queue_clear(L0, L1, head.r);
                            if (g.start) g.start[base + head.id] = t;
                            if (g.finish) g.finish[base + head.id] = fh;
                            if (g.latw) g.latw[base + head.id] = ((uint64_t)j << 32) | (uint32_t)(fh - head.a);
                        }
                        tel += fh - head.a;
                        mk = fh > mk ? fh : mk;
                        ++started; ++decisions;
                        // promote the second; fetch the record behind it one admission ahead
                        head = second;
                        second.r = INT_MAX;
                        if (head.r != INT_MAX) {
                            const int r = queue_first_ge(L0, L1, n, nL1, head.r + 1);
                            if (r != INT_MAX) {
                                const int4 qv = req[r];
                                second.r = r; second.s = qv.x; second.o = qv.y; second.id = qv.z; second.a = qv.w;
                            }
                        }
                    }
                    if (head.r != INT_MAX) ++decisions;          // one blocked-head evaluation
                }
                if (started == n) break;
                // 4. ADVANCE to the next step at which anything can change (exact, R16)
                int64_t t_arr = INT_MAX;
                if (next < n) {
                    if (next >= wb + 32) { wb = next; load_window(); }
                    t_arr = __shfl_sync(FULL, aw, next - wb);
                }
                if (minf <= t) {          // the earliest finisher completed and nothing was evaluated since
                    int kmax = (hw + THREADS - 1) / THREADS; kmax = kmax < K ? kmax : K;
                    int mf = INT_MAX;
#pragma unroll
                    for (int k = 0; k < K; ++k) {
                        if (k >= kmax) break;
                        if (f[k] > t) mf = f[k] < mf ? f[k] : mf;
                    }
                    for (int q = REGCAP + tid; q < hw; q += THREADS) { const int fk = ef[q - REGCAP]; if (fk > t) mf = fk < mf ? fk : mf; }
                    minf = reduce_min1<THREADS>(mf, red, rparity);
                }
                int64_t tn = t_arr < (int64_t)minf ? t_arr : (int64_t)minf;
                if (head.r != INT_MAX) {                      // blocked head waits
                    const int64_t t_lb = (int64_t)t + wait;
                    tn = t_lb < tn ? t_lb : tn;
                    rounds += tn - t - 1;
                    decisions += tn - t - 1;
                }
                t = (int32_t)tn;
            }
        }
        if (COUNT) {
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) { cntE += __shfl_xor_sync(FULL, cntE, d); cntU += __shfl_xor_sync(FULL, cntU, d); }
            if (lane == 0 && g.work_counts) {
                atomicAdd(&g.work_counts[0], (unsigned long long)cntE);
                atomicAdd(&g.work_counts[1], (unsigned long long)cntU);
            }
        }
        if (tid == 0) {
            if (g.tel) g.tel[j] = tel;
            if (g.peak) g.peak[j] = peak;
            if (g.rounds) g.rounds[j] = rounds;
            if (g.decisions) g.decisions[j] = decisions;
            if (g.makespan) g.makespan[j] = mk;
            if (g.status) g.status[j] = status;
        }
        G::sync();
    }
}

}  // namespace svf
