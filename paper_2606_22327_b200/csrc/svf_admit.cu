// a1-a5: one stateless admission decision (P:L358-366 engine loop; P:L507-524 order, no bypass,
// forward-looking check; P:L926 maxima at completion times).
//   keys (svf_keys.cu) -> onesweep sort of the packed words on the key bits [32, 64)
//   running set: words (2^32-1-rem, index) sorted the same way -> latest finish first
//   k_admit_prefix (the usual path): feasibility is MONOTONE in the candidate set (adding a request
//   adds a positive amount at every time it is alive), so the greedy loop's answer is the maximal
//   feasible prefix of the priority order.  One CTA takes the running set and the
//   first K_c candidates (K_c = min(n_wait, 8192 - n_run)), sorts them together by remaining steps
//   (descending; stable radix passes in shared memory), keeps each thread's eight consecutive
//   entries in registers and BISECTS the prefix length m: one check = the completion-time form of
//   the forward-looking test on running + {candidates of rank < m} = a masked block scan of
//   (kv, count) + max, about a microsecond; 14 checks instead of thousands of serial admissions.
//   A queue and a running set that fit the CTA together (n_wait + n_run <= 8192) take NOTHING else: the
//   same kernel validates, computes the keys and sorts the queue in shared memory first (one launch).
//   Only if all K_c candidates fit and more are waiting (or n_run > 4096) the serial path runs:
//   k_admit: one CTA builds (f_j, A_j) in finish order with a block scan (svf_state.cuh) and checks
//   the running set; then k_admit_slots (M < 2^30) takes the set into REGISTER SLOTS and pops the
//   sorted queue with the fused evaluation pass of svf_sim_slots.cuh while the check passes;
//   for M >= 2^30 k_admit itself pops the queue on the sorted (f, A) arrays in 64-bit.
#include <limits.h>

#include "svf_internal.cuh"
#include "svf_state.cuh"
#include "svf_sim_slots.cuh"
#include "svf_segsort.cuh"

namespace svf {

namespace {

constexpr int ADMIT_THREADS = 1024;

// first offending waiting index (ERANGE before EUNSORTED at the same index), running-set range
struct AdmitFlags {
    unsigned long long first_bad;   // (index << 1) | (0 range, 1 unsorted); ~0 if none
    uint32_t run_bad;
    int32_t key_status;             // from the keys kernel
};

__global__ void k_admit_init(AdmitFlags* fl) { fl->first_bad = ~0ull; fl->run_bad = 0; fl->key_status = 0; }

__global__ void __launch_bounds__(256) k_admit_validate(int64_t n_wait, const int32_t* __restrict__ w_s,
                                                        const int32_t* __restrict__ w_o,
                                                        const int32_t* __restrict__ w_a, int64_t n_run,
                                                        const int32_t* __restrict__ r_kv,
                                                        const int32_t* __restrict__ r_rem,
                                                        uint64_t* __restrict__ rwords, AdmitFlags* fl)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long bad = ~0ull;
    for (int64_t i = gid; i < n_wait; i += stride) {
        const int32_t ai = w_a[i];
        unsigned long long b = ~0ull;
        if (w_o[i] < 1 || w_s[i] < 0 || ai < 0) b = (unsigned long long)i << 1;
        else if (i > 0 && ai < w_a[i - 1]) b = ((unsigned long long)i << 1) | 1ull;
        bad = b < bad ? b : bad;
    }
    if (bad != ~0ull) atomicMin(&fl->first_bad, bad);
    bool rb = false;
    for (int64_t i = gid; i < n_run; i += stride) {
        const int32_t rem = r_rem[i];
        if (rem < 1 || r_kv[i] < 0) rb = true;
        // ascending order of (2^32-1-rem) = latest finish first; ties keep the input order
        rwords[i] = ((uint64_t)(0xffffffffu - (uint32_t)rem) << 32) | (uint64_t)(uint32_t)i;
    }
    if (rb) atomicOr(&fl->run_bad, 1u);
}

__device__ __forceinline__ int64_t block_incl_scan_i64(int64_t v, int64_t* warp_tot, int64_t& total)
{
    const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { int64_t x = __shfl_up_sync(FULL, v, d); if (lane >= d) v += x; }
    if (lane == 31) warp_tot[wrp] = v;
    __syncthreads();
    int64_t off = 0, tot = 0;
    for (int w = 0; w < ADMIT_THREADS / 32; ++w) { int64_t x = warp_tot[w]; if (w < wrp) off += x; tot += x; }
    __syncthreads();
    total = tot;
    return v + off;
}

// ---- the maximal feasible prefix by bisection (a4 + a5), one CTA -------------------------------
constexpr int AP_THREADS = 1024;                     // the wide form: up to 8,192 entries on chip
constexpr int AP_IPT = 8;
constexpr int AP_CAP = AP_THREADS * AP_IPT;          // running + candidate entries held on chip
constexpr int AP_RUN_MAX = AP_CAP / 2;               // larger running sets take the serial path
constexpr size_t ap_smem_bytes(int threads) { return (size_t)2 * threads * AP_IPT * 8 + (size_t)threads * AP_IPT * 4 + (size_t)(threads / 32) * SORT_RADIX * 4; }
constexpr size_t AP_SMEM = ap_smem_bytes(AP_THREADS);

// fast[0] = 1: this kernel has answered (outputs written); 0: the serial kernels must run, and
// rsorted_out holds the running set in their order (latest finish first, ties in input order).
// FUSED (n_wait + n_run <= 8192, the size of a real serving queue): the WHOLE decision in this one launch --
// validation, keys (a1), packing (a2), the radix sort of the queue in shared memory (a3), then the
// bisection; nothing else is launched.  Otherwise the queue arrives sorted by the device-wide sort.
struct AdmitFused {
    int policy; int32_t O0, O1;
    const int32_t* w_a; const uint8_t* w_bit;
    uint64_t* sorted_words_out;              // or NULL
};

template <bool FUSED, int AP_THREADS>
__global__ void __launch_bounds__(AP_THREADS, 1) k_admit_prefix(int64_t M, int64_t n_wait, const int32_t* __restrict__ w_s,
                                                                const int32_t* __restrict__ w_o, int n_run,
                                                                const int32_t* __restrict__ r_kv,
                                                                const int32_t* __restrict__ r_rem,
                                                                const SortPlan* __restrict__ wplan,
                                                                const AdmitFlags* __restrict__ fl,
                                                                uint64_t* __restrict__ rsorted_out, int* __restrict__ fast,
                                                                int64_t* __restrict__ n_admitted_out,
                                                                int32_t* __restrict__ admitted_idx_out,
                                                                int32_t* __restrict__ status_out, AdmitFused fu)
{
    constexpr int WARPS = AP_THREADS / 32;
    constexpr int AP_CAP = AP_THREADS * AP_IPT;          // running + candidate entries held on chip
    extern __shared__ __align__(16) char ap_smem[];
    uint64_t* buf0 = reinterpret_cast<uint64_t*>(ap_smem);
    uint64_t* buf1 = buf0 + AP_CAP;
    int32_t* kv_e = reinterpret_cast<int32_t*>(buf1 + AP_CAP);          // kv by entry id
    uint32_t* whist = reinterpret_cast<uint32_t*>(kv_e + AP_CAP);
    __shared__ uint32_t toff_s[SORT_RADIX];
    __shared__ uint32_t warp_tot[WARPS];
    __shared__ int64_t wsum_s[WARPS];
    __shared__ int wcnt_s[WARPS];
    __shared__ int red_s[2];
    const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;

    const int R = n_run;
    int32_t status = SVF_OK;
    if (!FUSED) {
        if (fl->first_bad != ~0ull) status = (fl->first_bad & 1ull) ? SVF_EUNSORTED : SVF_ERANGE;
        else if (fl->run_bad) status = SVF_ERANGE;
        else if (fl->key_status != SVF_OK) status = fl->key_status;
    } else {
        // validation (first offending waiting index: range before order at the same index; then the
        // running set; then the key width), keys and packed words, all on this CTA
        __shared__ unsigned long long first_bad_s;
        __shared__ uint32_t vflags_s[2];                    // [0] running set out of range, [1] OR of the keys' high words
        if (tid == 0) { first_bad_s = ~0ull; vflags_s[0] = 0; vflags_s[1] = 0; }
        if (tid < 2) red_s[tid] = 0;
        __syncthreads();
        unsigned long long bad = ~0ull;
        uint32_t kor = 0, khi = 0, rb = 0;
        const int nw = (int)n_wait;
        for (int i = tid; i < nw; i += AP_THREADS) {
            const int32_t si = w_s[i], oi = w_o[i], ai = fu.w_a[i];
            unsigned long long b = ~0ull;
            if (oi < 1 || si < 0 || ai < 0) b = (unsigned long long)i << 1;
            else if (i > 0 && ai < fu.w_a[i - 1]) b = ((unsigned long long)i << 1) | 1ull;
            bad = b < bad ? b : bad;
            const uint32_t bt = fu.policy == SVF_SVF_1BIT ? (uint32_t)fu.w_bit[i] : 0u;
            const uint64_t key = (oi >= 1 && si >= 0 && ai >= 0) ? priority_key(fu.policy, si, oi, ai, bt, fu.O0, fu.O1) : 0ull;
            khi |= (uint32_t)(key >> 32);
            kor |= (uint32_t)key;
            buf0[i] = (key << 32) | (uint32_t)i;
        }
        for (int i = tid; i < R; i += AP_THREADS) if (r_rem[i] < 1 || r_kv[i] < 0) rb = 1;
        if (bad != ~0ull) atomicMin(&first_bad_s, bad);
        if (rb) atomicOr(&vflags_s[0], 1u);
        khi = __reduce_or_sync(FULL, khi); kor = __reduce_or_sync(FULL, kor);
        if (lane == 0) { if (khi) atomicOr(&vflags_s[1], khi); if (kor) atomicOr(reinterpret_cast<unsigned int*>(&red_s[1]), kor); }
        __syncthreads();
        if (first_bad_s != ~0ull) status = (first_bad_s & 1ull) ? SVF_EUNSORTED : SVF_ERANGE;
        else if (vflags_s[0]) status = SVF_ERANGE;
        else if (vflags_s[1]) status = SVF_EOVERFLOW;
    }
    if (status != SVF_OK) {
        if (tid == 0) { *n_admitted_out = 0; if (status_out) *status_out = status; if (fast) *fast = 1; }
        return;
    }
    if (FUSED) {
        // a3: the queue in priority order: stable radix passes over the significant key bytes; the order
        // is kept as the input indices at kv_e[R + rank] (overwritten in place by kv below)
        const int nw = (int)n_wait;
        const uint32_t kall = (uint32_t)red_s[1];
        const int npass = ((kall ? 32 - __clz(kall) : 0) + SORT_RADIX_BITS - 1) / SORT_RADIX_BITS;
        const int ipt = (nw + AP_THREADS - 1) / AP_THREADS;
        for (int p = 0; p < npass; ++p) {
            seg_pass<AP_THREADS, AP_IPT>(buf0, buf1, nw, ipt, 32 + p * SORT_RADIX_BITS, whist, toff_s, warp_tot);
            uint64_t* tmp = buf0; buf0 = buf1; buf1 = tmp;
        }
        __syncthreads();
        for (int i = tid; i < nw; i += AP_THREADS) {
            const uint64_t w = buf0[i];
            kv_e[R + i] = (int32_t)(uint32_t)w;
            if (fu.sorted_words_out) fu.sorted_words_out[i] = w;
            if (admitted_idx_out) admitted_idx_out[i] = (int32_t)(uint32_t)w;      // the first k of them are the answer
        }
        __syncthreads();
    }

    // entries: e < R the running set as given (kv, rem); e >= R the candidate of priority rank e - R,
    // started now: it holds s now and has o steps left
    const uint64_t* __restrict__ wsorted = FUSED ? nullptr : wplan->result;
    const int Kc = (int)(n_wait < (int64_t)(AP_CAP - R) ? n_wait : (int64_t)(AP_CAP - R));
    const int E = R + Kc;
    int rem_l[AP_IPT];
    int maxrem = 0;
    {   // two rounds of independent loads (the candidates' (s, o) are gathered through their sorted words)
        uint32_t h[AP_IPT];
        int kvv[AP_IPT];
#pragma unroll
        for (int i = 0; i < AP_IPT; ++i) {
            const int e = tid + i * AP_THREADS;
            h[i] = (e >= R && e < E) ? (FUSED ? (uint32_t)kv_e[e] : (uint32_t)wsorted[e - R]) : 0u;
        }
#pragma unroll
        for (int i = 0; i < AP_IPT; ++i) {
            const int e = tid + i * AP_THREADS;
            const bool run = e < R, cand = e >= R && e < E;
            kvv[i] = run ? r_kv[e] : (cand ? w_s[h[i]] : 0);
            rem_l[i] = run ? r_rem[e] : (cand ? w_o[h[i]] : 0);
        }
#pragma unroll
        for (int i = 0; i < AP_IPT; ++i) {
            const int e = tid + i * AP_THREADS;
            if (e < E) kv_e[e] = kvv[i];
            maxrem = rem_l[i] > maxrem ? rem_l[i] : maxrem;
        }
    }
    maxrem = __reduce_max_sync(FULL, maxrem);
    __syncthreads();                           // (FUSED: every thread has read its candidates' indices out of kv_e)
    if (tid < 2) red_s[tid] = 0;
    __syncthreads();
    if (lane == 0) atomicMax(&red_s[0], maxrem);
    __syncthreads();
    maxrem = red_s[0];
    // word = (maxrem - rem) << 32 | e: ascending = latest finish first, equal rem in entry order
    uint32_t kor = 0;
#pragma unroll
    for (int i = 0; i < AP_IPT; ++i) {
        const int e = tid + i * AP_THREADS;
        if (e < E) {
            const uint32_t key = (uint32_t)(maxrem - rem_l[i]);
            buf0[e] = ((uint64_t)key << 32) | (uint32_t)e;
            kor |= key;
        }
    }
    kor = __reduce_or_sync(FULL, kor);
    if (lane == 0 && kor) atomicOr(reinterpret_cast<unsigned int*>(&red_s[1]), kor);
    __syncthreads();
    const uint32_t kall = (uint32_t)red_s[1];
    const int npass = ((kall ? 32 - __clz(kall) : 0) + SORT_RADIX_BITS - 1) / SORT_RADIX_BITS;
    const int ipt = (E + AP_THREADS - 1) / AP_THREADS;
    for (int p = 0; p < npass; ++p) {
        seg_pass<AP_THREADS, AP_IPT>(buf0, buf1, E, ipt, 32 + p * SORT_RADIX_BITS, whist, toff_s, warp_tot);
        uint64_t* tmp = buf0; buf0 = buf1; buf1 = tmp;
    }
    __syncthreads();

    // this thread's eight consecutive entries of the completion-time order, in registers
    int kv[AP_IPT], rem[AP_IPT], rk[AP_IPT];          // rk: priority rank, -1 = running (always in the set)
#pragma unroll
    for (int i = 0; i < AP_IPT; ++i) {
        const int p = tid * AP_IPT + i;
        kv[i] = 0; rem[i] = 0; rk[i] = INT_MAX;       // past the end: never in the set
        if (p < E) {
            const uint64_t w = buf0[p];
            const int e = (int)(uint32_t)w;
            rem[i] = maxrem - (int)(uint32_t)(w >> 32);
            kv[i] = kv_e[e];
            rk[i] = e < R ? -1 : e - R;
        }
    }

    // feasible(m): with S_m = running + {candidates of rank < m} in this order, every entry of S_m
    // has  sum_{earlier or same, in S_m} kv + rem * #{earlier or same, in S_m}  <= M   (an
    // entry inside a group of equal rem sees a partial sum, which is below the group's last entry)
    auto feasible = [&](int m) -> bool {
        int64_t s = 0; int c = 0;
#pragma unroll
        for (int i = 0; i < AP_IPT; ++i) if (rk[i] < m) { s += kv[i]; ++c; }
        int64_t si = s; int ci = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int64_t x = __shfl_up_sync(FULL, si, d); const int y = __shfl_up_sync(FULL, ci, d);
            if (lane >= d) { si += x; ci += y; }
        }
        if (lane == 31) { wsum_s[wrp] = si; wcnt_s[wrp] = ci; }
        __syncthreads();
        int64_t ws = lane < WARPS ? wsum_s[lane] : 0; int wc = lane < WARPS ? wcnt_s[lane] : 0;       // one warp total per lane
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int64_t x = __shfl_up_sync(FULL, ws, d); const int y = __shfl_up_sync(FULL, wc, d);
            if (lane >= d) { ws += x; wc += y; }
        }
        int64_t pre = si - s + (wrp > 0 ? __shfl_sync(FULL, ws, wrp - 1) : 0);
        int cnt = ci - c + (wrp > 0 ? __shfl_sync(FULL, wc, wrp - 1) : 0);
        bool bad = false;
#pragma unroll
        for (int i = 0; i < AP_IPT; ++i)
            if (rk[i] < m) { pre += kv[i]; ++cnt; bad |= pre + (int64_t)rem[i] * cnt > M; }
        return __syncthreads_or(bad) == 0;               // also fences wsum_s / wcnt_s for the next call
    };
    static_assert(WARPS <= 32, "the second scan level holds one warp total per lane");
    // the same probe in 32 bits when the numbers allow it (M < 2^26 and rem * count < 2^30: every config
    // of the paper's shape): sums SATURATE at 2^26 > M (all terms are >= 0, so a saturated sum is a
    // violated one and saturating addition stays associative), one shuffle per scan step instead of
    // three, and the warp totals are combined by one hardware reduction
    constexpr uint32_t SAT = 1u << 26;
    const bool narrow = M < (int64_t)SAT && (int64_t)maxrem * E < ((int64_t)1 << 30);
    __shared__ uint32_t wsum32_s[WARPS];
    auto feasible32 = [&](int m) -> bool {
        uint32_t s = 0; int c = 0;
#pragma unroll
        for (int i = 0; i < AP_IPT; ++i) if (rk[i] < m) { s += (uint32_t)kv[i]; s = s < SAT ? s : SAT; ++c; }
        uint32_t packed_c = (uint32_t)c;
        uint32_t si = s; uint32_t ci = packed_c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t x = __shfl_up_sync(FULL, si, d), y = __shfl_up_sync(FULL, ci, d);
            if (lane >= d) { si += x; si = si < SAT ? si : SAT; ci += y; }
        }
        if (lane == 31) { wsum32_s[wrp] = si; wcnt_s[wrp] = (int)ci; }
        __syncthreads();
        // exclusive prefix over the warps before mine: 32 warp totals <= 2^26 each sum below 2^31
        const uint32_t wv = lane < wrp ? wsum32_s[lane] : 0u;
        const int wcv = lane < wrp ? wcnt_s[lane] : 0;
        uint32_t pre = __reduce_add_sync(FULL, wv); pre = pre < SAT ? pre : SAT;
        int cnt = __reduce_add_sync(FULL, wcv);
        pre += si - s; pre = pre < SAT ? pre : SAT;          // (si - s: this warp's lanes before mine, saturated alike)
        cnt += (int)ci - c;
        bool bad = false;
        const uint32_t Mu = (uint32_t)M;
#pragma unroll
        for (int i = 0; i < AP_IPT; ++i)
            if (rk[i] < m) { pre += (uint32_t)kv[i]; pre = pre < SAT ? pre : SAT; ++cnt; bad |= pre + (uint32_t)rem[i] * (uint32_t)cnt > Mu; }
        return __syncthreads_or(bad) == 0;
    };

    int lo = 0, hi = Kc + 1;                                 // feasible(lo) (or nobody fits at all), !feasible(hi)
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (narrow ? feasible32(mid) : feasible(mid)) lo = mid; else hi = mid;
    }
    if (!FUSED && lo == Kc && (int64_t)Kc < n_wait) {
        // every candidate held here fits and more are waiting: the serial kernels take over; give
        // them the running set in finish order (its entries, compacted from the order above)
        int c = 0;
#pragma unroll
        for (int i = 0; i < AP_IPT; ++i) c += rk[i] == -1;
        int ci = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const int y = __shfl_up_sync(FULL, ci, d); if (lane >= d) ci += y; }
        if (lane == 31) wcnt_s[wrp] = ci;
        __syncthreads();
        int wc = lane < WARPS ? wcnt_s[lane] : 0;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const int y = __shfl_up_sync(FULL, wc, d); if (lane >= d) wc += y; }
        int q = ci - c + (wrp > 0 ? __shfl_sync(FULL, wc, wrp - 1) : 0);
#pragma unroll
        for (int i = 0; i < AP_IPT; ++i) {
            if (rk[i] == -1) {
                const uint32_t e = (uint32_t)buf0[tid * AP_IPT + i];
                rsorted_out[q++] = ((uint64_t)(0xffffffffu - (uint32_t)rem[i]) << 32) | e;
            }
        }
        if (tid == 0) *fast = 0;
        return;
    }
    if (!FUSED && admitted_idx_out)
        for (int k = tid; k < lo; k += AP_THREADS) admitted_idx_out[k] = (int32_t)(uint32_t)wsorted[k];
    if (tid == 0) { *n_admitted_out = lo; if (status_out) *status_out = SVF_OK; if (fast) *fast = 1; }
}

__global__ void __launch_bounds__(ADMIT_THREADS) k_admit(int64_t M, int32_t t, int64_t n_wait,
                                                         const int32_t* __restrict__ w_s,
                                                         const int32_t* __restrict__ w_o,
                                                         int64_t n_run, const int32_t* __restrict__ r_kv,
                                                         const int32_t* __restrict__ r_rem,
                                                         const SortPlan* __restrict__ wplan,
                                                         const SortPlan* __restrict__ rplan,
                                                         const uint64_t* __restrict__ rsorted_direct /* or NULL: rplan */,
                                                         const int* __restrict__ fast /* or NULL */,
                                                         const AdmitFlags* __restrict__ fl,
                                                         int32_t* __restrict__ f, int64_t* __restrict__ A,
                                                         int64_t* __restrict__ n_admitted_out,
                                                         int32_t* __restrict__ admitted_idx_out,
                                                         int32_t* __restrict__ status_out,
                                                         int* __restrict__ handoff /* NULL: admit here */)
{
    __shared__ int scratch[2][64];
    __shared__ int64_t warp_tot[ADMIT_THREADS / 32];
    if (handoff && threadIdx.x == 0) *handoff = 0;
    if (fast && *fast) return;                 // k_admit_prefix has answered
    int parity = 0;
    const int tid = threadIdx.x;

    int32_t status = SVF_OK;
    if (fl->first_bad != ~0ull) status = (fl->first_bad & 1ull) ? SVF_EUNSORTED : SVF_ERANGE;
    else if (fl->run_bad) status = SVF_ERANGE;
    else if (fl->key_status != SVF_OK) status = fl->key_status;
    if (status != SVF_OK) {
        if (tid == 0) { *n_admitted_out = 0; if (status_out) *status_out = status; }
        return;
    }

    // running set, latest finish first: f_j = rem_j (time is counted from now), A_j = sum_{i<=j}
    // kv_i + rem_j (j+1) = mem at its completion
    const uint64_t* __restrict__ rsorted = rsorted_direct ? rsorted_direct : rplan->result;
    int64_t carry = 0;
    uint32_t bad = 0;
    for (int64_t c = 0; c < n_run; c += ADMIT_THREADS) {
        const int64_t jx = c + tid;
        int64_t kv = 0; int32_t rem = 0;
        if (jx < n_run) { const uint32_t i = (uint32_t)rsorted[jx]; kv = r_kv[i]; rem = r_rem[i]; }
        int64_t tot;
        const int64_t P = carry + block_incl_scan_i64(kv, warp_tot, tot);
        carry += tot;
        if (jx < n_run) {
            const int64_t Aj = P + (int64_t)rem * (jx + 1);
            f[jx] = rem; A[jx] = Aj;
            if (Aj > M) bad = 1;
        }
    }
    __syncthreads();
    bad = Group<ADMIT_THREADS>::or_u32(bad, scratch, parity);

    if (handoff && !bad) {       // the register-slot kernel takes over from the (f, A) arrays
        if (tid == 0) *handoff = 1;
        return;
    }
    int64_t k = 0;
    if (!bad) {        // an infeasible running set admits nobody (every check would fail)
        const uint64_t* __restrict__ wsorted = wplan->result;
        int R = (int)n_run;
        for (; k < n_wait; ++k) {
            const uint32_t h = (uint32_t)wsorted[k];
            const int32_t sh = w_s[h], oh = w_o[h];
            const Verdict v = evaluate_head<ADMIT_THREADS>(f, A, R, 0, sh, oh, M, scratch, parity);
            if (!v.ok) break;                          // blocked head: nobody may bypass it
            insert_head<ADMIT_THREADS>(f, A, R, v.pos, 0, sh, oh, v.Ah);
            ++R;
            if (tid == 0 && admitted_idx_out) admitted_idx_out[k] = (int32_t)h;
        }
    }
    (void)t;
    if (tid == 0) { *n_admitted_out = k; if (status_out) *status_out = SVF_OK; }
}

// a4 + a5 with the running set in REGISTER SLOTS (the passes of svf_sim_slots.cuh at t = 0): one
// CTA, 16 slots per thread, the overflow in ext arrays; taken when M < 2^30.  Picks up the running
// set (f, A) that k_admit built in finish order, then pops the sorted queue while the check holds.
template <int THREADS>
__global__ void __launch_bounds__(THREADS) k_admit_slots(int64_t M, int64_t n_wait, const int32_t* __restrict__ w_s,
                                                         const int32_t* __restrict__ w_o, int64_t n_run,
                                                         const int32_t* __restrict__ r_kv,
                                                         const SortPlan* __restrict__ wplan,
                                                         const SortPlan* __restrict__ rplan,
                                                         const uint64_t* __restrict__ rsorted_direct /* or NULL: rplan */,
                                                         const int* __restrict__ handoff,
                                                         const int32_t* __restrict__ f_arr, const int64_t* __restrict__ A_arr,
                                                         int32_t* __restrict__ ef, uint32_t* __restrict__ eB,
                                                         uint32_t* __restrict__ ec,
                                                         int64_t* __restrict__ n_admitted_out,
                                                         int32_t* __restrict__ admitted_idx_out,
                                                         int32_t* __restrict__ status_out)
{
    constexpr int K = 16, WARPS = THREADS / 32, REGCAP = THREADS * K, TSHIFT = 8;
    constexpr bool COUNT = false;
    static_assert(THREADS == 256, "TSHIFT");
    __shared__ int red[2][WARPS][3];
    int rparity = 0;
    long long cntE = 0, cntU = 0;
    (void)cntE; (void)cntU;
    if (*handoff == 0) return;               // data error or infeasible running set: k_admit has answered
    const int tid = threadIdx.x;
    const int Mi = (int)M;
    const uint32_t one = n_run >= 0 ? 1u : 0u;           // 1, but not to the compiler (SVF_ACC_GE)
    (void)one;
    const uint64_t* __restrict__ rsorted = rsorted_direct ? rsorted_direct : rplan->result;
    const uint64_t* __restrict__ wsorted = wplan->result;
    const int R = (int)n_run;
    int f[K]; uint32_t B[K], c[K];
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const int q = k * THREADS + tid;
        f[k] = 0; B[k] = 0; c[k] = 0;
        if (q < R) { f[k] = f_arr[q]; B[k] = (uint32_t)A_arr[q] + (uint32_t)f[k]; c[k] = (uint32_t)r_kv[(uint32_t)rsorted[q]]; }
    }
    for (int q = REGCAP + tid; q < R; q += THREADS) {
        const int e = q - REGCAP;
        ef[e] = f_arr[q]; eB[e] = (uint32_t)A_arr[q] + (uint32_t)f_arr[q]; ec[e] = (uint32_t)r_kv[(uint32_t)rsorted[q]];
    }
    int hw = R;
    const uint32_t t1 = 1u;                  // now = 0: a slot is live iff f > 0
    int64_t k = 0;
    uint32_t nh = 0; int32_t nsh = 0, noh = 0;
    if (n_wait > 0) { nh = (uint32_t)wsorted[0]; nsh = w_s[nh]; noh = w_o[nh]; }
    for (; k < n_wait; ++k) {
        const uint32_t h = nh;
        const int32_t sh = nsh, ohi = noh;
        if (k + 1 < n_wait) { nh = (uint32_t)wsorted[k + 1]; nsh = w_s[nh]; noh = w_o[nh]; }   // one head ahead
        if ((int64_t)sh + ohi > M) break;                    // could never run: blocked (and it blocks the rest)
        const int fh = ohi;
        const uint32_t oh = (uint32_t)ohi, fhu = (uint32_t)fh;
        const uint32_t Kc = (uint32_t)sh - (uint32_t)Mi, add = (uint32_t)sh;
        uint32_t acc = 0, acc1 = 0, dm = 0;
        int viol = INT_MIN;
        int kmax = (hw + THREADS - 1) >> TSHIFT; kmax = kmax < K ? kmax : K;
        const int g4 = (kmax + 3) >> 2;
        const bool use_ext = hw > REGCAP;
        SVF_SLOT_GROUPS(g4, SVF_EVAL)
        const uint32_t dmx = dm | (1u << (4 * g4));          // sentinel: the first slot past the groups in use (16 = none)
        int fkey = (int)(((dmx & (0u - dmx)) << TSHIFT) | (uint32_t)tid);
        int eidx = INT_MAX;
        if (use_ext) {
            for (int q = REGCAP + tid; q < hw; q += THREADS) {
                const int e = q - REGCAP;
                const int fk = ef[e];
                const uint32_t x = (uint32_t)fk - t1;
                if (fk >= fh) acc += ec[e] + fhu;
                if (x < oh) { viol = __viaddmax_s32((int)eB[e], (int)Kc, viol); eB[e] += add + (uint32_t)fk; }
                if (x >> 31) eidx = eidx < q ? eidx : q;
            }
        }
        acc += acc1;
        reduce_add_max_min<THREADS>(acc, viol, fkey, red, rparity);
        const int Ah = sh + ohi + (int)acc;
        if (viol > 0 || Ah > Mi) break;                      // blocked head: nobody may bypass it
        const uint32_t Bh = (uint32_t)Ah + fhu;
        int idx;
        if (fkey < (1 << (K + TSHIFT))) {
            const int ik = 31 - __clz(fkey >> TSHIFT);
            const bool mine = (fkey & (THREADS - 1)) == tid;
            idx = (ik << TSHIFT) + (fkey & (THREADS - 1));
            SVF_PUT16(ik, SVF_PUT)
        } else {
            if (use_ext) { uint32_t z = 0; int zmax = 0; reduce_add_max_min<THREADS>(z, zmax, eidx, red, rparity); }
            idx = eidx == INT_MAX ? hw : eidx;
            if (((idx - REGCAP) & (THREADS - 1)) == tid) { const int e = idx - REGCAP; ef[e] = fh; eB[e] = Bh; ec[e] = add; }
        }
        hw = idx + 1 > hw ? idx + 1 : hw;
        if (tid == 0 && admitted_idx_out) admitted_idx_out[k] = (int32_t)h;
    }
    if (tid == 0) { *n_admitted_out = k; if (status_out) *status_out = SVF_OK; }
}

struct AdmitWs {
    SortWs wsort, rsort;
    uint64_t *w0, *w1, *r0, *r1;
    int32_t* f; int64_t* A;
    int32_t* ef; uint32_t *eB, *ec;   // ext slots of the register-slot kernel
    int* handoff;
    int* fast;              // written by k_admit_prefix: 1 = answered, 0 = the serial kernels run
    AdmitFlags* flags;
    size_t total;
};

void admit_ws_layout(AdmitWs* w, char* base, int64_t n_wait, int64_t n_run)
{
    size_t p = 0;
    const size_t sw = align_up(sort_ws_bytes(n_wait, 32, 64), 256), sr = align_up(sort_ws_bytes(n_run, 32, 64), 256);
    if (base) { sort_ws_carve(&w->wsort, base + p, n_wait, 32, 64); }
    p += sw;
    if (base) { sort_ws_carve(&w->rsort, base + p, n_run, 32, 64); }
    p += sr;
    w->w0 = (uint64_t*)(base + p); p += align_up((size_t)n_wait * 8, 256);
    w->w1 = (uint64_t*)(base + p); p += align_up((size_t)n_wait * 8, 256);
    w->r0 = (uint64_t*)(base + p); p += align_up((size_t)n_run * 8, 256);
    w->r1 = (uint64_t*)(base + p); p += align_up((size_t)n_run * 8, 256);
    const size_t cap = (size_t)(n_wait + n_run + 1);
    w->A = (int64_t*)(base + p); p += align_up(cap * 8, 256);
    w->f = (int32_t*)(base + p); p += align_up(cap * 4, 256);
    w->ef = (int32_t*)(base + p); p += align_up(cap * 4, 256);
    w->eB = (uint32_t*)(base + p); p += align_up(cap * 4, 256);
    w->ec = (uint32_t*)(base + p); p += align_up(cap * 4, 256);
    w->handoff = (int*)(base + p); w->fast = w->handoff + 1; p += 256;
    w->flags = (AdmitFlags*)(base + p); p += 256;
    w->total = p;
}

thread_local int64_t g_launches_admit = 0;
thread_local bool g_admit_events_valid = false;
thread_local cudaEvent_t g_admit_ev[4] = {nullptr, nullptr, nullptr, nullptr};

void admit_mark(int i, cudaStream_t st)
{
    if (!profiling_mode()) return;
    if (!g_admit_ev[0])
        for (int k = 0; k < 4; ++k) cudaEventCreate(&g_admit_ev[k]);
    cudaEventRecord(g_admit_ev[i], st);
    if (i == 3) g_admit_events_valid = true;
}

}  // namespace

int64_t admit_last_launches() { return g_launches_admit; }

}  // namespace svf

using namespace svf;

extern "C" size_t svf_admit_workspace_bytes(int64_t n_wait, int64_t n_run)
{
    if (n_wait < 0 || n_run < 0) return 0;
    AdmitWs w;
    admit_ws_layout(&w, nullptr, n_wait, n_run);
    return w.total + 256;
}

extern "C" int svf_admit(int policy, int64_t M, int32_t t, int64_t n_wait, const int32_t* w_s,
                         const int32_t* w_o, const int32_t* w_a, const uint8_t* w_bit, int32_t O0,
                         int32_t O1, int64_t n_run, const int32_t* r_kv, const int32_t* r_rem,
                         int64_t* n_admitted_out, int32_t* admitted_idx_out, uint64_t* sorted_words_out,
                         int32_t* status_out, void* ws, size_t ws_bytes, void* stream)
{
    g_launches_admit = 0;
    const int64_t LIM = (int64_t)1 << 30;
    if (policy < 0 || policy > 3 || n_wait < 0 || n_run < 0 || n_wait >= LIM || n_run >= LIM || M < 0) return SVF_EINVAL;
    if (policy == SVF_SVF_1BIT && ((n_wait > 0 && !w_bit) || O0 < 1 || O1 < 1)) return SVF_EINVAL;
    if (!n_admitted_out) return SVF_EINVAL;
    if (n_wait > 0 && (!w_s || !w_o || !w_a)) return SVF_EINVAL;
    if (n_run > 0 && (!r_kv || !r_rem)) return SVF_EINVAL;
    if (!ws) return SVF_EWORKSPACE;
    char* base = (char*)align_up((size_t)(uintptr_t)ws, 256);
    AdmitWs w;
    admit_ws_layout(&w, base, n_wait, n_run);
    if ((size_t)(base - (char*)ws) + w.total > ws_bytes) return SVF_EWORKSPACE;
    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count < 1) return SVF_ECUDA;
    cudaStream_t st = (cudaStream_t)stream;

    g_admit_events_valid = false;
    admit_mark(0, st);
    if (n_wait + n_run <= AP_CAP) {
        // a queue and a running set that fit one CTA's shared memory: the whole decision in ONE launch
        AdmitFused fu{policy, O0, O1, w_a, w_bit, sorted_words_out};
        // the narrowest CTA that holds the entries: every barrier and block scan of the sorts and of the
        // 14 bisection probes costs by the warps taking part (kernel 29 -> 17 ... 23 us for a serving queue)
#define SVF_AP_LAUNCH(T)                                                                                        \
        do {                                                                                                    \
            if (cudaFuncSetAttribute(k_admit_prefix<true, T>, cudaFuncAttributeMaxDynamicSharedMemorySize,      \
                                     (int)ap_smem_bytes(T)) != cudaSuccess) return SVF_ECUDA;                   \
            admit_mark(1, st);                                                                                  \
            admit_mark(2, st);                                                                                  \
            k_admit_prefix<true, T><<<1, T, ap_smem_bytes(T), st>>>(M, n_wait, w_s, w_o, (int)n_run, r_kv, r_rem, nullptr, nullptr, \
                                                                    nullptr, nullptr, n_admitted_out, admitted_idx_out, status_out, fu); \
        } while (0)
        const int64_t entries = n_wait + n_run;
        if (entries <= 256 * AP_IPT) SVF_AP_LAUNCH(256);
        else if (entries <= 512 * AP_IPT) SVF_AP_LAUNCH(512);
        else SVF_AP_LAUNCH(AP_THREADS);
#undef SVF_AP_LAUNCH
        ++g_launches_admit;
        admit_mark(3, st);
        return cudaGetLastError() == cudaSuccess ? SVF_OK : SVF_ECUDA;
    }
    k_admit_init<<<1, 1, 0, st>>>(w.flags);
    ++g_launches_admit;
    // a1 + a2
    int rc = keys_launch(policy, n_wait, w_s, w_o, w_a, w_bit, O0, O1, w.w0, &w.flags->key_status, st, &g_launches_admit);
    if (rc) return SVF_ECUDA;
    {
        const int64_t m = n_wait > n_run ? n_wait : n_run;
        int64_t blocks = ceil_div(m > 0 ? m : 1, 256);
        const int64_t capb = (int64_t)sm_count() * 8;
        if (blocks > capb) blocks = capb;
        k_admit_validate<<<(unsigned)blocks, 256, 0, st>>>(n_wait, w_s, w_o, w_a, n_run, r_kv, r_rem, w.r0, w.flags);
        ++g_launches_admit;
    }
    admit_mark(1, st);
    // a3: the waiting queue in priority order; the running set by finish time
    rc = sort_u64(w.wsort, w.w0, w.w1, w.w0, n_wait, 32, 64, st, &g_launches_admit);
    if (rc) return SVF_ECUDA;
    // a4 + a5: the maximal feasible prefix by bisection on one CTA; it also orders the running set
    // (for the serial kernels, should they be needed), so the device-wide sort of it is skipped
    const bool prefix = n_run <= AP_RUN_MAX;
    if (prefix) admit_mark(2, st);            // (else the running set's device-wide sort still belongs to phase 1)
    if (prefix) {
        if (cudaFuncSetAttribute(k_admit_prefix<false, AP_THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)AP_SMEM) != cudaSuccess) return SVF_ECUDA;
        k_admit_prefix<false, AP_THREADS><<<1, AP_THREADS, AP_SMEM, st>>>(M, n_wait, w_s, w_o, (int)n_run, r_kv, r_rem, w.wsort.plan, w.flags, w.r1,
                                                              w.fast, n_admitted_out, admitted_idx_out, status_out, AdmitFused{});
        ++g_launches_admit;
    } else {
        rc = sort_u64(w.rsort, w.r0, w.r1, w.r0, n_run, 32, 64, st, &g_launches_admit);
        if (rc) return SVF_ECUDA;
        admit_mark(2, st);
    }
    const uint64_t* rdirect = prefix ? w.r1 : nullptr;
    const int* fast = prefix ? w.fast : nullptr;
    const bool slots = M < ((int64_t)1 << 30);        // 32-bit wrapping arithmetic of the slot passes is exact
    k_admit<<<1, ADMIT_THREADS, 0, st>>>(M, t, n_wait, w_s, w_o, n_run, r_kv, r_rem, w.wsort.plan, w.rsort.plan, rdirect, fast,
                                         w.flags, w.f, w.A, n_admitted_out, admitted_idx_out, status_out,
                                         slots ? w.handoff : nullptr);
    ++g_launches_admit;
    if (slots) {
        k_admit_slots<256><<<1, 256, 0, st>>>(M, n_wait, w_s, w_o, n_run, r_kv, w.wsort.plan, w.rsort.plan, rdirect, w.handoff,
                                              w.f, w.A, w.ef, w.eB, w.ec, n_admitted_out, admitted_idx_out, status_out);
        ++g_launches_admit;
    }
    if (sorted_words_out) {
        rc = sort_result_to(w.wsort, sorted_words_out, n_wait, st, &g_launches_admit);
        if (rc) return SVF_ECUDA;
    }
    admit_mark(3, st);
    return cudaGetLastError() == cudaSuccess ? SVF_OK : SVF_ECUDA;
}

extern "C" int svf_admit_phase_ms(float* ms_out)
{
    if (!ms_out || !g_admit_events_valid) return SVF_EINVAL;
    if (cudaEventSynchronize(g_admit_ev[3]) != cudaSuccess) return SVF_ECUDA;
    cudaEventElapsedTime(&ms_out[0], g_admit_ev[0], g_admit_ev[1]);
    cudaEventElapsedTime(&ms_out[1], g_admit_ev[1], g_admit_ev[2]);
    cudaEventElapsedTime(&ms_out[2], g_admit_ev[2], g_admit_ev[3]);
    cudaEventElapsedTime(&ms_out[3], g_admit_ev[0], g_admit_ev[3]);
    return SVF_OK;
}
