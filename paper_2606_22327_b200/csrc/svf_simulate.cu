// a1-a7: the batched discrete-time simulator of the paper's KV-cache model under the
// SVF / 1-bit SVF / SJF / FCFS admission rule (Alg. 1 Process 2).
//
// Phase A (presort, HBM-bound): the priority order of every instance under every policy of the
//     call.  Instances of at most 4096 requests: k_seg_sort, one CTA per instance, keys (Eq. 1 /
//     Eq. 2) + stable radix passes + rank entirely in shared memory (svf_sort.cu).  Larger ones:
//     k_sim_pack  keys packed as [ instance | key (32) | local id (sb) ]  ->  device-wide onesweep
//     on [sb, sb+32+ib) (stable; input in (instance, arrival, id) order, so the result is the
//     (instance, key, arrival, id) order)  ->  k_sim_rank  order[] / rank[] / records.
// Phase B (persistent, on-chip):  k_sim_slots (svf_sim_slots.cuh)  one thread group (warp or CTA)
//     per (policy, instance) work item, handed out by an atomic counter; running set in registers,
//     waiting bitmap and records in registers / shared memory; validates the data, simulates,
//     selects p99.  For M >= 2^30 (32-bit slot arithmetic not exact): k_sim below, sorted (f, A)
//     arrays in shared memory in 64 bit, one policy per launch, p99 by one more onesweep sort
//     (phase C).
//
// Time advance is event driven but exact (R1, R16): steps on which nothing can happen are
// jumped over and still counted into rounds/decisions exactly as the step-by-step definition
// counts them (closed forms in the header of svf_sim_slots.cuh).
#include <limits.h>

#include "svf_internal.cuh"
#include "svf_state.cuh"
#include "svf_sim_slots.cuh"

namespace svf {

namespace {

struct SimArgs {
    int64_t I, N, M, max_instance;
    int policy; int32_t O0, O1;
    int sb;                          // bits of the local-id field
    const int64_t* off;
    const int32_t *a, *s, *o;
    const int32_t* okey;             // [N] predicted lengths for the SVF / SJF key, or NULL
    const uint8_t* bit;
    const uint32_t* order;           // [N] local id at (instance offset + rank)
    const uint32_t* rank;            // [N] rank of (instance offset + local id)
    int4* req;                       // [N] (s, o, id, a) at (instance offset + rank)
    int32_t *start, *finish;
    int64_t *tel, *peak, *rounds, *decisions;
    int32_t *makespan, *status;
    uint64_t* latw;                  // [N] (instance << 32) + latency, or NULL
    unsigned long long* work_ctr;
    const uint32_t* layout_bad;      // one word: the offsets of the call are not monotone (k_sim_check_layout)
    char* gstate;                    // per-CTA state slots when the state is not in shared memory
    size_t slot_bytes;
    int cap;                         // entries per state slot
};

__host__ __device__ inline size_t state_bytes(int cap)
{
    int nL0 = (cap + 31) / 32, nL1 = (nL0 + 31) / 32;
    return align_up((size_t)cap * 8, 16) + align_up((size_t)cap * 4, 16) + align_up((size_t)nL0 * 4, 16) +
           align_up((size_t)nL1 * 4, 16);
}

// The offsets of a call must be non-decreasing from 0 to N: otherwise two instances that each look
// valid could overlap and their presorts would race on order[] / rank[].  One flag word for the
// whole call; when it is set every instance reports SVF_EINVAL and nothing is simulated.
__global__ void __launch_bounds__(256) k_sim_check_layout(int64_t I, int64_t N, const int64_t* __restrict__ off,
                                                          uint32_t* __restrict__ layout_bad)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    bool bad = false;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < I; j += stride) {
        const int64_t lo = off[j], hi = off[j + 1];
        if (lo > hi || lo < 0 || hi > N || (j == 0 && lo != 0) || (j == I - 1 && hi != N)) bad = true;
    }
    if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(layout_bad, 1u);
}

// ---- Phase A ---------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_sim_pack(SimArgs g, uint64_t* __restrict__ words)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const uint64_t seq_mask = g.sb >= 64 ? ~0ull : ((1ull << g.sb) - 1ull);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < g.N; i += stride) {
        // instance of request i: last j with off[j] <= i
        int64_t lo = 0, hi = g.I - 1;
        while (lo < hi) {
            int64_t mid = (lo + hi + 1) >> 1;
            if (__ldg(g.off + mid) <= i) lo = mid; else hi = mid - 1;
        }
        const int64_t seq = i - __ldg(g.off + lo);
        const uint32_t b = g.policy == SVF_SVF_1BIT ? (uint32_t)__ldg(g.bit + i) : 0u;
        const uint64_t key = priority_key(g.policy, __ldg(g.s + i), __ldg((g.okey ? g.okey : g.o) + i), __ldg(g.a + i), b, g.O0, g.O1);
        words[i] = ((uint64_t)lo << (32 + g.sb)) | ((key & 0xffffffffull) << g.sb) | ((uint64_t)seq & seq_mask);
    }
}

__global__ void __launch_bounds__(256) k_sim_rank(SimArgs g, const SortPlan* __restrict__ plan,
                                                  uint32_t* __restrict__ order, uint32_t* __restrict__ rank)
{
    const uint64_t* __restrict__ sorted = plan->result;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const uint64_t seq_mask = g.sb >= 64 ? ~0ull : ((1ull << g.sb) - 1ull);
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < g.N; p += stride) {
        const uint64_t w = sorted[p];
        const int64_t j = (int64_t)(w >> (32 + g.sb));
        const int64_t seq = (int64_t)(w & seq_mask);
        if (j >= g.I) continue;                       // only reachable with a corrupt layout
        const int64_t base = __ldg(g.off + j);
        const int64_t r = p - base;
        order[p] = (uint32_t)seq;
        if (r >= 0 && base + seq < g.N) {
            rank[base + seq] = (uint32_t)r;
            const int64_t i = base + seq;
            if (g.req) g.req[p] = make_int4(__ldg(g.s + i), __ldg(g.o + i), (int)seq, __ldg(g.a + i));
        }
    }
}

// ---- Phase B ---------------------------------------------------------------------------------
template <int THREADS, bool SMEM>
__global__ void __launch_bounds__(THREADS) k_sim(SimArgs g)
{
    using G = Group<THREADS>;
    extern __shared__ __align__(16) char dyn_smem[];
    __shared__ int scratch[2][64];
    __shared__ long long inst_s;
    int parity = 0;
    const int tid = threadIdx.x, lane = tid & 31;

    char* sbase = SMEM ? dyn_smem : g.gstate + (size_t)blockIdx.x * g.slot_bytes;
    const int cap = g.cap;
    const int capL0 = (cap + 31) / 32, capL1 = (capL0 + 31) / 32;
    int64_t* A = reinterpret_cast<int64_t*>(sbase);
    int32_t* f = reinterpret_cast<int32_t*>(sbase + align_up((size_t)cap * 8, 16));
    uint32_t* L0 = reinterpret_cast<uint32_t*>(reinterpret_cast<char*>(f) + align_up((size_t)cap * 4, 16));
    uint32_t* L1 = reinterpret_cast<uint32_t*>(reinterpret_cast<char*>(L0) + align_up((size_t)capL0 * 4, 16));

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
            g.off[0] != 0 || g.off[g.I] != g.N || *g.layout_bad)
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
            const int32_t ki = g.okey ? g.okey[base + i] : oi;      // length the key sees
            if (oi < 1 || si < 0 || ai < 0 || ki < 1) flags |= F_RANGE;
            if (i > 0 && ai < a[i - 1]) flags |= F_UNSORTED;
            if ((int64_t)si + oi > g.M) flags |= F_INFEASIBLE;
            const uint32_t b = g.policy == SVF_SVF_1BIT ? (uint32_t)g.bit[base + i] : 0u;
            if (oi >= 1 && si >= 0 && ai >= 0 && ki >= 1 && (priority_key(g.policy, si, ki, ai, b, g.O0, g.O1) >> 32)) flags |= F_OVERFLOW;
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

        if (status != SVF_OK || n == 0) {
            const int nn = (flags & F_LAYOUT) ? 0 : (int)n64;
            for (int i = tid; i < nn; i += THREADS) {
                if (g.start) g.start[base + i] = -1;
                if (g.finish) g.finish[base + i] = -1;
                if (g.latw) g.latw[base + i] = (uint64_t)j << 32;
            }
        } else {
            const uint32_t* __restrict__ order = g.order + base;
            const uint32_t* __restrict__ rnk = g.rank + base;
            const int nL0 = (n + 31) / 32, nL1 = (nL0 + 31) / 32;
            for (int i = tid; i < nL0; i += THREADS) L0[i] = 0;
            for (int i = tid; i < nL1; i += THREADS) L1[i] = 0;
            G::sync();

            int R = 0, next = 0, started = 0;
            int32_t t = a[0];
            int hr = INT_MAX;                        // rank of the head of the queue
            int32_t hid = 0, sh = 0, oh = 0;         // its id, s, o
            bool head_loaded = false;

            while (started < n) {
                // 1. COMPLETE: entries with f == t are the tail of the array
                while (R > 0) {
                    const int jx = R - 1 - lane;
                    const int32_t fj = jx >= 0 ? f[jx] : -1;
                    const uint32_t m = __ballot_sync(FULL, fj == t);
                    const int c = (m == FULL) ? 32 : (__ffs(~m) - 1);
                    if (c > 0) { const int64_t Al = A[R - 1]; peak = Al > peak ? Al : peak; }
                    R -= c;
                    if (c < 32) break;
                }
                // 2. ARRIVE: a_i <= t join the queue (every warp tracks the count, warp 0 writes)
                bool any_arrival = false;
                while (next < n) {
                    const int idx = next + lane;
                    const bool v = idx < n && a[idx] <= t;
                    const uint32_t m = __ballot_sync(FULL, v);
                    const int c = __popc(m);
                    int r = INT_MAX;
                    if (v) { r = (int)rnk[idx]; if (tid < 32) queue_set(L0, L1, r); }
                    r = __reduce_min_sync(FULL, r);
                    if (r < hr) { hr = r; head_loaded = false; }
                    next += c;
                    any_arrival |= c > 0;
                    if (c < 32) break;
                }
                if (any_arrival) G::sync();
                // 3. ADMIT
                int64_t wait = 1;
                if (next > started) {
                    rounds += 1;
                    while (next > started) {
                        if (!head_loaded) {
                            hid = (int32_t)order[hr]; sh = s[hid]; oh = o[hid];
                            head_loaded = true;
                        }
                        const Verdict v = evaluate_head<THREADS>(f, A, R, t, sh, oh, g.M, scratch, parity);
                        if (!v.ok) { wait = v.wait; break; }
                        insert_head<THREADS>(f, A, R, v.pos, t, sh, oh, v.Ah);
                        ++R;
                        const int32_t fh = t + oh;
                        if (tid == 0) {
                            queue_clear(L0, L1, hr);
                            if (g.start) g.start[base + hid] = t;
                            if (g.finish) g.finish[base + hid] = fh;
                            if (g.latw) g.latw[base + hid] = ((uint64_t)j << 32) | (uint32_t)(fh - a[hid]);
                        }
                        tel += fh - a[hid];
                        mk = fh > mk ? fh : mk;
                        ++started; ++decisions;
                        G::sync();
                        head_loaded = false;
                        hr = (next > started) ? queue_min(L0, L1, nL1, hr >> 10) : INT_MAX;
                    }
                    if (next > started) ++decisions;          // one blocked-head evaluation
                }
                if (started == n) break;
                // 4. ADVANCE to the next step at which anything can change
                const int64_t t_arr = next < n ? (int64_t)a[next] : (int64_t)INT_MAX;
                const int64_t t_cmp = R > 0 ? (int64_t)f[R - 1] : (int64_t)INT_MAX;
                int64_t tn = t_arr < t_cmp ? t_arr : t_cmp;
                if (next > started) {                         // blocked head waits
                    const int64_t t_lb = (int64_t)t + wait;
                    tn = t_lb < tn ? t_lb : tn;
                    rounds += tn - t - 1;
                    decisions += tn - t - 1;
                }
                t = (int32_t)tn;
            }
            // drain: the remaining completions only matter for the peak
            int64_t pk = 0;
            for (int jx = tid; jx < R; jx += THREADS) { const int64_t Al = A[jx]; pk = Al > pk ? Al : pk; }
            pk = G::max_i64_nonneg(pk, scratch, parity);
            peak = pk > peak ? pk : peak;
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

// ---- Phase C ---------------------------------------------------------------------------------
__global__ void k_sim_p99(int64_t I, const int64_t* __restrict__ off, const SortPlan* __restrict__ plan,
                          const int32_t* __restrict__ status, int64_t* __restrict__ p99)
{
    const uint64_t* __restrict__ sorted = plan->result;
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= I) return;
    const int64_t base = off[j], n = off[j + 1] - base;
    int64_t v = 0;
    if (n > 0 && status[j] == SVF_OK) {
        const int64_t rank = (99 * n + 99) / 100;       // nearest rank ceil(0.99 n), 1-based (R13)
        v = (int64_t)(uint32_t)sorted[base + rank - 1];
    }
    p99[j] = v;
}

// ---- NEXT-2: the volume lower bound of Proposition 3.1 (Eq. 5) -------------------------
// LB_j = sum_{r=0..n-1} (n - r) vol_(r), volumes ascending = the SVF priority order of the
// presort; one CTA per instance, 128-bit accumulation, overflow (>= 2^63) reported, never wrapped.
__global__ void __launch_bounds__(256) k_volume_lb(int64_t I, int64_t N, int64_t max_instance,
                                                   const int64_t* __restrict__ off, const int32_t* __restrict__ s,
                                                   const int32_t* __restrict__ o, const uint32_t* __restrict__ order,
                                                   const uint32_t* __restrict__ layout_bad,
                                                   int64_t* __restrict__ lb_out, int32_t* __restrict__ status_out)
{
    __shared__ unsigned long long part[8][2];
    __shared__ uint32_t flags_s;
    const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
    for (int64_t j = blockIdx.x; j < I; j += gridDim.x) {
        const int64_t base = off[j], n = off[j + 1] - base;
        uint32_t flags = 0;
        if (n < 0 || n > max_instance || base < 0 || base + (n > 0 ? n : 0) > N || off[0] != 0 || off[I] != N || *layout_bad) flags |= F_LAYOUT;
        if (tid == 0) flags_s = 0;
        __syncthreads();
        unsigned __int128 acc = 0;
        if (!flags) {
            for (int64_t r = tid; r < n; r += 256) {
                const int64_t i = base + order[base + r];
                const int32_t si = s[i], oi = o[i];
                if (oi < 1 || si < 0) flags |= F_RANGE;
                const uint64_t vol = priority_key(SVF_SVF, si, oi, 0, 0u, 0, 0);
                if (oi >= 1 && si >= 0 && (vol >> 32)) flags |= F_OVERFLOW;   // the presort orders 32-bit keys (R11)
                acc += (unsigned __int128)vol * (unsigned long long)(n - r);
            }
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            const unsigned long long lo = __shfl_xor_sync(FULL, (unsigned long long)acc, d);
            const unsigned long long hi = __shfl_xor_sync(FULL, (unsigned long long)(acc >> 64), d);
            acc += ((unsigned __int128)hi << 64) | lo;
        }
        flags = __reduce_or_sync(FULL, flags);
        if (lane == 0) { part[wrp][0] = (unsigned long long)acc; part[wrp][1] = (unsigned long long)(acc >> 64); if (flags) atomicOr(&flags_s, flags); }
        __syncthreads();
        if (tid == 0) {
            unsigned __int128 tot = 0;
            for (int w = 0; w < 8; ++w) tot += ((unsigned __int128)part[w][1] << 64) | part[w][0];
            uint32_t f = flags_s;
            if (!f && (tot >> 63)) f |= F_OVERFLOW;
            lb_out[j] = f ? 0 : (int64_t)tot;
            if (status_out) status_out[j] = status_from_flags(f);
        }
        __syncthreads();
    }
}

struct SimWs {
    SortWs sort;            // sized for the larger of the two sorts
    uint64_t* words0;       // [N] sort ping-pong (device-wide presort, p99 sort of the wide kernel)
    uint64_t* words1;       // [N]
    uint32_t* order[MAX_POLICIES];    // [N] each
    uint32_t* rank[MAX_POLICIES];     // [N] each
    int4* req[MAX_POLICIES];          // [N] each
    uint32_t* lat[MAX_POLICIES];      // [N] each: latencies for the in-kernel p99 selection
    int32_t* status_tmp[MAX_POLICIES];// [I] each, when the caller does not want status
    unsigned long long* counts;   // [4] E, U, evaluations, blocked evaluations of the counting variant
    unsigned long long* work_ctr;
    uint32_t* layout_bad;         // one word, 8 bytes behind work_ctr (zeroed with it)
    char* gstate;
    size_t slot_bytes;
    int grid_slots;
    size_t total;
};

struct SimConfig {
    bool slots;             // register-resident kernel (M < 2^30); else the wide sorted-array kernel
    int ecap, qcap;         // slots kernel: ext slots per instance, bitmap capacity
    bool qreg;              // slots kernel: waiting bitmap in registers, qw words per lane (<= 1024 qw ranks)
    int qw;
    bool ext_global;        // slots kernel, one warp per item: bitmaps in shared memory, ext slots in a global slot
    int k;                  // slots kernel: register slots per thread (16; 32: one warp with 1,024 slots)
    size_t state_bytes;     // per-CTA state (shared memory, or a global slot when smem is false)
    size_t gslot_bytes;     // bytes of the per-CTA slot in global memory (0: none)
    int max_cta_per_sm;     // bound on resident CTAs per SM (sizes the global slots)
    int threads;
    bool smem;
    int cap;
    size_t dyn_smem;
    int sb, ib;
    int sort_lo, sort_hi;
};

constexpr size_t SMEM_STATE_LIMIT = 200 * 1024;
constexpr size_t SMEM_WARP_STATE_LIMIT = 12 * 1024;   // one-warp groups: keep >= 16 CTAs per SM
constexpr int SLOT_K = 16;                            // register slots per thread
// The budget M reaches sim_config through ONE estimate, r_est = min(max_instance, M / 512) running
// requests, and through M >= 2^30 (the wide kernel).  r_est is only ever compared with these four
// breakpoints, so one probe per class of r_est (at most a break, just above each) plus one wide M
// visits every kernel form a trace can get: sim_workspace_bytes sizes for the largest of them.
constexpr int64_t R_EST_TOKENS = 512;
constexpr int64_t R_EST_WARP = 32 * SLOT_K, R_EST_WARP_SPARE = 48 * SLOT_K, R_EST_WARP32 = 100 * SLOT_K,
                  R_EST_CTA256 = 128 * SLOT_K;
constexpr int64_t R_EST_BREAKS[4] = {R_EST_WARP, R_EST_WARP_SPARE, R_EST_WARP32, R_EST_CTA256};

SimConfig sim_config(const svf_trace_t* tr, int64_t M, int P = 1)
{
    SimConfig c;
    const int64_t I = tr->n_instances, mx = tr->max_instance > 0 ? tr->max_instance : 1;
    c.sb = bits_for_count(mx);
    c.ib = bits_for_count(I);
    c.sort_lo = c.sb;
    c.sort_hi = c.sb + 32 + c.ib;
    c.cap = (int)((mx + 31) / 32 * 32);
    c.slots = M < ((int64_t)1 << 30);
    c.ecap = 0; c.qcap = c.cap; c.qreg = false; c.qw = 1; c.ext_global = false; c.k = SLOT_K;
    // group width.  Register-slot kernels: one WARP per item (512 register slots) unless the running
    // set can outgrow them and there are warps to spare: R is at most mx and, at a few hundred
    // tokens per running request, about M / 512.  Measured: a CTA-wide group is slower than a warp
    // whenever the set fits the warp's registers (one more barrier and a replicated scalar part per
    // evaluation); 128 threads beat 256 until R passes 2048 (configs[3] 190 vs 201 ms, configs[4]
    // 5.6 vs 10.9 ms).  The wide 64-bit kernel keeps the occupancy rule (about 16 warps per SM).
    const int64_t target_warps = (int64_t)sm_count() * 16;
    int64_t w = I > 0 ? target_warps / (I * (P > 0 ? P : 1)) : 1;   // P policies share one launch
    int threads = 32;
    if (c.slots) {
        const int64_t r_est = mx < M / R_EST_TOKENS ? mx : M / R_EST_TOKENS;
        // (an estimate just above the warp's 512 slots -- configs[2]: 585, peaks of 530 -- is served better by
        // the warp and a few ext slots unless warps are plentiful; far above it the CTA wins even at w = 2)
        // and the register-queue warp kernel (instances up to 2,048 requests) beats the CTA at any w
        const bool regq = mx <= QREG_RANKS * QREG_MAX_WORDS;
        if ((r_est > R_EST_WARP && w >= 4 && !regq) || (r_est > R_EST_WARP_SPARE && w >= 2)) threads = 128;
        if (r_est > R_EST_CTA256 && w >= 8) threads = 256;
        // ... unless ONE warp with 32 slots per thread holds the set (estimates up to 1,600: the estimate
        // counts 512 tokens per running request, real sets are smaller): no barrier, no scalar part
        // replicated in four warps (configs[4] at M = 800k: 10.4 ms with CTAs)
        if (threads == 128 && r_est <= R_EST_WARP32) { threads = 32; c.k = 32; }
    } else {
        while (threads < 1024 && (threads * 2) / 32 <= w && threads * 4 <= mx) threads *= 2;
        if (threads == 64) threads = 128;
        if (threads == 512) threads = 1024;
    }
    c.gslot_bytes = 0; c.max_cta_per_sm = 2;
    if (c.slots) {
        auto ext_of = [&](int th) { int64_t e = mx - (int64_t)th * c.k; e = e > 0 ? (e + 3) / 4 * 4 : 0; return (int)e; };
        // the register queue: instances up to 2,048 requests with 8-byte records (16 slots per thread);
        // up to 8,192 requests with packed records (16 or 32 slots per thread)
        c.qreg = threads == 32 && (c.k == SLOT_K ? mx <= QREG_RANKS * QREG_MAX_WORDS : (mx > 2 * QREG_RANKS && mx <= QREG_RANKS * QREG_MAX_WORDS));
        if (c.qreg) {
            // records + bitmap mirror in shared memory, ext slots in a global slot per CTA
            c.qw = mx <= QREG_RANKS ? 1 : (mx <= 2 * QREG_RANKS ? 2 : QREG_MAX_WORDS);
            c.qcap = 0;
            c.ecap = ext_of(32);
            c.state_bytes = qreg_smem_bytes(c.qw, c.qw > 2);
            c.smem = true;
            c.gslot_bytes = align_up(qreg_ext_bytes(c.ecap), 256);
            c.max_cta_per_sm = c.qw > 2 ? 8 : 32;
        } else if (threads == 32 && slot_state_bytes(c.qcap, ext_of(32)) > SMEM_WARP_STATE_LIMIT &&
                   slot_state_bytes(c.qcap, 0) <= SMEM_WARP_STATE_LIMIT) {
            // one warp per item, more than 1024 requests per instance: the bitmaps stay in shared
            // memory, the ext slots (only touched when more than 512 requests run at once, which the
            // choice of the group width above makes unlikely) go to a global slot per CTA
            c.ecap = ext_of(32);
            c.state_bytes = slot_state_bytes(c.qcap, 0);
            c.smem = true; c.ext_global = true;
            c.gslot_bytes = align_up(qreg_ext_bytes(c.ecap), 256);
            c.max_cta_per_sm = 32;
        } else {
            if (threads == 32 && slot_state_bytes(c.qcap, ext_of(32)) > SMEM_WARP_STATE_LIMIT) { threads = 128; c.k = SLOT_K; }
            c.ecap = ext_of(threads);
            c.state_bytes = slot_state_bytes(c.qcap, c.ecap);
            c.smem = c.state_bytes <= (threads == 32 ? SMEM_WARP_STATE_LIMIT : SMEM_STATE_LIMIT);
            if (!c.smem && threads > 32 && slot_state_bytes(c.qcap, 0) <= SMEM_STATE_LIMIT) {
                // a CTA-wide group whose ext slots outgrow shared memory (configs[3]: 2.4 MB of them, hardly
                // ever touched): the two-level bitmap (searched after every admission) stays in shared
                // memory, only the ext slots go to the global slot
                c.state_bytes = slot_state_bytes(c.qcap, 0);
                c.smem = true; c.ext_global = true;
                c.gslot_bytes = align_up(qreg_ext_bytes(c.ecap), 256);
            } else if (!c.smem) {
                c.gslot_bytes = align_up(c.state_bytes, 256);
            }
        }
    } else {
        c.state_bytes = state_bytes(c.cap);
        c.smem = c.state_bytes <= SMEM_STATE_LIMIT;
        if (!c.smem) c.gslot_bytes = align_up(c.state_bytes, 256);
    }
    c.dyn_smem = c.smem ? c.state_bytes : 0;
    c.threads = threads;
    return c;
}

template <int THREADS, bool SMEM>
int sim_grid(const SimConfig& c, int64_t I)
{
    int per_sm = 0;
    if (SMEM) cudaFuncSetAttribute(k_sim<THREADS, SMEM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.dyn_smem);
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_sim<THREADS, SMEM>, THREADS, c.dyn_smem) != cudaSuccess || per_sm < 1)
        per_sm = 1;
    int64_t grid = (int64_t)per_sm * sm_count();
    if (grid > I) grid = I;
    if (grid < 1) grid = 1;
    return (int)grid;
}

template <int THREADS, bool SMEM, bool QREG, int QW = 1, int KS = SLOT_K>
int slots_grid(const SimConfig& c, int64_t I)
{
    constexpr bool REC4 = QW > 2;
    int per_sm = 0;
    if (SMEM) {
        cudaFuncSetAttribute(k_sim_slots<THREADS, KS, SMEM, false, QREG, QW, REC4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.dyn_smem);
        cudaFuncSetAttribute(k_sim_slots<THREADS, KS, SMEM, true, QREG, QW, REC4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c.dyn_smem);
    }
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_sim_slots<THREADS, KS, SMEM, false, QREG, QW, REC4>, THREADS, c.dyn_smem) != cudaSuccess || per_sm < 1)
        per_sm = 1;
    int64_t grid = (int64_t)per_sm * sm_count();
    if (grid > I) grid = I;
    if (grid < 1) grid = 1;
    return (int)grid;
}

int sim_grid_any(const SimConfig& c, int64_t I)
{
    if (c.slots) {
        if (c.qreg && c.qw > 2) return c.k == 32 ? slots_grid<32, true, true, QREG_MAX_WORDS, 32>(c, I) : slots_grid<32, true, true, QREG_MAX_WORDS>(c, I);
        if (c.qreg) return c.qw == 2 ? slots_grid<32, true, true, 2>(c, I) : slots_grid<32, true, true, 1>(c, I);
        if (c.k == 32) return slots_grid<32, true, false, 1, 32>(c, I);
        if (c.smem) {
            switch (c.threads) {
            case 32: return slots_grid<32, true, false>(c, I);
            case 128: return slots_grid<128, true, false>(c, I);
            default: return slots_grid<256, true, false>(c, I);
            }
        }
        switch (c.threads) {
        case 32: return slots_grid<32, false, false>(c, I);
        case 128: return slots_grid<128, false, false>(c, I);
        default: return slots_grid<256, false, false>(c, I);
        }
    }
    if (c.smem) {
        switch (c.threads) {
        case 32: return sim_grid<32, true>(c, I);
        case 128: return sim_grid<128, true>(c, I);
        case 256: return sim_grid<256, true>(c, I);
        default: return sim_grid<1024, true>(c, I);
        }
    }
    switch (c.threads) {
    case 32: return sim_grid<32, false>(c, I);
    case 128: return sim_grid<128, false>(c, I);
    case 256: return sim_grid<256, false>(c, I);
    default: return sim_grid<1024, false>(c, I);
    }
}

// workspace layout for P policies; base may be nullptr (sizes only)
void sim_ws_layout(SimWs* w, char* base, const svf_trace_t* tr, const SimConfig& c, int grid_slots, int P)
{
    const int64_t N = tr->n_requests, I = tr->n_instances;
    size_t p = 0;
    const size_t s1 = sort_ws_bytes(N, c.sort_lo, c.sort_hi), s2 = sort_ws_bytes(N, 0, 32 + c.ib);
    const size_t sort_bytes = s1 > s2 ? s1 : s2;
    if (base) {
        if (s1 >= s2) sort_ws_carve(&w->sort, base, N, c.sort_lo, c.sort_hi);
        else          sort_ws_carve(&w->sort, base, N, 0, 32 + c.ib);
    }
    p += align_up(sort_bytes, 256);
    w->words0 = (uint64_t*)(base + p); p += align_up((size_t)N * 8, 256);
    w->words1 = (uint64_t*)(base + p); p += align_up((size_t)N * 8, 256);
    for (int q = 0; q < P; ++q) {
        w->order[q] = (uint32_t*)(base + p);  p += align_up((size_t)N * 4, 256);
        w->rank[q] = (uint32_t*)(base + p);   p += align_up((size_t)N * 4, 256);
        w->req[q] = (int4*)(base + p);        p += align_up((size_t)N * 16, 256);
        w->lat[q] = (uint32_t*)(base + p);    p += align_up((size_t)N * 4, 256);
        w->status_tmp[q] = (int32_t*)(base + p); p += align_up((size_t)(I > 0 ? I : 1) * 4, 256);
    }
    w->counts = (unsigned long long*)(base + p); p += 256;
    w->work_ctr = (unsigned long long*)(base + p);
    w->layout_bad = (uint32_t*)(base + p + 8); p += 256;
    w->slot_bytes = c.gslot_bytes;
    w->grid_slots = grid_slots;
    w->gstate = base + p; p += w->slot_bytes * (size_t)grid_slots;
    w->total = p;
}

thread_local int64_t g_launches_sim = 0;
thread_local int g_profiling = 0;
thread_local unsigned long long* g_counts_dev = nullptr;
thread_local bool g_events_valid = false;
thread_local cudaEvent_t g_ev[4] = {nullptr, nullptr, nullptr, nullptr};

void prof_mark(int i, cudaStream_t st)
{
    if (!g_profiling) return;
    if (!g_ev[0])
        for (int k = 0; k < 4; ++k) cudaEventCreate(&g_ev[k]);
    cudaEventRecord(g_ev[i], st);
    if (i == 3) g_events_valid = true;
}

}  // namespace

int64_t sim_last_launches() { return g_launches_sim; }
int profiling_mode() { return g_profiling; }

}  // namespace svf

using namespace svf;

namespace svf {
namespace {

// bytes a call with budget M lays out, with as many global slots as the launch can have CTAs
size_t sim_layout_bytes_at(const svf_trace_t* tr, int P, int64_t M)
{
    SimConfig c = sim_config(tr, M, P);
    SimWs w;
    int64_t slots = c.gslot_bytes ? (int64_t)c.max_cta_per_sm * sm_count() : 0;
    if (slots > tr->n_instances * P) slots = tr->n_instances * P;
    sim_ws_layout(&w, nullptr, tr, c, (int)slots, P);
    return w.total;
}

bool sim_ws_args_ok(const svf_trace_t* tr, int P)
{
    return tr && tr->n_instances >= 0 && tr->n_requests >= 0 && tr->max_instance >= 0 && P >= 1 && P <= MAX_POLICIES;
}

size_t sim_workspace_bytes(const svf_trace_t* tr, int P)
{
    if (!sim_ws_args_ok(tr, P)) return 0;
    // M is not known here and picks the kernel family: size for the largest layout over one probe per
    // class of r_est (see R_EST_BREAKS) and one wide budget
    size_t need = sim_layout_bytes_at(tr, P, 0);
    for (int64_t brk : R_EST_BREAKS) {
        const size_t b = sim_layout_bytes_at(tr, P, R_EST_TOKENS * (brk + 1));
        need = b > need ? b : need;
    }
    const size_t wide = sim_layout_bytes_at(tr, P, (int64_t)1 << 30);
    need = wide > need ? wide : need;
    return need + 256;
}

// the wide sorted-array kernel (M >= 2^30): one policy per call
int simulate_wide(const svf_trace_t* tr, int policy, int64_t M, const svf_result_t* out, const SimConfig& c,
                  SimWs& w, int grid, cudaStream_t st)
{
    const int64_t I = tr->n_instances, N = tr->n_requests;
    SimArgs g;
    g.I = I; g.N = N; g.M = M; g.max_instance = tr->max_instance;
    g.policy = policy; g.O0 = tr->O0; g.O1 = tr->O1; g.sb = c.sb;
    g.off = tr->offsets; g.a = tr->arrival; g.s = tr->prompt; g.o = tr->output; g.okey = tr->output_key; g.bit = tr->bit;
    g.order = w.order[0]; g.rank = w.rank[0]; g.req = w.req[0];
    g.start = out->start; g.finish = out->finish; g.tel = out->total_latency; g.peak = out->peak_kv;
    g.rounds = out->rounds; g.decisions = out->decisions; g.makespan = out->makespan;
    g.status = out->status ? out->status : w.status_tmp[0];
    g.latw = out->p99_latency ? w.words0 : nullptr;
    g.work_ctr = w.work_ctr; g.layout_bad = w.layout_bad; g.gstate = w.gstate; g.slot_bytes = w.slot_bytes; g.cap = c.cap;
    if (cudaMemsetAsync(w.work_ctr, 0, sizeof(unsigned long long), st) != cudaSuccess) return SVF_ECUDA;
    if (N > 0) {
        int64_t blocks = ceil_div(N, 256);
        const int64_t capb = (int64_t)sm_count() * 8;
        if (blocks > capb) blocks = capb;
        k_sim_pack<<<(unsigned)blocks, 256, 0, st>>>(g, w.words0);
        ++g_launches_sim;
        if (sort_u64(w.sort, w.words0, w.words1, w.words0, N, c.sort_lo, c.sort_hi, st, &g_launches_sim)) return SVF_ECUDA;
        k_sim_rank<<<(unsigned)blocks, 256, 0, st>>>(g, w.sort.plan, w.order[0], w.rank[0]);
        ++g_launches_sim;
    }
    prof_mark(1, st);
#define SVF_SIM_LAUNCH(T, S) k_sim<T, S><<<grid, T, c.dyn_smem, st>>>(g)
    if (c.smem) {
        switch (c.threads) {
        case 32: SVF_SIM_LAUNCH(32, true); break;
        case 128: SVF_SIM_LAUNCH(128, true); break;
        case 256: SVF_SIM_LAUNCH(256, true); break;
        default: SVF_SIM_LAUNCH(1024, true); break;
        }
    } else {
        switch (c.threads) {
        case 32: SVF_SIM_LAUNCH(32, false); break;
        case 128: SVF_SIM_LAUNCH(128, false); break;
        case 256: SVF_SIM_LAUNCH(256, false); break;
        default: SVF_SIM_LAUNCH(1024, false); break;
        }
    }
#undef SVF_SIM_LAUNCH
    ++g_launches_sim;
    if (cudaGetLastError() != cudaSuccess) return SVF_ECUDA;
    prof_mark(2, st);
    if (out->p99_latency) {
        if (sort_u64(w.sort, w.words0, w.words1, w.words0, N > 0 ? N : 0, 0, N > 0 ? 32 + c.ib : 32, st, &g_launches_sim)) return SVF_ECUDA;
        k_sim_p99<<<(unsigned)ceil_div(I, 128), 128, 0, st>>>(I, tr->offsets, w.sort.plan, g.status, out->p99_latency);
        ++g_launches_sim;
    }
    return cudaGetLastError() == cudaSuccess ? SVF_OK : SVF_ECUDA;
}

int simulate_impl(const svf_trace_t* tr, int P, const int* policies, int64_t M, const svf_result_t* outs,
                  void* ws, size_t ws_bytes, void* stream)
{
    if (!tr || !outs || !policies || P < 1 || P > MAX_POLICIES) return SVF_EINVAL;
    const int64_t I = tr->n_instances, N = tr->n_requests;
    if (I < 0 || N < 0 || N >= ((int64_t)1 << 30) || tr->max_instance < 0 || tr->max_instance > N) return SVF_EINVAL;
    if (M < 0) return SVF_EINVAL;
    for (int q = 0; q < P; ++q) {
        if (policies[q] < 0 || policies[q] > 3) return SVF_EINVAL;
        if (policies[q] == SVF_SVF_1BIT && ((N > 0 && !tr->bit) || tr->O0 < 1 || tr->O1 < 1)) return SVF_EINVAL;
    }
    if (I == 0) return SVF_OK;
    if (!tr->offsets || (N > 0 && (!tr->arrival || !tr->prompt || !tr->output))) return SVF_EINVAL;
    SimConfig c = sim_config(tr, M, P);
    if (c.sb + 32 + c.ib > 64) return SVF_EINVAL;          // packed sort word would not fit
    if (!ws) return SVF_EWORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    // the caller's buffer must hold what the matching *_workspace_bytes call asks for (less its 256
    // bytes of alignment slack) behind the alignment pad: checked before anything touches the device
    char* base = (char*)align_up((size_t)(uintptr_t)ws, 256);
    if ((size_t)(base - (char*)ws) + (sim_workspace_bytes(tr, P) - 256) > ws_bytes) return SVF_EWORKSPACE;

    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count < 1) return SVF_ECUDA;

    int grid = sim_grid_any(c, I * P);
    if (c.gslot_bytes && grid > c.max_cta_per_sm * sm_count()) grid = c.max_cta_per_sm * sm_count();
    SimWs w;
    sim_ws_layout(&w, base, tr, c, c.gslot_bytes ? grid : 0, P);
    if ((size_t)(base - (char*)ws) + w.total > ws_bytes) return SVF_EWORKSPACE;

    g_events_valid = false;
    prof_mark(0, st);
    // the call-wide layout flag (zeroed here; the per-policy work counter is zeroed again below)
    if (cudaMemsetAsync(w.work_ctr, 0, 16, st) != cudaSuccess) return SVF_ECUDA;
    {
        int64_t blocks = ceil_div(I, 256);
        const int64_t capb = (int64_t)sm_count() * 4;
        if (blocks > capb) blocks = capb;
        k_sim_check_layout<<<(unsigned)blocks, 256, 0, st>>>(I, N, tr->offsets, w.layout_bad);
        ++g_launches_sim;
    }
    if (!c.slots) {
        // M >= 2^30: the wide kernel, one policy after the other
        int rc = SVF_OK;
        for (int q = 0; q < P && rc == SVF_OK; ++q) rc = simulate_wide(tr, policies[q], M, &outs[q], c, w, grid, st);
        prof_mark(3, st);
        return rc;
    }

    // ---- phase A: the priority order of every instance under every policy ---------------------
    SlotArgs q;
    q.I = I; q.N = N; q.M = M; q.max_instance = tr->max_instance;
    q.O0 = tr->O0; q.O1 = tr->O1;
    q.off = tr->offsets; q.a = tr->arrival; q.s = tr->prompt; q.o = tr->output; q.okey = tr->output_key; q.bit = tr->bit;
    q.n_policies = P;
    const bool seg = N > 0 && tr->max_instance <= SEG_SORT_MAX;
    SegSortArgs sa;
    sa.I = I; sa.N = N; sa.cap = 0; sa.off = tr->offsets; sa.s = tr->prompt; sa.o = tr->output; sa.okey = tr->output_key;
    sa.a = tr->arrival; sa.bit = tr->bit; sa.O0 = tr->O0; sa.O1 = tr->O1; sa.n_policies = P;
    for (int k = 0; k < P; ++k) {
        const svf_result_t* out = &outs[k];
        PolicyIO& io = q.io[k];
        io.policy = policies[k];
        io.req = c.qreg ? nullptr : w.req[k];
        io.rank = w.rank[k]; io.order = w.order[k];
        io.start = out->start; io.finish = out->finish; io.tel = out->total_latency; io.peak = out->peak_kv;
        io.rounds = out->rounds; io.decisions = out->decisions; io.p99 = out->p99_latency;
        io.makespan = out->makespan; io.status = out->status;
        io.lat = w.lat[k];
        sa.policy[k] = policies[k]; sa.order[k] = w.order[k]; sa.rank[k] = w.rank[k]; sa.req[k] = c.qreg ? nullptr : w.req[k];
        if (!seg && N > 0) {
            SimArgs g;
            g.I = I; g.N = N; g.M = M; g.max_instance = tr->max_instance;
            g.policy = policies[k]; g.O0 = tr->O0; g.O1 = tr->O1; g.sb = c.sb;
            g.off = tr->offsets; g.a = tr->arrival; g.s = tr->prompt; g.o = tr->output; g.okey = tr->output_key; g.bit = tr->bit;
            g.req = c.qreg ? nullptr : w.req[k];
            int64_t blocks = ceil_div(N, 256);
            const int64_t capb = (int64_t)sm_count() * 8;
            if (blocks > capb) blocks = capb;
            k_sim_pack<<<(unsigned)blocks, 256, 0, st>>>(g, w.words0);
            ++g_launches_sim;
            if (sort_u64(w.sort, w.words0, w.words1, w.words0, N, c.sort_lo, c.sort_hi, st, &g_launches_sim)) return SVF_ECUDA;
            k_sim_rank<<<(unsigned)blocks, 256, 0, st>>>(g, w.sort.plan, w.order[k], w.rank[k]);
            ++g_launches_sim;
        }
    }
    // small instances: keys + stable radix sort + rank in shared memory, one CTA per instance, every
    // policy of the call in ONE launch
    if (seg && seg_sort_keys(sa, tr->max_instance, st, &g_launches_sim)) return SVF_ECUDA;
    prof_mark(1, st);

    // ---- phase B: one persistent launch over P x I work items -------------------------------------
    q.work_ctr = w.work_ctr; q.work_counts = w.counts; q.layout_bad = w.layout_bad;
    q.gstate = w.gstate; q.slot_bytes = w.slot_bytes; q.ecap = c.ecap; q.qcap = c.qcap; q.ext_global = c.ext_global ? 1 : 0;
    const bool count = g_profiling == 2;
    if (count) {
        if (cudaMemsetAsync(w.counts, 0, 4 * sizeof(unsigned long long), st) != cudaSuccess) return SVF_ECUDA;
        g_counts_dev = w.counts;
    }
#define SVF_SLOTS_LAUNCH(T, S, Q, ...)                                                              \
    do {                                                                                            \
        if (count) k_sim_slots<T, SLOT_K, S, true, Q, ##__VA_ARGS__><<<grid, T, c.dyn_smem, st>>>(q);   \
        else       k_sim_slots<T, SLOT_K, S, false, Q, ##__VA_ARGS__><<<grid, T, c.dyn_smem, st>>>(q);  \
    } while (0)
    if (c.qreg && c.qw > 2) {
        if (c.k == 32) {
            if (count) k_sim_slots<32, 32, true, true, true, QREG_MAX_WORDS, true><<<grid, 32, c.dyn_smem, st>>>(q);
            else       k_sim_slots<32, 32, true, false, true, QREG_MAX_WORDS, true><<<grid, 32, c.dyn_smem, st>>>(q);
        } else {
            SVF_SLOTS_LAUNCH(32, true, true, QREG_MAX_WORDS, true);
        }
    } else if (c.qreg) {
        if (c.qw == 2) SVF_SLOTS_LAUNCH(32, true, true, 2);
        else           SVF_SLOTS_LAUNCH(32, true, true, 1);
    } else if (c.k == 32) {
        if (count) k_sim_slots<32, 32, true, true, false><<<grid, 32, c.dyn_smem, st>>>(q);
        else       k_sim_slots<32, 32, true, false, false><<<grid, 32, c.dyn_smem, st>>>(q);
    } else if (c.smem) {
        switch (c.threads) {
        case 32: SVF_SLOTS_LAUNCH(32, true, false); break;
        case 128: SVF_SLOTS_LAUNCH(128, true, false); break;
        default: SVF_SLOTS_LAUNCH(256, true, false); break;
        }
    } else {
        switch (c.threads) {
        case 32: SVF_SLOTS_LAUNCH(32, false, false); break;
        case 128: SVF_SLOTS_LAUNCH(128, false, false); break;
        default: SVF_SLOTS_LAUNCH(256, false, false); break;
        }
    }
#undef SVF_SLOTS_LAUNCH
    ++g_launches_sim;
    if (cudaGetLastError() != cudaSuccess) return SVF_ECUDA;
    prof_mark(2, st);
    prof_mark(3, st);       // phase C (p99) happens inside the kernel
    return SVF_OK;
}

}  // namespace
}  // namespace svf

extern "C" size_t svf_simulate_workspace_bytes(const svf_trace_t* tr) { return sim_workspace_bytes(tr, 1); }

extern "C" size_t svf_simulate_policies_workspace_bytes(const svf_trace_t* tr, int n_policies)
{
    return sim_workspace_bytes(tr, n_policies);
}

extern "C" size_t svf_simulate_layout_bytes(const svf_trace_t* tr, int n_policies, int64_t M)
{
    if (!sim_ws_args_ok(tr, n_policies) || M < 0) return 0;
    return sim_layout_bytes_at(tr, n_policies, M) + 256;
}

extern "C" int svf_simulate(const svf_trace_t* tr, int policy, int64_t M, const svf_result_t* out,
                            void* ws, size_t ws_bytes, void* stream)
{
    g_launches_sim = 0;
    return simulate_impl(tr, 1, &policy, M, out, ws, ws_bytes, stream);
}

extern "C" int svf_simulate_policies(const svf_trace_t* tr, int n_policies, const int* policies, int64_t M,
                                     const svf_result_t* outs, void* ws, size_t ws_bytes, void* stream)
{
    g_launches_sim = 0;
    return simulate_impl(tr, n_policies, policies, M, outs, ws, ws_bytes, stream);
}

extern "C" size_t svf_volume_lower_bound_workspace_bytes(const svf_trace_t* tr) { return sim_workspace_bytes(tr, 1); }

extern "C" int svf_volume_lower_bound(const svf_trace_t* tr, int64_t* lb_out, int32_t* status_out, void* ws,
                                      size_t ws_bytes, void* stream)
{
    g_launches_sim = 0;
    if (!tr || !lb_out) return SVF_EINVAL;
    const int64_t I = tr->n_instances, N = tr->n_requests;
    if (I < 0 || N < 0 || N >= ((int64_t)1 << 30) || tr->max_instance < 0 || tr->max_instance > N) return SVF_EINVAL;
    if (I == 0) return SVF_OK;
    if (!tr->offsets || (N > 0 && (!tr->prompt || !tr->output))) return SVF_EINVAL;
    SimConfig c = sim_config(tr, 0, 1);
    if (c.sb + 32 + c.ib > 64) return SVF_EINVAL;
    if (!ws) return SVF_EWORKSPACE;
    char* base = (char*)align_up((size_t)(uintptr_t)ws, 256);
    if ((size_t)(base - (char*)ws) + (sim_workspace_bytes(tr, 1) - 256) > ws_bytes) return SVF_EWORKSPACE;
    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count < 1) return SVF_ECUDA;
    cudaStream_t st = (cudaStream_t)stream;
    SimWs w;
    sim_ws_layout(&w, base, tr, c, 0, 1);
    if (cudaMemsetAsync(w.work_ctr, 0, 16, st) != cudaSuccess) return SVF_ECUDA;
    {
        int64_t blocks = ceil_div(I, 256);
        const int64_t capb = (int64_t)sm_count() * 4;
        if (blocks > capb) blocks = capb;
        k_sim_check_layout<<<(unsigned)blocks, 256, 0, st>>>(I, N, tr->offsets, w.layout_bad);
        ++g_launches_sim;
    }
    // volumes ascending = the SVF order under the TRUE lengths (no predicted keys here)
    if (N > 0 && tr->max_instance <= SEG_SORT_MAX) {
        SegSortArgs sa;
        sa.I = I; sa.N = N; sa.cap = 0; sa.off = tr->offsets; sa.s = tr->prompt; sa.o = tr->output; sa.okey = nullptr;
        sa.a = tr->prompt /* not read: no records are written */; sa.bit = nullptr; sa.O0 = 0; sa.O1 = 0; sa.n_policies = 1;
        sa.policy[0] = SVF_SVF; sa.order[0] = w.order[0]; sa.rank[0] = w.rank[0]; sa.req[0] = nullptr;
        if (seg_sort_keys(sa, tr->max_instance, st, &g_launches_sim)) return SVF_ECUDA;
    } else if (N > 0) {
        SimArgs g;
        g.I = I; g.N = N; g.M = 0; g.max_instance = tr->max_instance;
        g.policy = SVF_SVF; g.O0 = 0; g.O1 = 0; g.sb = c.sb;
        g.off = tr->offsets; g.a = tr->prompt; g.s = tr->prompt; g.o = tr->output; g.okey = nullptr; g.bit = nullptr;
        g.req = nullptr;
        int64_t blocks = ceil_div(N, 256);
        const int64_t capb = (int64_t)sm_count() * 8;
        if (blocks > capb) blocks = capb;
        k_sim_pack<<<(unsigned)blocks, 256, 0, st>>>(g, w.words0);
        ++g_launches_sim;
        if (sort_u64(w.sort, w.words0, w.words1, w.words0, N, c.sort_lo, c.sort_hi, st, &g_launches_sim)) return SVF_ECUDA;
        k_sim_rank<<<(unsigned)blocks, 256, 0, st>>>(g, w.sort.plan, w.order[0], w.rank[0]);
        ++g_launches_sim;
    }
    int64_t grid = (int64_t)sm_count() * 8;
    if (grid > I) grid = I;
    k_volume_lb<<<(unsigned)grid, 256, 0, st>>>(I, N, tr->max_instance, tr->offsets, tr->prompt, tr->output, w.order[0],
                                                w.layout_bad, lb_out, status_out);
    ++g_launches_sim;
    return cudaGetLastError() == cudaSuccess ? SVF_OK : SVF_ECUDA;
}

extern "C" void svf_set_profiling(int mode) { g_profiling = mode == 2 ? 2 : (mode ? 1 : 0); if (mode != 2) g_counts_dev = nullptr; }

extern "C" int svf_simulate_work_counts(uint64_t* counts_out)
{
    if (!counts_out || !g_counts_dev) return SVF_EINVAL;
    unsigned long long h[4] = {0, 0, 0, 0};
    if (cudaMemcpy(h, g_counts_dev, sizeof(h), cudaMemcpyDeviceToHost) != cudaSuccess) return SVF_ECUDA;
    for (int k = 0; k < 4; ++k) counts_out[k] = h[k];
    return SVF_OK;
}

extern "C" int svf_simulate_phase_ms(float* ms_out)
{
    if (!ms_out || !g_events_valid) return SVF_EINVAL;
    if (cudaEventSynchronize(g_ev[3]) != cudaSuccess) return SVF_ECUDA;
    cudaEventElapsedTime(&ms_out[0], g_ev[0], g_ev[1]);
    cudaEventElapsedTime(&ms_out[1], g_ev[1], g_ev[2]);
    cudaEventElapsedTime(&ms_out[2], g_ev[2], g_ev[3]);
    cudaEventElapsedTime(&ms_out[3], g_ev[0], g_ev[3]);
    return SVF_OK;
}
