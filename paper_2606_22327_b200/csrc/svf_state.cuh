// The on-chip admission state shared by svf_simulate and svf_admit (device code only).
//
// RUNNING SET (a4, a5).  Requests in flight are kept ordered by finish time f, latest first
// (index 0 = largest f, index R-1 = next to complete).  Entry j stores
//     f_j          absolute finish step                                         (int32)
//     A_j          memory held at time f_j by entries 0..j = mem(f_j) of Eq. 3c  (int64)
// Memory of a fixed set rises by one token per live request per step and only falls after a
// completion, so its future maxima sit at completion times: the set is feasible iff
// every A_j <= M.  A_j does not depend on the current time, so nothing is touched on a step
// without admissions; completions pop from the tail.
//
// ADMITTING h at time t (s_h, o_h; f_h = t + o_h, it holds s_h + (tau - t) at tau in (t, f_h]):
//     pos = #{ j : f_j >= f_h }                       entries that outlive h keep their A_j
//     (1) A_h = A_{pos-1} - pos (f_{pos-1} - f_h) + s_h + o_h  <= M    (A_h = s_h + o_h if pos = 0)
//     (2) for every j >= pos:  A_j + s_h + (f_j - t) <= M
// (1) is mem(f_h) with h added: the pos entries alive at f_{pos-1} each hold (f_{pos-1} - f_h)
// fewer tokens at the earlier time f_h, plus h's own s_h + o_h.  (2) adds h's tokens at each
// earlier completion time.  Both are the forward-looking check of P:L516 / Eq. 3c evaluated
// at the only times where a maximum can occur.  On admission entries j >= pos move one slot
// down with A_j += s_h + f_j - t, and (f_h, A_h) is written at pos.
//
// Entries with equal f: h goes after them; an entry that is not the last of its group then
// carries a partial sum, which is smaller than the group's last entry (every term is > 0), so
// it never decides the check (same argument as in the oracle's completion-time form).
//
// WAITING QUEUE (D2).  Keys do not depend on time, so the priority order of an instance is
// fixed by the presort: the queue at time t is { rank r : arrived and not started }, held as a
// two-level bitmap over ranks; head = lowest set bit.
#pragma once

#include "svf_internal.cuh"

namespace svf {

constexpr uint32_t FULL = 0xffffffffu;

template <int THREADS>
struct Group {
    static constexpr int WARPS = THREADS / 32;

    __device__ static __forceinline__ void sync()
    {
        if (THREADS == 32) __syncwarp(); else __syncthreads();
    }
    // (sum of a, max of b) over the group; scratch: int[2][2*32], parity alternates per call
    __device__ static __forceinline__ void sum_max(int& a, int& b, int (*scratch)[64], int& parity)
    {
        a = __reduce_add_sync(FULL, a);
        b = __reduce_max_sync(FULL, b);
        if (THREADS > 32) {
            const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
            int* sc = scratch[parity];
            parity ^= 1;
            if (lane == 0) { sc[2 * wrp] = a; sc[2 * wrp + 1] = b; }
            __syncthreads();
            int va = lane < WARPS ? sc[2 * lane] : 0;
            int vb = lane < WARPS ? sc[2 * lane + 1] : INT32_MIN;
            a = __reduce_add_sync(FULL, va);
            b = __reduce_max_sync(FULL, vb);
        }
    }
    __device__ static __forceinline__ uint32_t or_u32(uint32_t v, int (*scratch)[64], int& parity)
    {
        v = __reduce_or_sync(FULL, v);
        if (THREADS > 32) {
            const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
            int* sc = scratch[parity];
            parity ^= 1;
            if (lane == 0) sc[wrp] = (int)v;
            __syncthreads();
            v = __reduce_or_sync(FULL, lane < WARPS ? (uint32_t)sc[lane] : 0u);
        }
        return v;
    }
    // max of non-negative int64 (two 32-bit hardware reductions: high words, then low words)
    __device__ static __forceinline__ int64_t max_i64_nonneg(int64_t v, int (*scratch)[64], int& parity)
    {
        auto warp_max = [](int64_t x) {
            uint32_t hi = (uint32_t)((uint64_t)x >> 32), lo = (uint32_t)x;
            uint32_t mh = __reduce_max_sync(FULL, hi);
            uint32_t ml = __reduce_max_sync(FULL, hi == mh ? lo : 0u);
            return (int64_t)(((uint64_t)mh << 32) | ml);
        };
        v = warp_max(v);
        if (THREADS > 32) {
            const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
            int* sc = scratch[parity];
            parity ^= 1;
            if (lane == 0) { sc[2 * wrp] = (int)(uint32_t)((uint64_t)v >> 32); sc[2 * wrp + 1] = (int)(uint32_t)v; }
            __syncthreads();
            int64_t x = lane < WARPS ? (int64_t)(((uint64_t)(uint32_t)sc[2 * lane] << 32) | (uint32_t)sc[2 * lane + 1]) : 0;
            v = warp_max(x);
        }
        return v;
    }
    __device__ static __forceinline__ int64_t sum_i64(int64_t v, int (*scratch)[64], int& parity)
    {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(FULL, v, d);
        if (THREADS > 32) {
            const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
            int* sc = scratch[parity];
            parity ^= 1;
            if (lane == 0) { sc[2 * wrp] = (int)(uint32_t)((uint64_t)v >> 32); sc[2 * wrp + 1] = (int)(uint32_t)v; }
            __syncthreads();
            int64_t x = lane < WARPS ? (int64_t)(((uint64_t)(uint32_t)sc[2 * lane] << 32) | (uint32_t)sc[2 * lane + 1]) : 0;
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) x += __shfl_xor_sync(FULL, x, d);
            v = x;
        }
        return v;
    }
};

// Verdict of one forward-looking check
struct Verdict {
    int     pos;     // insertion slot
    int64_t Ah;      // mem(f_h) with h added
    bool    ok;      // (1) and (2) hold
    int     wait;    // if !ok: h stays blocked for at least this many steps (>= 1) while no
                     // completion or arrival happens (condition (2) relaxes by one per step)
};

// Evaluate the head (sh, oh) at time t against the running set (f, A)[0..R).  Uniform result in
// every thread of the group.
template <int THREADS>
__device__ __forceinline__ Verdict evaluate_head(const int32_t* f, const int64_t* A, int R, int32_t t,
                                                 int32_t sh, int32_t oh, int64_t M,
                                                 int (*scratch)[64], int& parity)
{
    const int64_t fh = (int64_t)t + oh;
    const int64_t T = M - sh + t;                 // (2): A_j + f_j <= M - s_h + t
    int cnt = 0, dmax = INT32_MIN;
    for (int j = threadIdx.x; j < R; j += THREADS) {
        const int32_t fj = f[j];
        if ((int64_t)fj >= fh) ++cnt;
        else {
            int64_t v = A[j] + fj - T;            // > 0: violated by v tokens
            int vi = v > (int64_t)INT32_MAX ? INT32_MAX : (v < (int64_t)INT32_MIN ? INT32_MIN : (int)v);
            dmax = vi > dmax ? vi : dmax;
        }
    }
    Group<THREADS>::sum_max(cnt, dmax, scratch, parity);
    Verdict v;
    v.pos = cnt;
    v.Ah = (int64_t)sh + oh;
    if (cnt > 0) v.Ah += A[cnt - 1] - (int64_t)cnt * ((int64_t)f[cnt - 1] - fh);
    const bool ok2 = dmax <= 0;
    v.ok = ok2 && v.Ah <= M;
    v.wait = ok2 ? 1 : dmax;
    return v;
}

// Insert the admitted head at slot pos (see header comment).  All threads of the group call it;
// the arrays are consistent for every thread after it returns.
template <int THREADS>
__device__ __forceinline__ void insert_head(int32_t* f, int64_t* A, int R, int pos, int32_t t,
                                            int32_t sh, int32_t oh, int64_t Ah)
{
    const int64_t add = (int64_t)sh - t;          // A_j += s_h + f_j - t
    for (int hi = R; hi > pos; hi -= THREADS) {   // chunks from the tail, so nothing is clobbered
        const int j = hi - 1 - (int)threadIdx.x;
        const bool act = j >= pos;
        int32_t fj = 0; int64_t Aj = 0;
        if (act) { fj = f[j]; Aj = A[j]; }
        Group<THREADS>::sync();
        if (act) { f[j + 1] = fj; A[j + 1] = Aj + add + fj; }
        Group<THREADS>::sync();
    }
    if (threadIdx.x == 0) { f[pos] = t + oh; A[pos] = Ah; }
    Group<THREADS>::sync();
}

// ---- waiting queue: two-level bitmap over ranks ------------------------------------------------
// L0: one bit per rank; L1: one bit per non-empty L0 word.  Lowest set bit at or above L1 word
// `from` (every warp computes it redundantly from the same shared data: no barrier needed).
__device__ __forceinline__ int queue_min(const uint32_t* L0, const uint32_t* L1, int nL1, int from)
{
    const int lane = threadIdx.x & 31;
    for (int w1 = from; w1 < nL1; w1 += 32) {
        const int idx = w1 + lane;
        const uint32_t v = idx < nL1 ? L1[idx] : 0u;
        const uint32_t b = __ballot_sync(FULL, v != 0u);
        if (b) {
            const int l = __ffs(b) - 1;
            const uint32_t word1 = __shfl_sync(FULL, v, l);
            const int i0 = (w1 + l) * 32 + (__ffs(word1) - 1);
            return i0 * 32 + (__ffs(L0[i0]) - 1);
        }
    }
    return INT32_MAX;
}
__device__ __forceinline__ void queue_set(uint32_t* L0, uint32_t* L1, int r)
{
    atomicOr(&L0[r >> 5], 1u << (r & 31));
    atomicOr(&L1[r >> 10], 1u << ((r >> 5) & 31));
}
// single thread
__device__ __forceinline__ void queue_clear(uint32_t* L0, uint32_t* L1, int r)
{
    const uint32_t w = L0[r >> 5] & ~(1u << (r & 31));
    L0[r >> 5] = w;
    if (w == 0u) L1[r >> 10] &= ~(1u << ((r >> 5) & 31));
}

}  // namespace svf
