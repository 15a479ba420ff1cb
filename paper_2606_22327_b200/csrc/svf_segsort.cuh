// One stable LSD radix pass (8-bit digit) over n 64-bit words held in shared memory, by the whole
// CTA: the building block of the in-CTA sorts (k_seg_sort: the per-instance presort of
// svf_simulate; k_admit_prefix: the completion-time order of svf_admit).  Device code only.
#pragma once

#include "svf_internal.cuh"

namespace svf {

// in -> out (both shared memory, n words each).  Element e = wrp*32*ipt + i*32 + lane is item i of
// lane `lane` of warp `wrp` (warp-striped inside a warp's block of 32*ipt elements), so ranks
// follow the input order = stability.  whist: [THREADS/32][256] words, toff_s: [256],
// warp_tot: [THREADS/32].  ipt = ceil(n / THREADS) <= IPT (IPT sizes the registers).  Ends with a
// barrier: out is complete and whist / toff_s may be reused.
template <int THREADS, int IPT>
__device__ __forceinline__ void seg_pass(const uint64_t* __restrict__ in, uint64_t* __restrict__ out, int n, int ipt,
                                         int shift, uint32_t* whist, uint32_t* toff_s, uint32_t* warp_tot)
{
    constexpr int WARPS = THREADS / 32;
    const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
    for (int i = tid; i < WARPS * SORT_RADIX; i += THREADS) whist[i] = 0;
    __syncthreads();
    const int wbase = wrp * 32 * ipt;
    uint32_t* wh = whist + wrp * SORT_RADIX;
    const uint32_t lt_mask = (1u << lane) - 1u;
    uint64_t key[IPT];            // IPT >= ipt: sized by the template so small segments stay cheap in registers
    uint32_t rank[IPT];
#pragma unroll
    for (int i = 0; i < IPT; ++i) {
        if (i >= ipt) break;                                   // uniform
        const int e = wbase + i * 32 + lane;
        const bool valid = e < n;
        key[i] = valid ? in[e] : 0ull;
        const uint32_t d = valid ? ((uint32_t)(key[i] >> shift) & 0xffu) : SORT_RADIX;
        const uint32_t peers = __match_any_sync(0xffffffffu, d);   // one segment per CTA: latency matters, not issue slots
        const int leader = 31 - __clz(peers);
        uint32_t base = 0;
        if (valid && lane == leader) { base = wh[d]; wh[d] = base + __popc(peers); }
        base = __shfl_sync(0xffffffffu, base, leader);
        __syncwarp();
        rank[i] = base + __popc(peers & lt_mask);
    }
    __syncthreads();
    // digit d (threads 0..255): exclusive scan over warps, then over digits
    uint32_t count = 0;
    if (tid < SORT_RADIX) {
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < WARPS; ++w) { uint32_t c = whist[w * SORT_RADIX + tid]; whist[w * SORT_RADIX + tid] = run; run += c; }
        count = run;
    }
    uint32_t inc = count;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { uint32_t v = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += v; }
    if (lane == 31) warp_tot[wrp] = inc;
    __syncthreads();
    if (tid < SORT_RADIX) {
        uint32_t off = 0;
        for (int w = 0; w < wrp; ++w) off += warp_tot[w];
        toff_s[tid] = off + inc - count;
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < IPT; ++i) {
        if (i >= ipt) break;
        if (wbase + i * 32 + lane < n) {
            const uint32_t d = (uint32_t)(key[i] >> shift) & 0xffu;
            out[toff_s[d] + wh[d] + rank[i]] = key[i];
        }
    }
    __syncthreads();
}

}  // namespace svf
