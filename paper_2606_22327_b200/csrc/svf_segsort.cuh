// One stable LSD radix pass (8-bit digit) over n 64-bit words held in shared memory, by the whole
// CTA: the building block of the in-CTA sorts (k_seg_sort: the per-instance presort of
// svf_simulate; k_admit_prefix: the completion-time order of svf_admit).  Device code only.
#pragma once

#include "svf_internal.cuh"

namespace svf {

// in -> out (both shared memory, n words each).  Element e = wrp*32*ipt + i*32 + lane is item i of
// lane `lane` of warp `wrp` (warp-striped inside a warp's block of 32*ipt elements), so ranks
// follow the input order = stability.  whist: [THREADS/32][256] words, toff_s: [256],
// warp_tot: [THREADS/32].  THREADS: 128 (two digits per thread in the scans), 256 or more.  ipt = ceil(n / THREADS) <= IPT (IPT sizes the registers).  Ends with a
// barrier: out is complete and whist / toff_s may be reused.
// lanes of the warp holding the same digit, by one ballot per digit bit (no MATCH instruction on
// the critical path: measured slower).  Four instructions per bit, written out in PTX because the
// compiler's own form of `peers &= bit ? m : ~m` took six to seven (extract, ISETP, VOTE, NOT, SEL,
// AND): test the bit into a predicate (one LOP3), ballot, complement the ballot where the own bit
// is clear (predicated), and it in.  An invalid lane (past the end of a ragged tile) matches the
// other invalid lanes only.
#ifndef SVF_SORT_USE_MATCH
#define SVF_SORT_USE_MATCH 0
#endif
template <bool FULL>
__device__ __forceinline__ uint32_t warp_match_digit(uint32_t d, bool valid)
{
#if SVF_SORT_USE_MATCH
    return __match_any_sync(0xffffffffu, FULL ? d : (valid ? d : SORT_RADIX));
#else
    uint32_t peers = 0xffffffffu;
    if (!FULL) {
        peers = __ballot_sync(0xffffffffu, valid);
        if (!valid) peers = ~peers;
    }
#pragma unroll
    for (int b = 0; b < SORT_RADIX_BITS; ++b) {
        asm("{\n\t.reg .pred p;\n\t.reg .b32 m, t;\n\t"
            "and.b32 t, %1, %2;\n\t"
            "setp.ne.u32 p, t, 0;\n\t"
            "vote.sync.ballot.b32 m, p, 0xffffffff;\n\t"
            "@!p not.b32 m, m;\n\t"
            "and.b32 %0, %0, m;\n\t}" : "+r"(peers) : "r"(d), "r"(1u << b));
    }
    return peers;
#endif
}

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
        const uint32_t d = (uint32_t)(key[i] >> shift) & 0xffu;
        const uint32_t peers = warp_match_digit<false>(d, valid);
        const int leader = 31 - __clz(peers);
        uint32_t base = 0;
        if (valid && lane == leader) { base = wh[d]; wh[d] = base + __popc(peers); }
        base = __shfl_sync(0xffffffffu, base, leader);
        __syncwarp();
        rank[i] = base + __popc(peers & lt_mask);
    }
    __syncthreads();
    // the first min(THREADS, 256) threads own DPT consecutive digits each: exclusive scan of the warp-
    // private counts over the warps (the digit's offset inside the segment is folded in afterwards, so
    // that the scatter needs one lookup per key), then over the digits
    constexpr int NT = THREADS < SORT_RADIX ? THREADS : SORT_RADIX;     // threads that own digits
    constexpr int DPT = SORT_RADIX / NT;                                 // digits per owning thread
    uint32_t cnt[DPT], tot = 0;
    if (tid < NT) {
#pragma unroll
        for (int q = 0; q < DPT; ++q) {
            const int d = tid * DPT + q;
            uint32_t run = 0;
#pragma unroll
            for (int w = 0; w < WARPS; ++w) { uint32_t c = whist[w * SORT_RADIX + d]; whist[w * SORT_RADIX + d] = run; run += c; }
            cnt[q] = run; tot += run;
        }
    }
    uint32_t inc = tot;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { uint32_t v = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += v; }
    if (lane == 31) warp_tot[wrp] = inc;
    __syncthreads();
    if (tid < NT) {
        uint32_t off = inc - tot;
        for (int w = 0; w < wrp; ++w) off += warp_tot[w];
#pragma unroll
        for (int q = 0; q < DPT; ++q) { toff_s[tid * DPT + q] = off; off += cnt[q]; }
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
