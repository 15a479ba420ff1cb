// The register-resident simulator kernel (a4-a7), included by svf_simulate.cu; svf_admit.cu reuses its slot passes.
//
// RUNNING SET as unordered SLOTS.  Slot j of an instance holds, for one request in flight,
//     f_j   absolute finish step (int32); the slot is DEAD (free) once f_j <= t (0 = never used)
//     B_j   A_j + f_j  (mod 2^32), A_j = mem(f_j) of Eq. 3c for the current running set
//     c_j   s_j - k_j  (mod 2^32)
// The memory of a fixed set peaks at completion times only, so the set is feasible iff
// every live A_j <= M.  Admitting h = (s_h, o_h) at time t, f_h = t + o_h:
//     (1)  A_h = s_h + o_h + sum_{f_i >= f_h} (c_i + f_h)                            <= M
//     (2)  for every live j with f_j <= f_h:   A_j + s_h + (f_j - t)                <= M
// and on admission every such j gets A_j += s_h + f_j - t.  Nothing depends on the ORDER of
// the slots: no sorted array, no shifting; a pass is straight-line code over the slots, the
// first THREADS*K of which live in REGISTERS (slot k*THREADS + tid is register k of thread
// tid); the rest (only when more than THREADS*K requests run at once) sit in an `ext` array
// that is only ever touched by the owning thread.
//
// ONE PASS per evaluation, straight-line code, per slot (compile-time register index):
//     x = f - (t+1)            as unsigned: x < 2^31 iff the slot is live (f > t)
//     in = x <u o_h            live and f <= f_h            (condition (2) applies)
//     ge = f >= f_h            (a dead slot has f <= t < f_h)
//     if (ge) acc += c + f_h                                (condition (1))
//     if (in) viol = max(viol, B + (s_h - t - M))           one VIADDMNMX
//     if (in) B += s_h - t + f                              the admission update, SPECULATIVELY
//     dead-bit of x shifted into a mask                     (free-slot search, one SHF)
// about 6.5 alu-pipe + 2 fma-pipe instructions; then one round of three warp reductions (sum,
// max, min).  If the head is admitted the update is already in place and the head is written into
// the lowest free slot; if it is BLOCKED one more pass takes the update back and finds how long
// the head must stay blocked (below).
//
// Arithmetic is 32 bit, wrapping: every TRUE value that is compared lies in [-M, 2M] and the
// host takes this kernel only when M < 2^30, so the wrapped result read as int32 is exact.
// peak_kv = max over all A values ever produced (each entry's final A_j is mem(f_j)).
//
// TIME ADVANCE (exact, R1/R16).  Completions are implicit.  With an empty queue nothing can
// happen before the next arrival.  A BLOCKED head h stays blocked while the running set only
// shrinks (nobody may bypass it), and each obstacle has a closed-form end:
//   * a violated (2) at slot j clears at min(f_j, t + v_j), v_j = A_j + s_h + f_j - t - M (it
//     relaxes by one token per step; A_j is fixed while nothing is admitted);
//   * a violated (1) holds at least until the first of the summed slots drops out of the sum:
//     t' + o_h > min{f_i : f_i >= f_h}.
// The head is re-evaluated at t_lb = the latest of these ends, or earlier if an arrival takes
// its place at the head of the queue; the steps in between are counted into rounds/decisions
// exactly as the step-by-step definition counts them (one blocked-head evaluation each).
//
// WAITING QUEUE: bitmap over ranks (keys are time-invariant, so the presort fixes the order).
//  * QREG (one warp per instance, at most 8,192 requests): QW 32-bit words per lane in registers
//    (QW = 1, 2 or 8: 1,024 ranks per word index), mirrored in shared memory where arrivals set their
//    bits with one atomic OR each; with one word per lane (the bench shape) the ranks are interleaved
//    over the lanes and the head is one warp reduction, with more words a lane holds consecutive ranks
//    and the head's word is cached uniformly (ILV in the kernel); the (s, o) of every request sits in shared memory by rank, staged
//    once per instance, so picking the next head never waits for global memory; id and arrival are
//    only looked up when the outputs are written.  Up to 2,048 requests the records are 8 bytes; above
//    (REC4) they are PACKED into one word, s in the low bits, the split taken from the widths of the
//    instance's own largest s and o (32 KB for 8,192 ranks: six warps per SM; an instance whose widths
//    do not fit 32 bits together reads the records from global memory instead: correct, slower).
//  * otherwise the two-level shared-memory bitmap of svf_state.cuh and (s, o, id, a) records in
//    priority order in global memory.
// The head of the queue is cached in registers (non-QREG: also the second, whose record is
// fetched one admission ahead to hide the L2 latency).  ARRIVALS come from a 32-wide register window over
// (a, s, o, rank), refilled once per 32 arrivals.  OUTPUTS (start, finish, latency word): QREG: the start
// time of an admitted request replaces its record in shared memory and everything is written at the
// end of the instance in index order (coalesced); otherwise buffered one admission per lane and written
// 32 at a time.  p99 (nearest rank) is a radix selection over the instance's latencies by the same
// thread group at the end of the instance.
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

// the register bitmap (QREG): lane l holds ranks [32 l, 32 l + 32).  Smallest set bit >= q.
__device__ __forceinline__ int qreg_first_ge(uint32_t word, int q)
{
    const int lane = threadIdx.x & 31;
    const int w0 = q >> 5;
    if (lane == w0) word &= ~0u << (q & 31);
    if (lane < w0) word = 0u;
    const uint32_t b = __ballot_sync(FULL, word != 0u);
    if (!b) return INT_MAX;
    const int l = __ffs(b) - 1;
    const uint32_t wv = __shfl_sync(FULL, word, l);
    return l * 32 + (__ffs(wv) - 1);
}

// per-policy inputs (the presorted order) and outputs of one launch
struct PolicyIO {
    int policy;
    const int4* req;                 // [N] (s, o, id, a) at (instance offset + rank); NULL under QREG
    const uint32_t* rank;            // [N] rank of (instance offset + local id)
    const uint32_t* order;           // [N] local id at (instance offset + rank)
    int32_t *start, *finish;
    int64_t *tel, *peak, *rounds, *decisions;
    int64_t* p99;                    // [I] or NULL
    int32_t *makespan, *status;
    uint32_t* lat;                   // [N] latency of (instance offset + local id): scratch of the p99 selection
};
constexpr int MAX_POLICIES = 8;

// One launch simulates n_policies x I work items (policy-major): a batch is usually compared
// under several policies, and one long queue of items keeps the tail of the launch short.
struct SlotArgs {
    int64_t I, N, M, max_instance;
    int32_t O0, O1;
    const int64_t* off;
    const int32_t *a, *s, *o;
    const int32_t* okey;             // [N] predicted lengths for the SVF / SJF key, or NULL
    const uint8_t* bit;
    int n_policies;
    PolicyIO io[MAX_POLICIES];
    unsigned long long* work_ctr;
    const uint32_t* layout_bad;      // one word: the offsets of the call are not monotone (k_sim_check_layout)
    unsigned long long* work_counts; // [4] E, U, evaluations, blocked evaluations (COUNT variant only)
    char* gstate; size_t slot_bytes; // per-CTA state when it does not fit in shared memory
    int ext_global;                  // bitmaps in shared memory, ext slots in the per-CTA global slot
    int ecap;                        // ext slots per instance
    int qcap;                        // bitmap capacity (ranks)
};

__host__ __device__ inline size_t slot_state_bytes(int qcap, int ecap)
{
    const int nL0 = (qcap + 31) / 32, nL1 = (nL0 + 31) / 32;
    return align_up((size_t)nL0 * 4, 16) + align_up((size_t)nL1 * 4, 16) + 3 * align_up((size_t)ecap * 4, 16);
}
// QREG: shared memory holds the (s, o) records by rank and the bitmap mirror; the ext slots
// (touched only when more than 32*K requests run at once) live in a global slot per CTA
// (QW bitmap words per lane: 1,024 ranks each; QW = 1 for the bench shape, 2 for instances up to 2,048,
// 8 for instances up to 8,192, whose (s, o) records are PACKED into one 32-bit word each (REC4): 32 KB
// instead of 64 KB per warp, six warps per SM instead of three)
constexpr int QREG_RANKS = 1024;
constexpr int QREG_MAX_WORDS = 8;
__host__ __device__ constexpr size_t qreg_smem_bytes(int qw, bool rec4 = false)      // (s, o) by rank (the start time once admitted), bitmap mirror
{
    return (size_t)QREG_RANKS * qw * (rec4 ? 4 : 8) + (size_t)32 * qw * 4;
}
constexpr size_t QREG_SMEM_BYTES = qreg_smem_bytes(1);
__host__ __device__ inline size_t qreg_ext_bytes(int ecap) { return 3 * align_up((size_t)ecap * 4, 16); }

// one reduction round over the group: a summed (mod 2^32), b maxed, c minned; uniform afterwards
template <int THREADS>
__device__ __forceinline__ void reduce_add_max_min(uint32_t& a, int& b, int& c, int (*red)[THREADS / 32][3], int& parity)
{
    a = __reduce_add_sync(FULL, a);
    b = __reduce_max_sync(FULL, b);
    c = __reduce_min_sync(FULL, c);
    if (THREADS > 32) {
        constexpr int WARPS = THREADS / 32;
        const int lane = threadIdx.x & 31, wrp = threadIdx.x >> 5;
        int (*sc)[3] = red[parity];
        parity ^= 1;
        if (lane == 0) { sc[wrp][0] = (int)a; sc[wrp][1] = b; sc[wrp][2] = c; }
        __syncthreads();
        // every thread combines the warps' triples itself (broadcast loads, a few ALU operations): a second
        // round of warp reductions costs their latency once more on the serial chain
        uint32_t sa = 0; int sb = INT_MIN, scn = INT_MAX;
#pragma unroll
        for (int w = 0; w < WARPS; ++w) {
            sa += (uint32_t)sc[w][0];
            sb = sc[w][1] > sb ? sc[w][1] : sb;
            scn = sc[w][2] < scn ? sc[w][2] : scn;
        }
        a = sa; b = sb; c = scn;
    }
}


// k-th smallest (k >= 1) of v[0..n) by MSB-first radix selection, all threads of the group, result
// uniform.  One 256-bin histogram in shared memory per significant byte; v was written by this
// group before a barrier (read with ld.cg, never through the non-coherent path).
template <int THREADS>
// (sub != NULL: the values are v[i] - sub[i]: the register-queue kernels store finish times and take the
// arrivals off here, in index order, instead of gathering a[id] in the output flush)
__device__ __forceinline__ uint32_t group_select_kth(const uint32_t* v, int n, int k, uint32_t* hist,
                                                     int (*scratch)[64], int& parity, const int32_t* sub = nullptr)
{
    using G = Group<THREADS>;
    const int tid = threadIdx.x, lane = tid & 31;
    uint32_t vor = 0;
#pragma unroll 8
    for (int i = tid; i < n; i += THREADS) vor |= __ldcg(v + i) - (sub ? (uint32_t)sub[i] : 0u);
    vor = G::or_u32(vor, scratch, parity);
    uint32_t prefix = 0, pmask = 0;
    for (int shift = vor ? ((31 - __clz(vor)) & ~7) : 0; shift >= 0; shift -= 8) {
        for (int i = tid; i < 256; i += THREADS) hist[i] = 0;
        G::sync();
#pragma unroll 8
        for (int i = tid; i < n; i += THREADS) {       // (unrolled: eight L2 loads in flight per thread)
            const uint32_t x = __ldcg(v + i) - (sub ? (uint32_t)sub[i] : 0u);
            if ((x & pmask) == prefix) atomicAdd(&hist[(x >> shift) & 255u], 1u);
        }
        G::sync();
        // every warp redundantly: lane l owns digits 8l .. 8l+7
        uint32_t c[8], s8 = 0;
#pragma unroll
        for (int q = 0; q < 8; ++q) { c[q] = hist[lane * 8 + q]; s8 += c[q]; }
        uint32_t inc = s8;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const uint32_t u = __shfl_up_sync(FULL, inc, d); if (lane >= d) inc += u; }
        const uint32_t b = __ballot_sync(FULL, inc >= (uint32_t)k);
        const int L = b ? __ffs(b) - 1 : 31;
        const int kk = k - (int)__shfl_sync(FULL, inc - s8, L);
        int d = 7; uint32_t cum = 0;
        {
            uint32_t run = 0; bool found = false;
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                if (!found && run + c[q] >= (uint32_t)kk) { d = q; cum = run; found = true; }
                run += c[q];
            }
        }
        d = __shfl_sync(FULL, d, L);
        cum = __shfl_sync(FULL, cum, L);
        k = kk - (int)cum;
        prefix |= (uint32_t)(L * 8 + d) << shift;
        pmask |= 255u << shift;
        G::sync();
    }
    return prefix;
}

// The slot passes are straight-line code over the register slots, no loop, no indexed branch.  A slot past
// the high-water mark is dead (f = 0) and costs its instructions only.
// k_admit_slots (svf_admit.cu): groups of four slots behind a ladder of uniform compares (g4 = groups in use)
#define SVF_SLOT_GROUPS(g4, OP)                                                               \
    if ((g4) >= 4) { OP(15) OP(14) OP(13) OP(12) }                                            \
    if ((g4) >= 3) { OP(11) OP(10) OP(9)  OP(8)  }                                            \
    if ((g4) >= 2) { OP(7)  OP(6)  OP(5)  OP(4)  }                                            \
    if ((g4) >= 1) { OP(3)  OP(2)  OP(1)  OP(0)  }
// k_sim_slots: sixteen slots in ONE basic block while more than eight slots per thread are in use, else eight
// (g4 is 4 or 2 here -- 8 with 32 slots per thread: sixteen more in a block of their own --, see the pass):
// sixteen independent chains per block, a fifth of the branches, half the code of one block per group of
// four -- measured on the bench kernel: 6.12 -> 6.05 ms (one block per group count 6.08, always sixteen
// 6.11, eight + eight 6.06), with the one-compare block choice 5.89; on a lone warp (configs[1]) 1.49 -> 1.34 ms
#define SVF_SLOT_GROUPS_8(g4, OP)                                                             \
    if ((g4) >= 3) { OP(15) OP(14) OP(13) OP(12) OP(11) OP(10) OP(9) OP(8) OP(7) OP(6) OP(5) OP(4) OP(3) OP(2) OP(1) OP(0) }  \
    else if ((g4) >= 1) { OP(7)  OP(6)  OP(5)  OP(4)  OP(3)  OP(2)  OP(1) OP(0) }
#define SVF_SLOT_GROUPS32_16(g4, OP)                                                          \
    if ((g4) >= 5) { OP(31) OP(30) OP(29) OP(28) OP(27) OP(26) OP(25) OP(24) OP(23) OP(22) OP(21) OP(20) OP(19) OP(18) OP(17) OP(16) }  \
    SVF_SLOT_GROUPS_8(g4, OP)
#define SVF_SLOTS(g4, OP) if constexpr (K == 32) { SVF_SLOT_GROUPS32_16(g4, OP) } else { SVF_SLOT_GROUPS_8(g4, OP) }

// write into register slot ik (uniform) of the owning thread: a tree of uniform branches
#define SVF_PUT2(ik, OP, k0)  if ((ik) & 1) { OP(k0 + 1) } else { OP(k0) }
#define SVF_PUT4(ik, OP, k0)  if ((ik) & 2) { SVF_PUT2(ik, OP, k0 + 2) } else { SVF_PUT2(ik, OP, k0) }
#define SVF_PUT8(ik, OP, k0)  if ((ik) & 4) { SVF_PUT4(ik, OP, k0 + 4) } else { SVF_PUT4(ik, OP, k0) }
// (two levels of uniform branches, then the four slots of the group under predicates: a quarter of the
// code of the full tree)
#define SVF_PUTG(ik, k0)  { const int j_ = (ik) & 3;                                          \
    if (mine && j_ == 0) { f[k0] = fh; B[k0] = Bh; c[k0] = add; }                                 \
    if (mine && j_ == 1) { f[k0 + 1] = fh; B[k0 + 1] = Bh; c[k0 + 1] = add; }                     \
    if (mine && j_ == 2) { f[k0 + 2] = fh; B[k0 + 2] = Bh; c[k0 + 2] = add; }                     \
    if (mine && j_ == 3) { f[k0 + 3] = fh; B[k0 + 3] = Bh; c[k0 + 3] = add; } }
#define SVF_PUT16G(ik)        if ((ik) & 8) { if ((ik) & 4) SVF_PUTG(ik, 12) else SVF_PUTG(ik, 8) } else { if ((ik) & 4) SVF_PUTG(ik, 4) else SVF_PUTG(ik, 0) }
#define SVF_PUT16(ik, OP)     if ((ik) & 8) { SVF_PUT8(ik, OP, 8) } else { SVF_PUT8(ik, OP, 0) }
#define SVF_PUT32(ik, OP)     if ((ik) & 16) { if ((ik) & 8) { SVF_PUT8(ik, OP, 24) } else { SVF_PUT8(ik, OP, 16) } } else { SVF_PUT16(ik, OP) }
#define SVF_PUT32G(ik)        if ((ik) & 16) { if ((ik) & 8) { if ((ik) & 4) SVF_PUTG(ik, 28) else SVF_PUTG(ik, 24) } else { if ((ik) & 4) SVF_PUTG(ik, 20) else SVF_PUTG(ik, 16) } } else { SVF_PUT16G(ik) }
// LAT (kernels that run as a few lone groups: latency matters, not the instruction count): the compact form
#define SVF_PUTK(ik, OP)      if constexpr (LAT) { if constexpr (K == 32) { SVF_PUT32G(ik) } else { SVF_PUT16G(ik) } }        \
                              else if constexpr (K == 32) { SVF_PUT32(ik, OP) } else { SVF_PUT16(ik, OP) }

// The per-slot operations of the passes.  They are macros over the LOCAL names of the calling
// kernel (k_sim_slots here, k_admit_slots in svf_admit.cu): slots f[], B[], c[]; the head's t1 =
// t + 1, oh = o_h, fh / fhu = f_h, Kc = s_h - t - M, add = s_h - t; accumulators acc, viol, dm
// (evaluation) and wmax, minge (blocked head); cntE / cntU under COUNT.
#ifndef SVF_EVAL_FMA
#define SVF_EVAL_FMA 1
#endif
#ifndef SVF_EVAL_FMA_B
#define SVF_EVAL_FMA_B 1
#endif
#if SVF_EVAL_FMA
// condition (1) on the FMA pipe: the alu pipe is the busy one (ISETP, VIADDMNMX, SHF, IADD3 take one
// warp instruction per two cycles per scheduler, and so does the fma pipe, which is nearly idle
// here), so the predicated accumulate is an IMAD by a register that holds 1 (`one`: a run-time
// value, or ptxas would turn it back into SEL + IADD3 on the alu pipe); two accumulators
#define SVF_ACC_GE(k) {                                                                        \
    const uint32_t tmp_ = c[k] + fhu;                                  \
    if ((k) & 1) asm("{\n\t.reg .pred p;\n\tsetp.ge.s32 p, %1, %2;\n\t@p mad.lo.u32 %0, %3, %4, %0;\n\t}" : "+r"(acc1) : "r"(f[k]), "r"(fh), "r"(tmp_), "r"(one)); \
    else         asm("{\n\t.reg .pred p;\n\tsetp.ge.s32 p, %1, %2;\n\t@p mad.lo.u32 %0, %3, %4, %0;\n\t}" : "+r"(acc) : "r"(f[k]), "r"(fh), "r"(tmp_), "r"(one)); \
}
#else
#define SVF_ACC_GE(k) { if (f[k] >= fh) acc += c[k] + fhu; }
#endif
#define SVF_EVAL(k) {                                                                          \
    const uint32_t x = (uint32_t)f[k] - t1;                            \
    SVF_ACC_GE(k)                                                      \
    if (x < oh) {                                                      \
        viol = __viaddmax_s32((int)B[k], (int)Kc, viol);               \
        if (SVF_EVAL_FMA_B && ((k) & 3) == 1) {                        \
            asm("mad.lo.u32 %0, %1, %2, %0;" : "+r"(B[k]) : "r"(f[k]), "r"(one));       \
            asm("mad.lo.u32 %0, %1, %2, %0;" : "+r"(B[k]) : "r"(add), "r"(one));        \
        } else B[k] += add + (uint32_t)f[k];                           \
        if (COUNT) cntU += 1;                                          \
    }                                                                  \
    dm = __funnelshift_l(x, dm, 1);                                    \
    if (COUNT) cntE += (long long)((x >> 31) ^ 1u);                    \
}
#define SVF_BLOCK(k) {                                                                         \
        const uint32_t x = (uint32_t)f[k] - t1;                        \
        if (x < oh) {                                                  \
            B[k] -= add + (uint32_t)f[k];                              \
            const int v = (int)(B[k] + Kc), d = (int)x + 1;            \
            const int w = v < d ? v : d;                               \
            wmax = w > wmax ? w : wmax;                                \
            if (COUNT) cntU -= 1;                                      \
        }                                                              \
        if (f[k] >= fh) minge = f[k] < minge ? f[k] : minge;           \
    }
// the same when only condition (2) failed: the end of a violated (1) (minge) is not needed
#define SVF_BLOCK2(k) {                                                                        \
        const uint32_t x = (uint32_t)f[k] - t1;                        \
        if (x < oh) {                                                  \
            B[k] -= add + (uint32_t)f[k];                              \
            const int v = (int)(B[k] + Kc), d = (int)x + 1;            \
            const int w = v < d ? v : d;                               \
            wmax = w > wmax ? w : wmax;                                \
            if (COUNT) cntU -= 1;                                      \
        }                                                              \
    }
#define SVF_PUT(k) if (mine) { f[k] = fh; B[k] = Bh; c[k] = add; }

// Register budget of the warp kernel: without a bound ptxas takes 127 registers (16 warps per SM);
// asked for 19 CTAs per SM it fits the kernel into 96 registers WITHOUT spills (21 warps per SM
// resident) and the launch is 5 % faster; 20 also gives 96 registers but a slower schedule, 17-18
// and 21 spill (all measured on configs[2], profiles/r01_kslots_full.md).
#ifndef SVF_WARP_MIN_CTAS
#define SVF_WARP_MIN_CTAS 19
#endif
template <int THREADS, int K, bool SMEM, bool COUNT, bool QREG, int QW = 1, bool REC4 = false>
__global__ void __launch_bounds__(THREADS, (THREADS == 32 && QREG) ? (QW == 1 ? SVF_WARP_MIN_CTAS : (QW == 2 ? 12 : 6)) : 1) k_sim_slots(SlotArgs g)
{
    static_assert(QW >= 1 && QW <= QREG_MAX_WORDS && (QREG || QW == 1), "QW: bitmap words per lane of the register queue");
    static_assert(!REC4 || QREG, "REC4: packed records of the register queue");
    constexpr int QRANKS = QREG_RANKS * QW;
    // the bench-shaped kernel (thousands of one-warp items: 20 warps per SM share the issue ports) is tuned
    // for instruction count; every other form runs as a few groups per SM and is tuned for the length of its
    // serial chain (measured: the choices below are worth 1-2 % each there and cost the bench kernel 0.5-3 %)
    constexpr bool LAT = !(QREG && QW == 1);
    // one bitmap word per lane (the bench shape): the bitmap is INTERLEAVED over the lanes, rank r = bit r >> 5
    // of lane r & 31, and the lowest waiting rank is ONE warp reduction (every lane offers its lowest set bit
    // as (bit << 5) | lane = the rank itself): no ballot + shuffle, no cached word of the head (5.53 -> 5.37 ms
    // per bench step).  With more words per lane the lanes hold consecutive ranks and the head's word is
    // cached (measured: the interleaved form costs configs[4] 10-20 % there)
    constexpr bool ILV = QREG && QW == 1;
    constexpr int RB = REC4 ? 4 : 8;                             // bytes of a waiting record in shared memory
    constexpr int OFF_BITS = QRANKS * RB;
    static_assert(K == 16 || (K == 32 && THREADS == 32 && (!QREG || REC4)), "the slot macros are written out for 16 slots per thread (32: one-warp groups)");
    static_assert(!QREG || (THREADS == 32 && SMEM), "QREG: one warp per instance, queue records in shared memory");
    using G = Group<THREADS>;
    constexpr int WARPS = THREADS / 32;
    constexpr int REGCAP = THREADS * K;
    constexpr int TSHIFT = THREADS == 32 ? 5 : (THREADS == 128 ? 7 : 8);
    static_assert((1 << TSHIFT) == THREADS, "THREADS must be 32, 128 or 256");
    extern __shared__ __align__(16) char dyn_smem[];
    __shared__ int scratch[2][64];
    __shared__ int red[2][WARPS][3];
    __shared__ long long inst_s;
    __shared__ __align__(16) int4 pre_s[2][WARPS];      // non-QREG: prefetched record of the second waiting request, per warp
    // the p99 selection's histogram: its own kilobyte, except under QREG where it reuses the (s, o)
    // records (dead once the instance is simulated; one kilobyte less per CTA = one more CTA per SM)
    __shared__ uint32_t hist_s[QREG ? 1 : 256];
    uint32_t* hist = QREG ? reinterpret_cast<uint32_t*>(dyn_smem) : hist_s;
    int parity = 0, rparity = 0;
    const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;

    // state placement: QREG: records + bitmap mirror in shared memory, ext slots in the global
    // slot; else bitmaps + ext slots together in shared memory (SMEM) or in the global slot
    char* sbase = (SMEM && !QREG) ? dyn_smem : g.gstate + (size_t)blockIdx.x * g.slot_bytes;
    const int capL0 = QREG ? 0 : (g.qcap + 31) / 32, capL1 = (capL0 + 31) / 32;
    uint32_t* L0 = reinterpret_cast<uint32_t*>(sbase);
    uint32_t* L1 = reinterpret_cast<uint32_t*>(sbase + align_up((size_t)capL0 * 4, 16));
    char* ebase = (QREG || !g.ext_global) ? reinterpret_cast<char*>(L1) + align_up((size_t)capL1 * 4, 16)
                                          : g.gstate + (size_t)blockIdx.x * g.slot_bytes;
    const size_t estride = align_up((size_t)g.ecap * 4, 16);
    int32_t* ef = reinterpret_cast<int32_t*>(ebase);
    uint32_t* eB = reinterpret_cast<uint32_t*>(ebase + estride);
    uint32_t* ec = reinterpret_cast<uint32_t*>(ebase + 2 * estride);
    int2* qrec = reinterpret_cast<int2*>(dyn_smem);                                   // QREG only (REC4: one packed word per rank)
    uint32_t* qrec4 = reinterpret_cast<uint32_t*>(dyn_smem);
    // QREG: the shared-memory window address of dyn_smem, held in ONE register (opaque to the compiler,
    // which otherwise re-derives it from SR_CgaCtaId inside the hot loop)
    uint32_t sm32 = 0;
    if constexpr (QREG) {
        sm32 = (uint32_t)__cvta_generic_to_shared(dyn_smem);
        asm volatile("" : "+r"(sm32));
    }
    const int Mi = (int)g.M;
    const int64_t n_items = g.I * g.n_policies;
    const uint32_t one = g.n_policies > 0 ? 1u : 0u;      // 1, but not to the compiler (SVF_ACC_GE)
    (void)one;

    while (true) {
        if (tid == 0) inst_s = (long long)atomicAdd(g.work_ctr, 1ull);
        __syncthreads();
        const int64_t item = inst_s;
        __syncthreads();
        if (item >= n_items) break;
        const int pi = (int)(item / g.I);            // policy-major
        const int64_t j = item - (int64_t)pi * g.I;

        const PolicyIO& io = g.io[pi];
        const int policy = io.policy;
        const bool want_start = io.start != nullptr, want_finish = io.finish != nullptr, want_p99 = io.p99 != nullptr;
        const int64_t base = g.off[j];
        const int64_t n64 = g.off[j + 1] - base;
        uint32_t flags = 0;
        if (n64 < 0 || n64 > g.max_instance || base < 0 || base + (n64 > 0 ? n64 : 0) > g.N ||
            g.off[0] != 0 || g.off[g.I] != g.N || (QREG && n64 > QRANKS) || *g.layout_bad)
            flags |= F_LAYOUT;
        const int n = (flags & F_LAYOUT) ? 0 : (int)n64;
        const int32_t* __restrict__ a = g.a + base;
        const int32_t* __restrict__ s = g.s + base;
        const int32_t* __restrict__ o = g.o + base;

        // ---- validation (data errors -> status[j], never UB) --------------------------------
        int64_t sum_o = 0;
        int max_a = 0, max_s = 0, max_o = 0;
        // (unrolled: the loads of several rounds in flight; the loop is 4 % of the stall samples of the bench kernel)
#pragma unroll (LAT ? 8 : 4)
        for (int i = tid; i < n; i += THREADS) {
            const int32_t ai = a[i], si = s[i], oi = o[i];
            const int32_t ki = g.okey ? g.okey[base + i] : oi;      // length the key sees
            if (oi < 1 || si < 0 || ai < 0 || ki < 1) flags |= F_RANGE;
            if (i > 0 && ai < a[i - 1]) flags |= F_UNSORTED;
            if ((int64_t)si + oi > g.M) flags |= F_INFEASIBLE;
            const uint32_t b = policy == SVF_SVF_1BIT ? (uint32_t)g.bit[base + i] : 0u;
            if (oi >= 1 && si >= 0 && ai >= 0 && ki >= 1 && (priority_key(policy, si, ki, ai, b, g.O0, g.O1) >> 32)) flags |= F_OVERFLOW;
            sum_o += oi > 0 ? oi : 0;
            max_a = ai > max_a ? ai : max_a;
            if (REC4) { max_s = si > max_s ? si : max_s; max_o = oi > max_o ? oi : max_o; }
            // QREG: the (s, o) of every request by RANK in shared memory, once per instance (the presort
            // wrote a permutation of [0, n) whatever the data was), so that picking a head never waits
            // for global memory
            // (REC4: packed below, once the widths are known)
            if (QREG && !REC4) qrec[io.rank[base + i] & (QRANKS - 1)] = make_int2(si, oi);
        }
        flags = G::or_u32(flags, scratch, parity);
        sum_o = G::sum_i64(sum_o, scratch, parity);
        { int z = 0; G::sum_max(z, max_a, scratch, parity); }
        if ((int64_t)max_a + sum_o >= ((int64_t)1 << 31)) flags |= F_OVERFLOW;   // horizon
        const int32_t status = status_from_flags(flags);

        int64_t tel = 0;                 // per-lane partial sums (warp 0), reduced at the end
        int mk = 0, peak = 0;
        uint32_t rounds = 0, decisions = 0;
        long long cntE = 0, cntU = 0;
        unsigned long long cntV = 0, cntBk = 0;   // uniform: evaluations, blocked evaluations
        int64_t p99v = 0;

        if (status != SVF_OK || n == 0) {
            for (int i = tid; i < n; i += THREADS) {
                if (want_start) io.start[base + i] = -1;
                if (want_finish) io.finish[base + i] = -1;
            }
        } else {
            // REC4: (s, o) of a waiting request packed into ONE word, s in the low `pshift` bits -- the
            // widths are this instance's own (bits of its largest s and o); an instance whose widths
            // do not fit 32 bits together (pshift < 0) leaves the records in global memory instead
            int pshift = 0; uint32_t pmask = 0;
            if constexpr (REC4) {
                max_s = __reduce_max_sync(FULL, max_s); max_o = __reduce_max_sync(FULL, max_o);
                const int bs = 32 - __clz(max_s), bo = 32 - __clz(max_o);
                pshift = bs + bo <= 32 ? bs : -1;
                pmask = pshift >= 0 ? (uint32_t)((1ull << pshift) - 1ull) : 0u;
                if (pshift >= 0)
                    for (int i = tid; i < n; i += THREADS)
                        qrec4[io.rank[base + i] & (QRANKS - 1)] = (uint32_t)s[i] | ((uint32_t)o[i] << pshift);     // (pshift <= 31: s < 2^31)
            }
            auto lds_rec = [&](int r) -> int2 {
                int2 v;
                if constexpr (REC4) {
                    if (pshift >= 0) {
                        uint32_t x; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(x) : "r"(sm32 + (uint32_t)r * 4u));
                        v.x = (int)(x & pmask); v.y = (int)(x >> pshift);
                    } else {
                        int pi_ = pi; long long b_ = base;
                        asm volatile("" : "+r"(pi_), "+l"(b_));
                        const int id = (int)g.io[pi_].order[b_ + r];
                        v.x = g.s[b_ + id]; v.y = g.o[b_ + id];
                    }
                } else {
                    asm volatile("ld.shared.v2.s32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(sm32 + (uint32_t)r * 8u));
                }
                return v;
            };
            const uint32_t* __restrict__ rnk = io.rank + base;
            const uint32_t* __restrict__ ord = io.order + base;
            const int4* __restrict__ req = io.req + base;
            int32_t* __restrict__ out_start = io.start + base;
            int32_t* __restrict__ out_finish = io.finish + base;
            uint32_t* out_lat = io.lat + base;
            const int nL0 = (n + 31) / 32, nL1 = (nL0 + 31) / 32;
            // QREG: bitmap word w of this lane covers the ranks [32 (32 w + lane), + 32); the registers are the truth
            uint32_t qword[QW];
#pragma unroll
            for (int w = 0; w < QW; ++w) qword[w] = 0;
            // lowest waiting rank (INT_MAX if none), the rest of its word above it, the word's first rank
            auto queue_head = [&](uint32_t& rest, int& wbase_, uint32_t& bit_) -> int {
                if constexpr (ILV) {        // (an empty lane offers (0 - 1) << 5 | lane, above every rank as unsigned)
                    const uint32_t key = __reduce_min_sync(FULL, ((uint32_t)(__ffs(qword[0]) - 1) << 5) | (uint32_t)lane);
                    return (int)key < 0 ? INT_MAX : (int)key;
                }
#pragma unroll
                for (int w = 0; w < QW; ++w) {
                    const uint32_t nz = __ballot_sync(FULL, qword[w] != 0u);
                    if (nz) {
                        const int l0 = __ffs(nz) - 1;
                        const uint32_t w0 = __shfl_sync(FULL, qword[w], l0);
                        wbase_ = (w * 32 + l0) * 32;
                        bit_ = w0 & (0u - w0);
                        rest = w0 ^ bit_;
                        return wbase_ + (31 - __clz(bit_));
                    }
                }
                return INT_MAX;
            };
            if (!QREG) {
                for (int i = tid; i < nL0; i += THREADS) L0[i] = 0;
                for (int i = tid; i < nL1; i += THREADS) L1[i] = 0;
            }

            int f[K]; uint32_t B[K], c[K];
#pragma unroll
            for (int k = 0; k < K; ++k) { f[k] = 0; B[k] = 0; c[k] = 0; }

            // arrival window: lane l holds request wb + l
            int wb = 0, aw, sw = 0, ow = 0, rw;
            // QREG (96 registers, none to spare): the rarely taken path (window refill every 32 arrivals)
            // re-derives its pointers from (policy index, base) behind an opaque copy, so that no 64-bit
            // pointer stays live across the hot loop
            auto load_window = [&]() {
                const int idx = wb + lane;
                const bool in = idx < n;
                if (QREG) {
                    int pi_ = pi; long long b_ = base;
                    asm volatile("" : "+r"(pi_), "+l"(b_));
                    aw = in ? g.a[b_ + idx] : INT_MAX;
                    rw = in ? (int)g.io[pi_].rank[b_ + idx] : INT_MAX;
                } else {
                    aw = in ? a[idx] : INT_MAX;
                    sw = in ? s[idx] : 0; ow = in ? o[idx] : 0;
                    rw = in ? (int)rnk[idx] : INT_MAX;
                }
            };
            load_window();
            auto win_rec = [&](int l, int r) {
                Rec x; x.r = r; x.s = __shfl_sync(FULL, sw, l); x.o = __shfl_sync(FULL, ow, l);
                x.a = __shfl_sync(FULL, aw, l); x.id = wb + l; return x;
            };
            // non-QREG output buffer: admission number m sits in lane m % 32 of warp 0 until 32 are there
            // (QREG: the start time waits at the request's rank in shared memory until the instance ends)
            int b_id = 0, b_t = 0, b_f = 0, b_lat = 0;
            auto flush = [&](int count) {
                if (!QREG && wrp == 0 && lane < count) {
                    const int id = b_id, lat = b_lat;
                    if (want_start) out_start[id] = b_t;
                    if (want_finish) out_finish[id] = b_f;
                    if (want_p99) out_lat[id] = (uint32_t)lat;
                    tel += lat;
                    mk = b_f > mk ? b_f : mk;
                }
            };
            G::sync();

            Rec head, second;
            // non-QREG: the record of `second` is prefetched by an ASYNCHRONOUS copy into a 16-byte slot of
            // shared memory per warp (cp.async: no register, no scoreboard) and read at the next promotion,
            // one evaluation later; sec_pend: the record of `second` is in that slot, not in registers.
            // (Prefetched into registers, ptxas settles the load's scoreboard at the loop header: the warp
            // waited there for the L2 round trip, 11 % of the stall samples of configs[3].)
            bool sec_pend = false;
            int pre_par = 0;
            head.r = INT_MAX; head.s = head.o = head.id = head.a = 0;
            second = head;
            int next = 0, started = 0, hw = 0;
            uint32_t hrest = 0, hbit = 0; int hbase = 0;    // QREG: the head's bitmap word above the head, the head's own bit in it (one-hot), the word's first rank
            int32_t t = a[0];
            int32_t t_lb = t;                     // first step at which the head must be (re)evaluated

            while (started < n) {
                // 2. ARRIVE (1. COMPLETE is implicit: a slot is dead once f <= t)
                bool arrived = false;
                int rmin = INT_MAX;                  // ILV: lowest rank among this step's arrivals
                while (next < n) {
                    if (next >= wb + 32) { wb = next; load_window(); }
                    const int idx = wb + lane;
                    const bool v = idx >= next && aw <= t;
                    const uint32_t m = __ballot_sync(FULL, v);
                    if (!m) break;
                    if (QREG) {
                        // the arrivals of a step set their bits in a shared-memory copy of the bitmap
                        if (!arrived) {
#pragma unroll
                            for (int w = 0; w < QW; ++w)
                                asm volatile("st.shared.u32 [%0], %1;" :: "r"(sm32 + (uint32_t)OFF_BITS + (uint32_t)(w * 32 + lane) * 4u), "r"(qword[w]) : "memory");
                            __syncwarp();
                        }
                        if (ILV) { const int rm = __reduce_min_sync(FULL, v ? rw : INT_MAX); rmin = rm < rmin ? rm : rmin; }
                        if (v) asm volatile("red.shared.or.b32 [%0], %1;" :: "r"(sm32 + (uint32_t)OFF_BITS + (uint32_t)(ILV ? (rw & 31) : (rw >> 5)) * 4u), "r"(1u << (ILV ? (rw >> 5) : (rw & 31))) : "memory");
                    } else {
                        // nobody may still be reading the bitmap for the previous step
                        if (!arrived) G::sync();
                        if (wrp == 0 && v) queue_set(L0, L1, rw);
                        const int r1 = __reduce_min_sync(FULL, v ? rw : INT_MAX);
                        if (r1 < second.r) {
                            const int l1 = __ffs(__ballot_sync(FULL, v && rw == r1)) - 1;
                            if (r1 < head.r) {
                                const int r2 = __reduce_min_sync(FULL, (v && lane != l1) ? rw : INT_MAX);
                                const Rec n1 = win_rec(l1, r1);
                                if (r2 < head.r) {
                                    const int l2 = __ffs(__ballot_sync(FULL, v && lane != l1 && rw == r2)) - 1;
                                    second = win_rec(l2, r2);
                                } else {
                                    second = head;
                                }
                                sec_pend = false;
                                head = n1;
                                t_lb = t;                 // a new head: evaluate it now
                            } else {
                                second = win_rec(l1, r1);
                                sec_pend = false;
                            }
                        }
                    }
                    arrived = true;
                    next += __popc(m);
                    if (next < wb + 32) break;
                }
                if (arrived) {
                    if (QREG) {
                        // reload the bitmap word; the head is its lowest set bit (arrivals set bits)
                        __syncwarp();
#pragma unroll
                        for (int w = 0; w < QW; ++w)
                            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(qword[w]) : "r"(sm32 + (uint32_t)OFF_BITS + (uint32_t)(w * 32 + lane) * 4u) : "memory");
                        // (ILV: the head after the arrivals is the lower of the old head and the lowest arriving rank:
                        // known before the bitmap has made its round trip through shared memory)
                        const int r0 = ILV ? (rmin < head.r ? rmin : head.r) : queue_head(hrest, hbase, hbit);      // (arrivals set bits: the queue is not empty)
                        if (r0 != head.r) {
                            const int2 v = lds_rec(r0);
                            head.r = r0; head.s = v.x; head.o = v.y;
                            t_lb = t;                     // a new head: evaluate it now
                        }
                    } else if (THREADS == 32) {
                        __syncwarp();
                    }
                }

                // 3. ADMIT
                if (head.r != INT_MAX) {
                    rounds += 1;
                    while (t >= t_lb) {
                        // ---- evaluation pass (with the update applied speculatively) -------------
                        const int fh = t + head.o;
                        const uint32_t t1 = (uint32_t)t + 1u, oh = (uint32_t)head.o, fhu = (uint32_t)fh;
                        const uint32_t Kc = (uint32_t)head.s - (uint32_t)t - (uint32_t)Mi;   // s_h - t - M (mod 2^32)
                        const uint32_t add = (uint32_t)head.s - (uint32_t)t;                  // A_j += s_h - t + f_j
                        uint32_t acc = 0, acc1 = 0, dm = 0;
                        int viol = INT_MIN;
                        // groups of four register slots processed per thread: 2 (eight slots), 4 (sixteen) or 8
                        // (thirty-two); slots past the high-water mark are dead (f = 0) and cost their instructions only
                        const int g4 = (K == 32 && hw > 16 * THREADS) ? 8 : (hw > 8 * THREADS ? 4 : 2);
                        const bool use_ext = hw > REGCAP;
                        SVF_SLOTS(g4, SVF_EVAL)
                        // lowest free register slot of this thread as a one-hot bit (bit k of dm =
                        // slot k is dead); the group takes the lowest (slot, thread) pair
                        // (a sentinel bit marks the first slot past the groups in use; slot 16 = none)
                        int fkey;
                        if constexpr (K == 32) {      // 32 slots: the key carries the slot NUMBER (32 = none)
                            const uint32_t dmx = dm | (g4 < 8 ? (1u << (4 * g4)) : 0u);
                            fkey = ((dmx ? __ffs(dmx) - 1 : K) << TSHIFT) | tid;
                        } else {       // (the sentinel keeps dmx non-zero; slot 16 = none)
                            const uint32_t dmx = dm | (1u << (4 * g4));
                            fkey = ((__ffs(dmx) - 1) << TSHIFT) | tid;
                        }
                        int eidx = INT_MAX;
                        if (use_ext) {
                            int elive = REGCAP - 1;             // highest live ext slot of this thread
                            for (int q = REGCAP + tid; q < hw; q += THREADS) {
                                const int e = q - REGCAP;
                                const int fk = ef[e];
                                const uint32_t x = (uint32_t)fk - t1;
                                if (fk >= fh) acc += ec[e] + fhu;
                                if (x < oh) {
                                    viol = __viaddmax_s32((int)eB[e], (int)Kc, viol);
                                    eB[e] += add + (uint32_t)fk;
                                    if (COUNT) cntU += 1;
                                }
                                if (x >> 31) eidx = eidx < q ? eidx : q; else elive = q;
                                if (COUNT) cntE += (long long)((x >> 31) ^ 1u);
                            }
                            // the mark comes back down to the highest live ext slot: once the running set fits the
                            // registers again, the passes stop walking dead ext slots in global memory (configs[3]
                            // under 1-bit SVF peaks at 2,355 running requests for a sixth of its admissions)
                            uint32_t z = 0; int emn = 0;
                            reduce_add_max_min<THREADS>(z, elive, emn, red, rparity);
                            hw = elive + 1;
                        }
                        acc += acc1;
                        reduce_add_max_min<THREADS>(acc, viol, fkey, red, rparity);
                        if (COUNT) ++cntV;
                        const int Ah = head.s + head.o + (int)acc;        // exact: 0 <= A_h <= 2M < 2^31
                        if (viol > 0 || Ah > Mi) {
                            // ---- blocked (no bypass): take the update back and find how
                            // long the head stays blocked at least --------------------------------
                            int wmax = 0, minge = INT_MAX;
                            if (COUNT) ++cntBk;
                            if (Ah > Mi) { SVF_SLOTS(g4, SVF_BLOCK) } else { SVF_SLOTS(g4, SVF_BLOCK2) }
                            if (use_ext) {
                                for (int q = REGCAP + tid; q < hw; q += THREADS) {
                                    const int e = q - REGCAP;
                                    const int fk = ef[e];
                                    const uint32_t x = (uint32_t)fk - t1;
                                    if (x < oh) {
                                        eB[e] -= add + (uint32_t)fk;
                                        const int v = (int)(eB[e] + Kc), d = (int)x + 1;
                                        const int w = v < d ? v : d;
                                        wmax = w > wmax ? w : wmax;
                                        if (COUNT) cntU -= 1;
                                    }
                                    if (fk >= fh) minge = fk < minge ? fk : minge;
                                }
                            }
                            uint32_t z = 0;
                            reduce_add_max_min<THREADS>(z, wmax, minge, red, rparity);
                            int lb = t + (wmax > 1 ? wmax : 1);
                            if (Ah > Mi) { const int l1 = minge - head.o + 1; lb = l1 > lb ? l1 : lb; }
                            t_lb = lb;
                            break;
                        }

                        // ---- admitted: the update is already in place; write the head into a slot --
                        const uint32_t Bh = (uint32_t)Ah + fhu;
                        int idx;
                        if (fkey < (K << TSHIFT)) {
                            const int ik = fkey >> TSHIFT;           // uniform
                            const bool mine = (fkey & (THREADS - 1)) == tid;
                            idx = (ik << TSHIFT) + (fkey & (THREADS - 1));
                            SVF_PUTK(ik, SVF_PUT)
                        } else {
                            // every register slot is live: the lowest dead ext slot, else a new one
                            if (use_ext) {
                                uint32_t z = 0; int zmax = 0;
                                reduce_add_max_min<THREADS>(z, zmax, eidx, red, rparity);
                            }
                            idx = eidx == INT_MAX ? hw : eidx;
                            if (((idx - REGCAP) & (THREADS - 1)) == tid) {
                                const int e = idx - REGCAP;
                                ef[e] = fh; eB[e] = Bh; ec[e] = add;
                            }
                        }
                        hw = idx + 1 > hw ? idx + 1 : hw;
                        {   // every final A_j is a mem(f_j): the new A_h and the raised in-range A_j
                            const int pj = Mi + viol;                  // INT_MIN + M: no in-range slot
                            const int p2 = Ah > pj ? Ah : pj;
                            peak = p2 > peak ? p2 : peak;
                        }
                        if (QREG) {
                            if constexpr (ILV) {
                                if (lane == (head.r & 31)) qword[0] &= ~(1u << (head.r >> 5));
                            } else if constexpr (QW <= 2) {
#pragma unroll
                                for (int w = 0; w < QW; ++w)      // the head's bit (a uniform one-hot word) leaves its lane's word
                                    if (w * 32 + lane == (hbase >> 5)) qword[w] ^= hbit;
                            } else {          // many words: one mask, applied to the head's word only
                                const int wi = head.r >> 10;
                                const uint32_t m = lane == ((head.r >> 5) & 31) ? ~(1u << (head.r & 31)) : ~0u;
#pragma unroll
                                for (int w = 0; w < QW; ++w) if (w == wi) qword[w] &= m;
                            }
// the start time takes the place of the admitted request's record (its s is not needed again):
                            // outputs leave the chip at the end of the instance, in index order
                            asm volatile("st.shared.u32 [%0], %1;" :: "r"(sm32 + (uint32_t)head.r * (uint32_t)RB), "r"(t) : "memory");
                        } else {
                            if (tid == 0) queue_clear(L0, L1, head.r);
                            if (lane == (started & 31)) { b_id = head.id; b_t = t; b_f = fh; b_lat = fh - head.a; }
                        }
                        ++started;                                     // (decisions: the admissions are added at the end)
                        if (!QREG && (started & 31) == 0) flush(32);
                        if (QREG) {
                            // next head: the next set bit of the word the head came from (a uniform copy
                            // of it, `hrest`), else the lowest set bit of the later words; its (s, o) come
                            // from shared memory
                            int r;
                            if (!ILV && hrest) {
                                hbit = hrest & (0u - hrest);
                                hrest ^= hbit;
                                r = hbase + (31 - __clz(hbit));
                            } else {
                                r = queue_head(hrest, hbase, hbit);
                                if (r == INT_MAX) { head.r = INT_MAX; break; }
                            }
                            const int2 v = lds_rec(r);
                            head.r = r; head.s = v.x; head.o = v.y;
                        } else {
                            // promote the second; fetch the record behind it one admission ahead
                            head = second;
                            if (sec_pend) {
                                asm volatile("cp.async.wait_all;" ::: "memory");
                                __syncwarp();
                                const int4 qv = pre_s[pre_par][wrp];
                                head.s = qv.x; head.o = qv.y; head.id = qv.z; head.a = qv.w;
                            }
                            second.r = INT_MAX;
                            if (head.r == INT_MAX) break;
                            const int r = queue_first_ge(L0, L1, n, nL1, head.r + 1);
                            if (r != INT_MAX) {
                                second.r = r;
                                sec_pend = true;
                                pre_par ^= 1;                 // (the slot just read is not overwritten while a lane may still read it)
                                if (lane == 0)
                                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"((uint32_t)__cvta_generic_to_shared(&pre_s[pre_par][wrp])), "l"(req + r) : "memory");
                            }
                        }
                    }
                    if (head.r != INT_MAX) ++decisions;          // one blocked-head evaluation (R16)
                }
                if (started == n) break;
                // 4. ADVANCE to the next step at which anything can change (exact, R16)
                int tn = INT_MAX;
                if (next < n) {
                    if (next >= wb + 32) { wb = next; load_window(); }
                    tn = __shfl_sync(FULL, aw, next - wb);
                }
                if (head.r != INT_MAX) {                      // blocked head waits
                    tn = t_lb < tn ? t_lb : tn;
                    rounds += (uint32_t)(tn - t - 1);
                    decisions += (uint32_t)(tn - t - 1);
                }
                if (tn == INT_MAX) break;                     // nothing left that could ever happen (corrupt rank[]): never spin
                t = tn;
            }
            if (!QREG) flush(started & 31);
            if (QREG) {
                // outputs of the whole instance in INDEX order (coalesced loads of rank / a / o, coalesced
                // stores): the start time of request i waits at its rank in shared memory
                __syncwarp();
#pragma unroll 4
                for (int i = lane; i < n; i += 32) {
                    const int r = (int)rnk[i] & (QRANKS - 1);
                    int st, oo;
                    if (REC4) { st = (int)qrec4[r]; oo = o[i]; } else { const int2 v = qrec[r]; st = v.x; oo = v.y; }
                    const int fin = st + oo, lat = fin - a[i];
                    if (want_start) out_start[i] = st;
                    if (want_finish) out_finish[i] = fin;
                    if (want_p99) out_lat[i] = (uint32_t)lat;
                    tel += lat;
                    mk = fin > mk ? fin : mk;
                }
            }
            decisions += (uint32_t)started;
            if (want_p99) {                       // nearest rank ceil(0.99 n), 1-based (R13)
                G::sync();
                p99v = (int64_t)group_select_kth<THREADS>(out_lat, n, (int)((99ll * n + 99) / 100), hist, scratch, parity);
            }
        }
        if (COUNT) {
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) { cntE += __shfl_xor_sync(FULL, cntE, d); cntU += __shfl_xor_sync(FULL, cntU, d); }
            if (lane == 0 && g.work_counts) {
                atomicAdd(&g.work_counts[0], (unsigned long long)cntE);
                atomicAdd(&g.work_counts[1], (unsigned long long)cntU);
                if (wrp == 0) { atomicAdd(&g.work_counts[2], cntV); atomicAdd(&g.work_counts[3], cntBk); }
            }
        }
        if (wrp == 0) {
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) tel += __shfl_xor_sync(FULL, tel, d);
            mk = __reduce_max_sync(FULL, mk);
        }
        if (tid == 0) {
            if (io.tel) io.tel[j] = tel;
            if (io.peak) io.peak[j] = (int64_t)peak;
            if (io.p99) io.p99[j] = p99v;
            if (io.rounds) io.rounds[j] = (int64_t)rounds;
            if (io.decisions) io.decisions[j] = (int64_t)decisions;
            if (io.makespan) io.makespan[j] = mk;
            if (io.status) io.status[j] = status;
        }
        G::sync();
    }
}

}  // namespace svf
