// Internal declarations shared by the translation units of libsvf_b200 (CUDA path only; the CPU
// oracle under oracle/ includes nothing from here).
#pragma once

#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include "../../include/svf.h"

namespace svf {

// ---------------------------------------------------------------------------------------------
// small host/device helpers
// ---------------------------------------------------------------------------------------------
__host__ __device__ inline int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }
__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// bits needed to write every value in [0, count): 0 for count <= 1
inline int bits_for_count(int64_t count)
{
    int b = 0;
    while (b < 63 && ((int64_t)1 << b) < count) ++b;
    return b;
}

// Priority key (a1).  Eq. 1 v = s o + (o^2 + o)/2;  Eq. 2 the same with the
// class proxy O_m in place of o;  SJF o;  FCFS a.  Computed in unsigned 64 bit so that
// a key >= 2^32 is seen, not wrapped.  Inputs already known to be >= 0.
__device__ __forceinline__ uint64_t priority_key(int policy, int32_t s, int32_t o, int32_t a,
                                                 uint32_t bit, int32_t O0, int32_t O1)
{
    uint64_t us = (uint64_t)(uint32_t)s, uo = (uint64_t)(uint32_t)o;
    switch (policy) {
    case SVF_SVF:      return us * uo + ((uo * uo + uo) >> 1);
    case SVF_SVF_1BIT: { uint64_t m = (uint64_t)(uint32_t)(bit ? O1 : O0);
                         return us * m + ((m * m + m) >> 1); }
    case SVF_SJF:      return uo;
    default:           return (uint64_t)(uint32_t)a;
    }
}

// data-check bits accumulated per instance; status_from_flags picks the lowest-numbered code
enum : uint32_t { F_RANGE = 1u, F_UNSORTED = 2u, F_INFEASIBLE = 4u, F_OVERFLOW = 8u, F_LAYOUT = 16u };
__host__ __device__ inline int32_t status_from_flags(uint32_t f)
{
    if (f & F_LAYOUT) return SVF_EINVAL;
    if (f & F_RANGE) return SVF_ERANGE;
    if (f & F_UNSORTED) return SVF_EUNSORTED;
    if (f & F_INFEASIBLE) return SVF_EINFEASIBLE;
    if (f & F_OVERFLOW) return SVF_EOVERFLOW;
    return SVF_OK;
}

// ---------------------------------------------------------------------------------------------
// onesweep radix sort (svf_sort.cu)
// ---------------------------------------------------------------------------------------------
constexpr int SORT_MAX_PASSES = 8;
constexpr int SORT_RADIX_BITS = 8;
constexpr int SORT_RADIX = 256;
constexpr int SORT_THREADS = 256;
constexpr int SORT_IPT = 16;
constexpr int SORT_TILE = SORT_THREADS * SORT_IPT;   // 4096 words = 32 KB of shared memory

// Written by the plan kernel, read by every pass and by the consumers of the sorted words.
struct SortPlan {
    const uint64_t* src[SORT_MAX_PASSES];
    uint64_t*       dst[SORT_MAX_PASSES];
    int32_t         skip[SORT_MAX_PASSES];   // 1: this digit is the same in every word
    const uint64_t* result;                  // where the sorted words ended up
};

struct SortWs {
    SortPlan* plan;
    uint32_t* hist;       // [SORT_MAX_PASSES][256] counts, then exclusive bases
    uint32_t* tile_ctr;   // [SORT_MAX_PASSES] dynamic tile ids
    uint32_t* status;     // [passes][tiles][256] decoupled look-back words
    size_t    status_bytes;
};

inline int sort_num_passes(int bit_lo, int bit_hi) { return (bit_hi - bit_lo + SORT_RADIX_BITS - 1) / SORT_RADIX_BITS; }
size_t sort_ws_bytes(int64_t n, int bit_lo, int bit_hi);               // control + look-back only
void   sort_ws_carve(SortWs* w, void* base, int64_t n, int bit_lo, int bit_hi);
// Sort n words held at `in` on bits [bit_lo, bit_hi).  Passes go in -> x -> y -> x ...; y may
// alias in (then the input is overwritten).  The final location is plan->result (device side).
// Returns a cudaError_t as int; adds the number of launches to *launches.
int sort_u64(const SortWs& w, const uint64_t* in, uint64_t* x, uint64_t* y, int64_t n, int bit_lo,
             int bit_hi, cudaStream_t st, int64_t* launches);
// Segmented sort of small segments in shared memory (one CTA per instance, max_instance <=
// SEG_SORT_MAX): for every policy of the call it computes the priority keys from the trace and writes
// order[] (local id at instance offset + rank), rank[] (rank of instance offset + local id) and, if
// req != nullptr, the (s, o, id, a) records in priority order.  ONE launch for all policies.
constexpr int SEG_SORT_MAX = 4096;
constexpr int SEG_SORT_MAX_POLICIES = 8;
struct SegSortArgs {
    int64_t I, N;
    int cap;                         // filled in by seg_sort_keys
    const int64_t* off;
    const int32_t *s, *o, *okey /* key lengths or NULL */, *a;
    const uint8_t* bit;
    int32_t O0, O1;
    int n_policies;
    int policy[SEG_SORT_MAX_POLICIES];
    uint32_t* order[SEG_SORT_MAX_POLICIES];
    uint32_t* rank[SEG_SORT_MAX_POLICIES];
    int4* req[SEG_SORT_MAX_POLICIES];
};
int seg_sort_keys(const SegSortArgs& A, int64_t max_instance, cudaStream_t st, int64_t* launches);
// copy plan->result to out unless it already is out
int sort_result_to(const SortWs& w, uint64_t* out, int64_t n, cudaStream_t st, int64_t* launches);

// ---------------------------------------------------------------------------------------------
// entry-point implementations (one .cu each)
// ---------------------------------------------------------------------------------------------
int keys_launch(int policy, int64_t n, const int32_t* s, const int32_t* o, const int32_t* a,
                const uint8_t* bit, int32_t O0, int32_t O1, uint64_t* words, int32_t* status,
                cudaStream_t st, int64_t* launches);

int sm_count();   // SMs of the current device (asked every time; 148 without a device)
int profiling_mode();   // svf_set_profiling's switch of this host thread (svf_simulate.cu)

}  // namespace svf
