// a1 + a2: priority keys and packed words, one streaming pass (HBM-bound, sm_100a).
//   word_i = (key_i << 32) + i,   key by Eq. 1 / Eq. 2 / o_i / a_i
// 128-bit loads of s, o (and a for FCFS, 32-bit loads of four bit bytes for 1-bit SVF), two
// 128-bit stores per four requests, no shared memory (no reuse), L1 bypassed on the streams.
#include "svf_internal.cuh"

namespace svf {

namespace {

__device__ __forceinline__ int4 ld_stream(const int4* p)
{
    int4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.s32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream(ulonglong2* p, uint64_t a, uint64_t b)
{
    asm volatile("st.global.L1::no_allocate.v2.u64 [%0], {%1,%2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}

template <int POLICY, bool VEC>
__global__ void __launch_bounds__(256) k_keys(int64_t n, const int32_t* __restrict__ s,
                                              const int32_t* __restrict__ o,
                                              const int32_t* __restrict__ a,
                                              const uint8_t* __restrict__ bit, int32_t O0, int32_t O1,
                                              uint64_t* __restrict__ words, int32_t* __restrict__ status)
{
    bool overflow = false;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (VEC) {
        const int64_t n4 = n >> 2;
        // two groups of four requests per thread and iteration: eight independent 128-bit loads in
        // flight before the first store
        for (int64_t q0 = gid; q0 < n4; q0 += 2 * stride) {
            int4 vs[2], vo[2], va[2];
            uint32_t vb[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int64_t q = q0 + u * stride;
                vs[u] = vo[u] = va[u] = make_int4(0, 0, 0, 0); vb[u] = 0;
                if (q < n4) {
                    if (POLICY == SVF_SVF || POLICY == SVF_SVF_1BIT) vs[u] = ld_stream(reinterpret_cast<const int4*>(s) + q);
                    if (POLICY == SVF_SVF || POLICY == SVF_SJF) vo[u] = ld_stream(reinterpret_cast<const int4*>(o) + q);
                    if (POLICY == SVF_FCFS) va[u] = ld_stream(reinterpret_cast<const int4*>(a) + q);
                    if (POLICY == SVF_SVF_1BIT) vb[u] = __ldg(reinterpret_cast<const uint32_t*>(bit) + q);
                }
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int64_t q = q0 + u * stride;
                if (q >= n4) break;
                const uint64_t i0 = (uint64_t)q << 2;
                uint64_t k0 = priority_key(POLICY, vs[u].x, vo[u].x, va[u].x, vb[u] & 0xffu, O0, O1);
                uint64_t k1 = priority_key(POLICY, vs[u].y, vo[u].y, va[u].y, (vb[u] >> 8) & 0xffu, O0, O1);
                uint64_t k2 = priority_key(POLICY, vs[u].z, vo[u].z, va[u].z, (vb[u] >> 16) & 0xffu, O0, O1);
                uint64_t k3 = priority_key(POLICY, vs[u].w, vo[u].w, va[u].w, (vb[u] >> 24) & 0xffu, O0, O1);
                overflow |= ((k0 | k1 | k2 | k3) >> 32) != 0;
                ulonglong2* out = reinterpret_cast<ulonglong2*>(words + i0);
                st_stream(out, (k0 << 32) + i0, (k1 << 32) + (i0 + 1));
                st_stream(out + 1, (k2 << 32) + (i0 + 2), (k3 << 32) + (i0 + 3));
            }
        }
        // ragged tail (< 4 requests)
        const int64_t i = (n4 << 2) + gid;
        if (i < n) {
            uint64_t k = priority_key(POLICY, s ? s[i] : 0, o ? o[i] : 0, a ? a[i] : 0, bit ? bit[i] : 0u, O0, O1);
            overflow |= (k >> 32) != 0;
            words[i] = (k << 32) + (uint64_t)i;
        }
    } else {
        for (int64_t i = gid; i < n; i += stride) {
            uint64_t k = priority_key(POLICY, s ? s[i] : 0, o ? o[i] : 0, a ? a[i] : 0, bit ? bit[i] : 0u, O0, O1);
            overflow |= (k >> 32) != 0;
            words[i] = (k << 32) + (uint64_t)i;
        }
    }
    if (status && __any_sync(__activemask(), overflow) && overflow) atomicMax(status, (int32_t)SVF_EOVERFLOW);
}

template <int POLICY>
void launch_policy(bool vec, unsigned blocks, cudaStream_t st, int64_t n, const int32_t* s,
                   const int32_t* o, const int32_t* a, const uint8_t* bit, int32_t O0, int32_t O1,
                   uint64_t* words, int32_t* status)
{
    if (vec) k_keys<POLICY, true><<<blocks, 256, 0, st>>>(n, s, o, a, bit, O0, O1, words, status);
    else     k_keys<POLICY, false><<<blocks, 256, 0, st>>>(n, s, o, a, bit, O0, O1, words, status);
}

inline bool aligned16(const void* p) { return p == nullptr || (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace

int keys_launch(int policy, int64_t n, const int32_t* s, const int32_t* o, const int32_t* a,
                const uint8_t* bit, int32_t O0, int32_t O1, uint64_t* words, int32_t* status,
                cudaStream_t st, int64_t* launches)
{
    if (status) {
        cudaError_t e = cudaMemsetAsync(status, 0, sizeof(int32_t), st);
        if (e != cudaSuccess) return (int)e;
    }
    if (n <= 0) return 0;
    const bool vec = aligned16(s) && aligned16(o) && aligned16(a) && aligned16(words) &&
                     (bit == nullptr || (reinterpret_cast<uintptr_t>(bit) & 3u) == 0);
    // 4 requests per thread and iteration; a grid of whole waves (8 CTAs of 256 threads per SM)
    int64_t blocks = ceil_div(ceil_div(n, 4), 256);
    const int64_t cap = (int64_t)sm_count() * 8;
    if (blocks > cap) blocks = cap;
    switch (policy) {
    case SVF_SVF:      launch_policy<SVF_SVF>(vec, (unsigned)blocks, st, n, s, o, a, bit, O0, O1, words, status); break;
    case SVF_SVF_1BIT: launch_policy<SVF_SVF_1BIT>(vec, (unsigned)blocks, st, n, s, o, a, bit, O0, O1, words, status); break;
    case SVF_SJF:      launch_policy<SVF_SJF>(vec, (unsigned)blocks, st, n, s, o, a, bit, O0, O1, words, status); break;
    default:           launch_policy<SVF_FCFS>(vec, (unsigned)blocks, st, n, s, o, a, bit, O0, O1, words, status); break;
    }
    ++*launches;
    return (int)cudaGetLastError();
}

}  // namespace svf
