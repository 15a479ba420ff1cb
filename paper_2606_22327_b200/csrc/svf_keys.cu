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
struct int8v { int v[8]; };
__device__ __forceinline__ int8v ld_stream8(const int32_t* p)      // one 256-bit load (sm_100: LDG.256)
{
    int8v r;
    asm volatile("ld.global.nc.L1::no_allocate.v8.s32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r.v[0]), "=r"(r.v[1]), "=r"(r.v[2]), "=r"(r.v[3]), "=r"(r.v[4]), "=r"(r.v[5]), "=r"(r.v[6]), "=r"(r.v[7]) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream(ulonglong2* p, uint64_t a, uint64_t b)
{
    asm volatile("st.global.L1::no_allocate.v2.u64 [%0], {%1,%2};" ::"l"(p), "l"(a), "l"(b) : "memory");
}
// one 256-bit store (sm_100: STG.256): a thread's four words cover a whole 32-byte sector, where two
// 128-bit stores each wrote half of every sector of the warp's range (the kernel is write bound)
__device__ __forceinline__ void st_stream4(uint64_t* p, uint64_t a, uint64_t b, uint64_t c, uint64_t d)
{
    asm volatile("st.global.L1::no_allocate.v4.u64 [%0], {%1,%2,%3,%4};" ::"l"(p), "l"(a), "l"(b), "l"(c), "l"(d) : "memory");
}

template <int POLICY, int VEC>      // VEC: 0 element by element, 1 128-bit accesses, 2 256-bit accesses
__global__ void __launch_bounds__(256) k_keys(int64_t n, const int32_t* __restrict__ s,
                                              const int32_t* __restrict__ o,
                                              const int32_t* __restrict__ a,
                                              const uint8_t* __restrict__ bit, int32_t O0, int32_t O1,
                                              uint64_t* __restrict__ words, int32_t* __restrict__ status)
{
    bool overflow = false;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (VEC == 2) {
        // eight requests per thread and iteration: 256-bit loads of s, o (a), eight bit bytes in one 64-bit
        // load, two 256-bit stores (a whole 32-byte sector each); two such groups in flight per thread
        const int64_t n8 = n >> 3;
        for (int64_t q0 = gid; q0 < n8; q0 += 2 * stride) {
            int8v vs[2], vo[2], va[2];
            uint64_t vb[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int64_t q = q0 + u * stride;
                vb[u] = 0;
#pragma unroll
                for (int e = 0; e < 8; ++e) { vs[u].v[e] = 0; vo[u].v[e] = 0; va[u].v[e] = 0; }
                if (q < n8) {
                    if (POLICY == SVF_SVF || POLICY == SVF_SVF_1BIT) vs[u] = ld_stream8(s + (q << 3));
                    if (POLICY == SVF_SVF || POLICY == SVF_SJF) vo[u] = ld_stream8(o + (q << 3));
                    if (POLICY == SVF_FCFS) va[u] = ld_stream8(a + (q << 3));
                    if (POLICY == SVF_SVF_1BIT) vb[u] = __ldg(reinterpret_cast<const unsigned long long*>(bit) + q);
                }
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int64_t q = q0 + u * stride;
                if (q >= n8) break;
                const uint64_t i0 = (uint64_t)q << 3;
                uint64_t w[8];
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const uint64_t k = priority_key(POLICY, vs[u].v[e], vo[u].v[e], va[u].v[e], (uint32_t)(vb[u] >> (8 * e)) & 0xffu, O0, O1);
                    overflow |= (k >> 32) != 0;
                    w[e] = (k << 32) + (i0 + e);
                }
                st_stream4(words + i0, w[0], w[1], w[2], w[3]);
                st_stream4(words + i0 + 4, w[4], w[5], w[6], w[7]);
            }
        }
        // ragged tail (< 8 requests)
        const int64_t i = (n8 << 3) + gid;
        if (i < n) {
            uint64_t k = priority_key(POLICY, s ? s[i] : 0, o ? o[i] : 0, a ? a[i] : 0, bit ? bit[i] : 0u, O0, O1);
            overflow |= (k >> 32) != 0;
            words[i] = (k << 32) + (uint64_t)i;
        }
    } else if (VEC == 1) {
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
void launch_policy(int vec, unsigned blocks, cudaStream_t st, int64_t n, const int32_t* s,
                   const int32_t* o, const int32_t* a, const uint8_t* bit, int32_t O0, int32_t O1,
                   uint64_t* words, int32_t* status)
{
    if (vec == 2)      k_keys<POLICY, 2><<<blocks, 256, 0, st>>>(n, s, o, a, bit, O0, O1, words, status);
    else if (vec == 1) k_keys<POLICY, 1><<<blocks, 256, 0, st>>>(n, s, o, a, bit, O0, O1, words, status);
    else               k_keys<POLICY, 0><<<blocks, 256, 0, st>>>(n, s, o, a, bit, O0, O1, words, status);
}

inline bool aligned_to(const void* p, uintptr_t a) { return p == nullptr || (reinterpret_cast<uintptr_t>(p) & (a - 1)) == 0; }

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
    // 256-bit accesses when every array allows it (torch allocations do), 128-bit, or element by element
    int vec = 0, per_thread = 1;
    if (aligned_to(s, 32) && aligned_to(o, 32) && aligned_to(a, 32) && aligned_to(words, 32) && aligned_to(bit, 8)) { vec = 2; per_thread = 8; }
    else if (aligned_to(s, 16) && aligned_to(o, 16) && aligned_to(a, 16) && aligned_to(words, 16) && aligned_to(bit, 4)) { vec = 1; per_thread = 4; }
    // a grid of whole waves (8 CTAs of 256 threads per SM)
    int64_t blocks = ceil_div(ceil_div(n, per_thread), 256);
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
