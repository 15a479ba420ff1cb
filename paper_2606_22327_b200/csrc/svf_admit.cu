// a1-a5: one stateless admission decision (P:L358-366 engine loop; P:L507-524 order, no bypass,
// forward-looking check; P:L926 maxima at completion times).
//   keys (svf_keys.cu) -> onesweep sort of the packed words on the key bits [32, 64)
//   running set: words (2^32-1-rem, index) sorted the same way -> latest finish first
//   k_admit: one CTA builds (f_j, A_j) with a block scan (svf_state.cuh), then pops the sorted
//   queue while the check passes.
#include <limits.h>

#include "svf_internal.cuh"
#include "svf_state.cuh"

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

__global__ void __launch_bounds__(ADMIT_THREADS) k_admit(int64_t M, int32_t t, int64_t n_wait,
                                                         const int32_t* __restrict__ w_s,
                                                         const int32_t* __restrict__ w_o,
                                                         int64_t n_run, const int32_t* __restrict__ r_kv,
                                                         const int32_t* __restrict__ r_rem,
                                                         const SortPlan* __restrict__ wplan,
                                                         const SortPlan* __restrict__ rplan,
                                                         const AdmitFlags* __restrict__ fl,
                                                         int32_t* __restrict__ f, int64_t* __restrict__ A,
                                                         int64_t* __restrict__ n_admitted_out,
                                                         int32_t* __restrict__ admitted_idx_out,
                                                         int32_t* __restrict__ status_out)
{
    __shared__ int scratch[2][64];
    __shared__ int64_t warp_tot[ADMIT_THREADS / 32];
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
    const uint64_t* __restrict__ rsorted = rplan->result;
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

struct AdmitWs {
    SortWs wsort, rsort;
    uint64_t *w0, *w1, *r0, *r1;
    int32_t* f; int64_t* A;
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
    w->flags = (AdmitFlags*)(base + p); p += 256;
    w->total = p;
}

thread_local int64_t g_launches_admit = 0;

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
    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count < 1) return SVF_ECUDA;
    char* base = (char*)align_up((size_t)(uintptr_t)ws, 256);
    const size_t avail = ws_bytes - (size_t)(base - (char*)ws);
    AdmitWs w;
    admit_ws_layout(&w, base, n_wait, n_run);
    if (w.total > avail) return SVF_EWORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;

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
    // a3: the waiting queue in priority order; the running set by finish time
    rc = sort_u64(w.wsort, w.w0, w.w1, w.w0, n_wait, 32, 64, st, &g_launches_admit);
    if (rc) return SVF_ECUDA;
    rc = sort_u64(w.rsort, w.r0, w.r1, w.r0, n_run, 32, 64, st, &g_launches_admit);
    if (rc) return SVF_ECUDA;
    // a4 + a5
    k_admit<<<1, ADMIT_THREADS, 0, st>>>(M, t, n_wait, w_s, w_o, n_run, r_kv, r_rem, w.wsort.plan, w.rsort.plan,
                                         w.flags, w.f, w.A, n_admitted_out, admitted_idx_out, status_out);
    ++g_launches_admit;
    if (sorted_words_out) {
        rc = sort_result_to(w.wsort, sorted_words_out, n_wait, st, &g_launches_admit);
        if (rc) return SVF_ECUDA;
    }
    return cudaGetLastError() == cudaSuccess ? SVF_OK : SVF_ECUDA;
}
