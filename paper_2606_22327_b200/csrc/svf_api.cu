// C-ABI entry points that are thin wrappers (svf_keys, svf_sort_words, strings, counters).
// svf_admit and svf_simulate live beside their kernels.
#include "svf_internal.cuh"

namespace svf {
int64_t sim_last_launches();
int64_t admit_last_launches();
namespace {
thread_local int64_t g_launches_keys = 0;
thread_local int64_t g_launches_sort = 0;

bool have_device()
{
    int c = 0;
    return cudaGetDeviceCount(&c) == cudaSuccess && c > 0;
}
}  // namespace
}  // namespace svf

using namespace svf;

extern "C" int svf_keys(int policy, int64_t n, const int32_t* s, const int32_t* o, const int32_t* a,
                        const uint8_t* bit, int32_t O0, int32_t O1, uint64_t* words_out,
                        int32_t* status_out, void* stream)
{
    g_launches_keys = 0;
    if (policy < 0 || policy > 3 || n < 0 || n > ((int64_t)1 << 32)) return SVF_EINVAL;
    if (policy == SVF_SVF_1BIT && (O0 < 1 || O1 < 1)) return SVF_EINVAL;
    if (n > 0) {
        if (!words_out) return SVF_EINVAL;
        if (policy == SVF_SVF_1BIT && !bit) return SVF_EINVAL;
        if ((policy == SVF_SVF || policy == SVF_SVF_1BIT) && !s) return SVF_EINVAL;
        if ((policy == SVF_SVF || policy == SVF_SJF) && !o) return SVF_EINVAL;
        if (policy == SVF_FCFS && !a) return SVF_EINVAL;
    }
    if (!have_device()) return SVF_ECUDA;
    int rc = keys_launch(policy, n, s, o, a, bit, O0, O1, words_out, status_out, (cudaStream_t)stream, &g_launches_keys);
    return rc == 0 ? SVF_OK : SVF_ECUDA;
}

extern "C" size_t svf_sort_workspace_bytes(int64_t n, int bit_lo, int bit_hi)
{
    if (n < 0 || bit_lo < 0 || bit_hi > 64 || bit_lo >= bit_hi) return 0;
    return align_up(sort_ws_bytes(n, bit_lo, bit_hi), 256) + align_up((size_t)n * 8, 256) + 256;
}

extern "C" int svf_sort_words(int64_t n, const uint64_t* words_in, uint64_t* words_out, int bit_lo,
                              int bit_hi, void* ws, size_t ws_bytes, void* stream)
{
    g_launches_sort = 0;
    if (n < 0 || n >= ((int64_t)1 << 30) || bit_lo < 0 || bit_hi > 64 || bit_lo >= bit_hi) return SVF_EINVAL;
    if (n > 0 && (!words_in || !words_out || words_in == words_out)) return SVF_EINVAL;
    if (!ws) return SVF_EWORKSPACE;
    char* base = (char*)align_up((size_t)(uintptr_t)ws, 256);
    const size_t need = svf_sort_workspace_bytes(n, bit_lo, bit_hi) - 256;
    if ((size_t)(base - (char*)ws) + need > ws_bytes) return SVF_EWORKSPACE;
    if (!have_device()) return SVF_ECUDA;
    SortWs w;
    sort_ws_carve(&w, base, n, bit_lo, bit_hi);
    uint64_t* tmp = (uint64_t*)(base + align_up(sort_ws_bytes(n, bit_lo, bit_hi), 256));
    cudaStream_t st = (cudaStream_t)stream;
    int rc = sort_u64(w, words_in, words_out, tmp, n, bit_lo, bit_hi, st, &g_launches_sort);
    if (rc) return SVF_ECUDA;
    rc = sort_result_to(w, words_out, n, st, &g_launches_sort);
    return rc == 0 ? SVF_OK : SVF_ECUDA;
}

extern "C" int64_t svf_last_launch_count(int which)
{
    switch (which) {
    case 0: return g_launches_keys;
    case 1: return admit_last_launches();
    case 2: return sim_last_launches();
    case 3: return g_launches_sort;
    default: return -1;
    }
}

extern "C" const char* svf_status_string(int status)
{
    switch (status) {
    case SVF_OK: return "ok";
    case SVF_EINVAL: return "invalid argument";
    case SVF_EWORKSPACE: return "workspace missing or too small";
    case SVF_ECUDA: return "CUDA error or no device";
    case SVF_ERANGE: return "request out of range (o < 1, s < 0, a < 0, rem < 1 or kv < 0)";
    case SVF_EUNSORTED: return "arrivals decrease inside an instance";
    case SVF_EINFEASIBLE: return "a request alone exceeds the budget (s + o > M)";
    case SVF_EOVERFLOW: return "key >= 2^32 or horizon >= 2^31";
    default: return "unknown status";
    }
}

extern "C" const char* svf_version(void) { return "svf-b200 0.1 (sm_100a)"; }
