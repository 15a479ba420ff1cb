// svf_admit_static: the admission decision of svf_admit for a host that is not allowed to allocate.
//
// Who needs it.  svf_admit takes its scratch ("ws") from the caller, which is fine for a program
// that owns a device allocator.  A scheduler that lives INSIDE a serving engine often does not:
// the engine sizes its KV-cache pool at start-up to whatever HBM the weights left over, so a
// cudaMalloc made later from the step loop can fail outright, and even when it succeeds cudaMalloc
// and cudaFree serialise against the whole device and stall the decode stream the scheduler is
// supposed to feed.  The same holds for a plug-in whose host forbids device allocation outside
// its own pool, and for code that cannot reach an allocator at all (a C caller with nothing but
// the CUDA driver context it was handed).  For those callers the scratch lives in this library's
// own image: a file-scope __device__ array that the CUDA runtime places in the memory of every
// GPU that loads the library and keeps there until the process exits.
//
// What it costs and what it limits.  SVF_ADMIT_STATIC_BYTES (3 MiB) per GPU, always, used or not;
// in exchange a queue of up to SVF_ADMIT_STATIC_MAX_WAIT waiting and SVF_ADMIT_STATIC_MAX_RUN
// running requests.  One array per GPU means one decision at a time per GPU: see the header.
#include <mutex>

#include "svf_internal.cuh"

namespace {

// The scratch itself.  256-byte aligned because the workspace carving of svf_admit aligns every
// piece to 256 and expects the base to allow that without slack.
static __device__ __align__(256) unsigned char g_admit_scratch[SVF_ADMIT_STATIC_BYTES];

// In host code `g_admit_scratch` is only a handle by which the runtime knows the symbol; it is
// NOT the address the GPU sees (handing it to a kernel would fault, or quietly scribble over
// host memory on a system where the GPU can reach it).  The device address is asked for once
// per device, with that device current, and remembered here.
constexpr int MAX_DEVICES = 64;
std::mutex g_setup_mutex;
void* g_scratch_on_device[MAX_DEVICES];

int scratch_of_current_device(void** out)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) return SVF_ECUDA;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_on_device[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_admit_scratch) != cudaSuccess || !p) {
            cudaGetLastError();   // leave no sticky error behind for the caller's next CUDA call
            return SVF_ECUDA;
        }
        g_scratch_on_device[dev] = p;
    }
    *out = g_scratch_on_device[dev];
    return SVF_OK;
}

}  // namespace

extern "C" int svf_admit_static(int policy, int64_t M, int32_t t, int64_t n_wait, const int32_t* w_s,
                                const int32_t* w_o, const int32_t* w_a, const uint8_t* w_bit, int32_t O0,
                                int32_t O1, int64_t n_run, const int32_t* r_kv, const int32_t* r_rem,
                                int64_t* n_admitted_out, int32_t* admitted_idx_out,
                                uint64_t* sorted_words_out, int32_t* status_out, void* stream)
{
    // argument errors are reported as svf_admit reports them, before size and device are looked at
    if (policy < 0 || policy > 3 || n_wait < 0 || n_run < 0 || M < 0 || !n_admitted_out) return SVF_EINVAL;
    if (policy == SVF_SVF_1BIT && ((n_wait > 0 && !w_bit) || O0 < 1 || O1 < 1)) return SVF_EINVAL;
    if ((n_wait > 0 && (!w_s || !w_o || !w_a)) || (n_run > 0 && (!r_kv || !r_rem))) return SVF_EINVAL;
    // the stated limit first, then the byte count it was derived from (belt and braces: should the
    // workspace layout of svf_admit ever grow, the call is refused rather than overrunning the array)
    if (n_wait > SVF_ADMIT_STATIC_MAX_WAIT || n_run > SVF_ADMIT_STATIC_MAX_RUN) return SVF_EWORKSPACE;
    const size_t need = svf_admit_workspace_bytes(n_wait, n_run);
    if (need == 0 || need > (size_t)SVF_ADMIT_STATIC_BYTES) return SVF_EWORKSPACE;
    // the timing aid of svf_admit creates CUDA events, which allocates: not on this entry point
    if (svf::profiling_mode() != 0) return SVF_EINVAL;
    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count < 1) return SVF_ECUDA;
    void* scratch = nullptr;
    const int rc = scratch_of_current_device(&scratch);
    if (rc != SVF_OK) return rc;
    // From here on this is svf_admit with `scratch` as its workspace.  That call already treats the
    // workspace as uninitialised memory (flags, histograms and tile counters are cleared on the
    // stream before they are read), so what the previous decision left in the array does no harm.
    return svf_admit(policy, M, t, n_wait, w_s, w_o, w_a, w_bit, O0, O1, n_run, r_kv, r_rem, n_admitted_out,
                     admitted_idx_out, sorted_words_out, status_out, scratch, (size_t)SVF_ADMIT_STATIC_BYTES,
                     stream);
}
