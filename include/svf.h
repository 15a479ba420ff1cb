/*
 * include/svf.h -- C ABI of libsvf_b200: the data-parallel hot path of "Geometry-Aware Online
 * Scheduling for LLM Serving" (arxiv/paper_2606_22327), hand-written CUDA for sm_100a.
 *
 * Citations: "P:L<n>" = line n of the paper text; "R<k>" = reading k of DESIGN.md 3.
 *
 * The model (Eq. 3a-3d): discrete time, KV budget M, request i = (a_i, s_i, o_i) =
 * (arrival step, prompt tokens, output tokens).  Started at k_i >= a_i it holds s_i + (t - k_i)
 * tokens at every t in {k_i+1 .. k_i+o_i} (Eq. 3c), finishes at f_i = k_i + o_i with latency
 * f_i - a_i, is never preempted; sum of held tokens <= M at every t.
 * The policy: order the waiting queue by ascending key --
 * volume v_i = s_i o_i + (o_i^2 + o_i)/2 (Eq. 1), proxy volume s_i O_m + (O_m^2 + O_m)/2 with
 * m = bit_i (Eq. 2), o_i (SJF) or a_i (FCFS) -- ties broken by (arrival, id);
 * admit the head while the forward-looking check passes (no future time exceeds M with it
 * added); a blocked head is never bypassed.
 *
 * Conventions for every entry point
 *  - DEVICE pointers are marked [dev]; HOST pointers [host].  The caller owns every buffer; the
 *    library allocates no device memory and the compute calls keep no state between calls: they
 *    are re-entrant and may run concurrently on different streams (each with its own `ws`).  The
 *    only state the library holds is per HOST THREAD and belongs to the measurement aids at the
 *    end of this header (launch counters, the profiling switch and its CUDA events).
 *  - Scratch comes from the caller: `ws` [dev], at least the bytes the matching *_workspace_bytes
 *    call returns (that figure includes the slack for aligning `ws` up to 256 bytes).  A NULL or
 *    short `ws` is SVF_EWORKSPACE, found on the host before anything touches the device.
 *  - An array that would only be read for requests that do not exist may be NULL: with n = 0
 *    (n_wait = 0, n_requests = 0) every per-request pointer may be NULL, `bit` included, also
 *    under SVF_SVF_1BIT (O0, O1 >= 1 are still required there).
 *  - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls only
 *    enqueue work; outputs are valid once the stream has been synchronised.
 *  - Return value: svf_status_t for errors the HOST can see (arguments, sizes, CUDA launch
 *    errors).  Errors that depend on the DATA are found on the device and written to a status
 *    word ([dev], per instance for svf_simulate); they are never undefined behaviour and one
 *    instance's error does not disturb the others.
 *  - All arithmetic is integer and exact; there is no CPU fallback: without a CUDA device every
 *    compute call returns SVF_ECUDA.
 */
#ifndef SVF_H_
#define SVF_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Priority rule. */
typedef enum { SVF_SVF = 0, SVF_SVF_1BIT = 1, SVF_SJF = 2, SVF_FCFS = 3 } svf_policy_t;

typedef enum {
    SVF_OK = 0,
    SVF_EINVAL = 1,       /* host: null pointer, negative size, unknown policy, O0/O1 < 1, missing bit;
                             data (svf_simulate, svf_volume_lower_bound): `offsets` not non-decreasing
                             from 0 to N, or an instance larger than max_instance -- then every
                             instance of the call reports it and nothing is simulated              */
    SVF_EWORKSPACE = 2,   /* host: ws is NULL or ws_bytes too small                                   */
    SVF_ECUDA = 3,        /* host: no device / launch failed (cudaGetLastError != success)           */
    SVF_ERANGE = 16,      /* data: o_i < 1, s_i < 0, a_i < 0 or output_key_i < 1 (running set: rem < 1 or kv < 0) */
    SVF_EUNSORTED = 17,   /* data: arrivals decrease inside an instance                              */
    SVF_EINFEASIBLE = 18, /* data: s_i + o_i > M, could never be admitted (paper assumes <= aM) */
    SVF_EOVERFLOW = 19    /* data: key >= 2^32, or max a + sum o >= 2^31 (horizon bound)       */
} svf_status_t;
/* When several data checks fail in one instance the lowest-numbered code is reported. */

/* A batch of independent instances ("n requests ... global capacity M"), SoA, instances
 * concatenated.  Instance j is the index range [offsets[j], offsets[j+1]); inside it requests
 * are in (arrival, id) order, i.e. arrivals are non-decreasing and the local index is the id. */
typedef struct {
    int64_t        n_instances;   /* [host] I >= 0                                                  */
    int64_t        n_requests;    /* [host] N = offsets[I], 0 <= N < 2^30                           */
    int64_t        max_instance;  /* [host] max_j (offsets[j+1]-offsets[j]); sizes the on-chip state */
    const int64_t* offsets;       /* [dev] [I+1], offsets[0] = 0, non-decreasing                    */
    const int32_t* arrival;       /* [dev] [N] a_i >= 0                                             */
    const int32_t* prompt;        /* [dev] [N] s_i >= 0                                             */
    const int32_t* output;        /* [dev] [N] o_i >= 1 (true length: drives dynamics AND the check, R7) */
    const uint8_t* bit;           /* [dev] [N] 0 = short, 1 = long; may be NULL unless SVF_SVF_1BIT */
    int32_t        O0, O1;        /* [host] integer proxy lengths of Eq. 2 (>= 1 for SVF_SVF_1BIT)   */
    const int32_t* output_key;    /* [dev] [N] or NULL: PREDICTED output lengths (>= 1) that replace
                                     o_i in the SVF (Eq. 1) and SJF keys only -- the deployable
                                     SVF / SJF of the paper; NULL = true lengths =
                                     "Oracle-SVF / Oracle-SJF".  Dynamics and the check
                                     always use `output` (R7).                                      */
} svf_trace_t;

/* Caller-allocated DEVICE outputs of svf_simulate.  Any pointer may be NULL (not wanted). */
typedef struct {
    int32_t* start;          /* [dev] [N] k_i  (-1 for requests of a rejected instance)            */
    int32_t* finish;         /* [dev] [N] f_i = k_i + o_i (-1 likewise)                             */
    int64_t* total_latency;  /* [dev] [I] sum_i (f_i - a_i)            (Eq. 3a)              */
    int64_t* p99_latency;    /* [dev] [I] nearest-rank: ceil(0.99 n)-th smallest latency (R13)      */
    int32_t* makespan;       /* [dev] [I] max_i f_i                                                 */
    int64_t* peak_kv;        /* [dev] [I] max_t mem(t) by Eq. 3c (always <= M)                      */
    int64_t* rounds;         /* [dev] [I] steps whose queue is non-empty after arrivals (R16)       */
    int64_t* decisions;      /* [dev] [I] admissions + one blocked-head evaluation per round that
                                          ends with a non-empty queue (R16)                         */
    int32_t* status;         /* [dev] [I] SVF_OK or a data error; a rejected instance reports zeros */
} svf_result_t;

/* a1 + a2 (Eq. 1 / Eq. 2 / SJF / FCFS): words_out[i] = (key_i << 32) + i,
 * i = index in the (arrival, id)-ordered input, so ascending word order IS the priority order
 * (key, arrival, id).  s, o: [dev][n]; a: [dev][n], needed for SVF_FCFS only (else may be NULL);
 * bit: [dev][n], needed for SVF_SVF_1BIT only.  status_out: [dev] one int32, set to SVF_OK or
 * SVF_EOVERFLOW (some key >= 2^32; that word holds the key modulo 2^32); may be NULL.
 * 0 <= n <= 2^32.  One streaming pass: 8-13 B read + 8 B written per request. */
int svf_keys(int policy, int64_t n, const int32_t* s, const int32_t* o, const int32_t* a,
             const uint8_t* bit, int32_t O0, int32_t O1, uint64_t* words_out,
             int32_t* status_out, void* stream);

/* a1-a5: one stateless admission decision.
 * Waiting requests [dev][n_wait] (w_s, w_o, w_a, w_bit) in (arrival, id) order; running
 * requests [dev][n_run] as r_kv (tokens held now) and r_rem (steps left, >= 1): r holds
 * r_kv + d tokens d steps from now, d = 1..r_rem.  The call computes the keys, radix-sorts the
 * packed words, and admits the longest prefix of the priority order whose members are jointly
 * feasible with the running set (a request admitted now holds w_s + d tokens for d = 1..w_o),
 * stopping at the first blocked head.  Outputs, all [dev]:
 *   n_admitted_out    one int64: k
 *   admitted_idx_out  [n_wait] int32: the first k entries are the admitted input indices in
 *                     priority order (the rest is unspecified); may be NULL
 *   sorted_words_out  [n_wait] uint64: the whole queue in priority order as (key << 32) + index;
 *                     may be NULL
 *   status_out        one int32: SVF_OK / SVF_ERANGE / SVF_EUNSORTED / SVF_EOVERFLOW; on error
 *                     k = 0
 * `t` only dates the decision (the check is relative to now).  0 <= n_wait, n_run < 2^30.
 * Cost: n_wait + n_run <= 8192 (a serving queue): ONE kernel launch on one CTA; larger queues: keys +
 * device-wide radix sort + one CTA that bisects the prefix length over the first 8192 - n_run
 * candidates (serial continuation only if all of those fit and more are waiting). */
size_t svf_admit_workspace_bytes(int64_t n_wait, int64_t n_run);
int svf_admit(int policy, int64_t M, int32_t t,
              int64_t n_wait, const int32_t* w_s, const int32_t* w_o, const int32_t* w_a,
              const uint8_t* w_bit, int32_t O0, int32_t O1,
              int64_t n_run, const int32_t* r_kv, const int32_t* r_rem,
              int64_t* n_admitted_out, int32_t* admitted_idx_out, uint64_t* sorted_words_out,
              int32_t* status_out, void* ws, size_t ws_bytes, void* stream);

/* svf_admit for a caller that may not allocate device memory: same arguments, outputs, data errors
 * and answer as svf_admit, minus `ws` / `ws_bytes`.  Meant for the place this decision is taken in
 * production -- the step loop of a serving engine, or a plug-in inside one.  Such a process gives
 * nearly all HBM to its KV-cache pool at start-up, so a later cudaMalloc may simply fail, and
 * cudaMalloc / cudaFree synchronise the device and would stall the decode stream every step; other
 * hosts forbid allocation outside their own pool, or offer no allocator to a plain C caller.
 * Here the scratch is a fixed array inside the library image (SVF_ADMIT_STATIC_BYTES of device
 * memory on EVERY GPU that loads the library, held until the process exits).  The call issues no
 * cudaMalloc / cudaFree and calls no allocating routine; inputs and outputs remain the caller's.
 *  - Limit: n_wait <= SVF_ADMIT_STATIC_MAX_WAIT and n_run <= SVF_ADMIT_STATIC_MAX_RUN; anything
 *    larger returns SVF_EWORKSPACE (take svf_admit with your own buffer), before the device is
 *    touched.  With svf_set_profiling switched on it returns SVF_EINVAL (that aid creates events).
 *  - First call on each device: it looks up the array's device address (the device that is current
 *    at the call), which may load the library's device code there.  Make that first call during
 *    start-up, ahead of any stream capture; later calls only enqueue kernels and memsets.
 *  - All calls on one GPU share the one array and it still holds whatever the previous call left;
 *    everything the kernels need zeroed is cleared on `stream` at the start of each call.  Two
 *    calls that can overlap on the same GPU (different streams, or different host threads) RACE:
 *    order them on one stream or with events.  svf_admit with separate buffers has no such limit. */
#define SVF_ADMIT_STATIC_MAX_WAIT 65536
#define SVF_ADMIT_STATIC_MAX_RUN  8192
#define SVF_ADMIT_STATIC_BYTES    (3 << 20)
int svf_admit_static(int policy, int64_t M, int32_t t,
                     int64_t n_wait, const int32_t* w_s, const int32_t* w_o, const int32_t* w_a,
                     const uint8_t* w_bit, int32_t O0, int32_t O1,
                     int64_t n_run, const int32_t* r_kv, const int32_t* r_rem,
                     int64_t* n_admitted_out, int32_t* admitted_idx_out, uint64_t* sorted_words_out,
                     int32_t* status_out, void* stream);

/* a1-a7: the batched discrete-time simulator (P:L87-104 model; Alg. 1 Process 2).
 * Per instance, from t = a_0:  COMPLETE (k_i + o_i == t) -> ARRIVE (a_i <= t) -> ADMIT (pop
 * the head of the (key, arrival, id) order while the forward-looking check passes; stop at the
 * first blocked head) -> t+1  (event order: R1), until every request has finished.
 * Presort: keys + a stable radix sort giving every instance its priority order (in shared
 * memory, one CTA per instance, when no instance has more than 4096 requests; else one
 * device-wide segmented onesweep sort); then one persistent kernel, one thread group per
 * instance, which also validates the data and selects p99.
 * `trace` and `out` are HOST structs holding DEVICE pointers (see above). */
size_t svf_simulate_workspace_bytes(const svf_trace_t* trace);
int svf_simulate(const svf_trace_t* trace, int policy, int64_t M, const svf_result_t* out,
                 void* ws, size_t ws_bytes, void* stream);

/* The same simulator under SEVERAL policies in one call (the paper compares SVF, 1-bit SVF, SJF
 * and FCFS on the same workload): policies[0 .. n_policies) [host], 1 <= n_policies <= 8,
 * results of policies[k] in outs[k] ([host] array of structs holding DEVICE pointers; output
 * buffers of different policies must not overlap).  Same semantics and error behaviour as
 * n_policies calls of svf_simulate; the instances of all policies share ONE persistent launch
 * (n_policies x I work items), which keeps the GPU full when I alone is only a wave or two. */
size_t svf_simulate_policies_workspace_bytes(const svf_trace_t* trace, int n_policies);
int svf_simulate_policies(const svf_trace_t* trace, int n_policies, const int* policies, int64_t M,
                          const svf_result_t* outs, void* ws, size_t ws_bytes, void* stream);

/* the volume lower bound of Proposition 3.1 (Eq. 5).  With the
 * volumes of an instance sorted ascending, vol_(1) <= ... <= vol_(n) (Eq. 1),
 *     lb_out[j] = sum_{k=1..n} sum_{i=1..k} vol_(i) = sum_i (n - i + 1) vol_(i),
 * so that for BURST input (all requests present at the start) M * TEL(any feasible schedule) >=
 * lb_out[j]; TEL(policy) * M / lb_out[j] upper-bounds the policy's approximation ratio where the
 * optimum cannot be computed.  Arrivals, `bit` and `output_key` are not read.  lb_out: [dev] [I]
 * int64; status_out: [dev] [I] int32 or NULL: SVF_OK, SVF_ERANGE (o_i < 1 or s_i < 0),
 * SVF_EOVERFLOW (bound >= 2^63; ALSO any volume >= 2^32: a limit of this library, whose presort
 * orders 32-bit keys -- Eq. 5 itself sets no width and the CPU oracle returns the exact bound there, R19),
 * SVF_EINVAL (bad offsets); lb_out[j] = 0 unless SVF_OK.
 * Keys + the same presort as svf_simulate + one reduction kernel. */
size_t svf_volume_lower_bound_workspace_bytes(const svf_trace_t* trace);
int svf_volume_lower_bound(const svf_trace_t* trace, int64_t* lb_out, int32_t* status_out, void* ws,
                           size_t ws_bytes, void* stream);

/* The sort subsystem on its own (a3), for tests and measurement: ascending, stable LSD
 * onesweep radix sort of n 64-bit words on the bit range [bit_lo, bit_hi) (0 <= bit_lo <
 * bit_hi <= 64; words that agree on that range keep their input order).  words_in: [dev][n]
 * (not modified); words_out: [dev][n].  0 <= n < 2^30. */
size_t svf_sort_workspace_bytes(int64_t n, int bit_lo, int bit_hi);
int svf_sort_words(int64_t n, const uint64_t* words_in, uint64_t* words_out, int bit_lo,
                   int bit_hi, void* ws, size_t ws_bytes, void* stream);

/* For tests of the sizing rule (host only, no device needed): the bytes a call of
 * svf_simulate_policies with THIS budget M carves from `ws` (M picks the kernel form, and the forms
 * differ in scratch).  Always <= svf_simulate_policies_workspace_bytes(trace, n_policies), which is
 * the maximum over every M and stays the size a caller must provide.  0 on bad arguments. */
size_t svf_simulate_layout_bytes(const svf_trace_t* trace, int n_policies, int64_t M);

/* Number of kernels the last call of each kind enqueued on this host thread (for the
 * "gpu_launches" count of bench.py); which: 0 = svf_keys, 1 = svf_admit, 2 = svf_simulate,
 * 3 = svf_sort_words. */
int64_t svf_last_launch_count(int which);

/* Measurement aids.  svf_set_profiling(1): later svf_simulate calls on this host thread record
 * CUDA events on their stream around the three phases.  svf_simulate_phase_ms waits for the
 * events of the last such call and writes ms_out ([host] float[4]): [0] phase A (keys +
 * presort + rank, every policy of the call), [1] phase B (the persistent simulator kernel), [2]
 * phase C (p99 sort + gather of the M >= 2^30 kernel; else 0: p99 is selected inside the simulator
 * kernel), [3] the whole call.  Returns SVF_EINVAL if profiling was off.
 * svf_set_profiling(2): as 1, and the simulator kernel also counts its algorithmic work (a
 * slower variant of the same kernel, same results; M < 2^30 only): svf_simulate_work_counts
 * synchronises and writes counts_out ([host] uint64[4]): [0] E = running entries examined,
 * summed over every head evaluation (a4), [1] U = running entries updated, summed over every
 * admission (a5), [2] head evaluations performed, [3] of them blocked.  The counts live in the
 * workspace of that call, which must still be allocated.  svf_set_profiling(0) switches both off. */
void svf_set_profiling(int mode);
int svf_simulate_phase_ms(float* ms_out);
int svf_simulate_work_counts(uint64_t* counts_out);
/* The same for svf_admit (profiling mode 1 or 2): ms_out ([host] float[4]): [0] a1 + a2 keys, packing
 * and validation, [1] a3 the sorts, [2] a4 + a5 the admission kernels (and the copy of the sorted
 * words, if asked for), [3] the whole call. */
int svf_admit_phase_ms(float* ms_out);

const char* svf_status_string(int status);
const char* svf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SVF_H_ */
