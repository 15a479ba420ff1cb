// a3: device-wide stable LSD radix sort of 64-bit words ("onesweep": one up-front histogram of
// every digit, then one chained-scan pass per digit with decoupled look-back), sm_100a.
//
// Serves the waiting-queue sort of the paper's admission rule (ascending key, P:L67, P:L351;
// unique tie-break P:L501) on packed (key, arrival, id) words, the segmented presort of
// svf_simulate (instance id in the top bits) and the per-instance latency sort behind p99.
//
// Design notes (B200):
//  * HBM-bound: 8 B/word for the histogram + 16 B/word per executed pass.  A pass whose digit is
//    identical in every word is detected from the histogram ON THE DEVICE and skipped, so the
//    host never reads anything back (key bits are bounded: < 2^24..2^26 for the paper-shaped
//    workloads).
//  * Each pass CTA owns one 4096-word tile (32 KB): the tile is staged global->shared with one
//    1-D TMA bulk copy (cp.async.bulk + mbarrier); its digit counts are taken first (shared-memory
//    atomics) and published as the tile's AGGREGATE before anything else, then the keys are ranked
//    per warp with one ballot per digit bit (stable; no MATCH instruction: measured slower),
//    scattered inside shared memory so the final global stores are coalesced runs per digit.
//  * Decoupled look-back, eight predecessor words per round trip to L2 (independent loads consumed
//    in order).  Tile ids come from an atomic counter, so a tile's predecessors are always
//    resident or done: the look-back spin cannot deadlock.
//  * The plan kernel ping-pongs the two buffers so that the last EXECUTED pass lands in the
//    caller's output buffer: no copy afterwards.
#include "svf_internal.cuh"
#include "svf_segsort.cuh"

namespace svf {

namespace {

constexpr uint32_t FLAG_AGG = 1u << 30, FLAG_INCL = 2u << 30, VALUE_MASK = (1u << 30) - 1u;

__device__ __forceinline__ uint32_t digit_of(uint64_t w, int shift, uint32_t mask)
{
    return (uint32_t)(w >> shift) & mask;
}

// ---- histogram of every digit in one read of the input ---------------------------------------
template <int NPASS>
__global__ void __launch_bounds__(512) k_sort_hist(const uint64_t* __restrict__ in, int64_t n,
                                                   int bit_lo, int bit_hi,
                                                   uint32_t* __restrict__ ghist)
{
    __shared__ uint32_t sh[NPASS * SORT_RADIX];
    for (int i = threadIdx.x; i < NPASS * SORT_RADIX; i += blockDim.x) sh[i] = 0;
    __syncthreads();

    int shift[NPASS]; uint32_t mask[NPASS];
#pragma unroll
    for (int p = 0; p < NPASS; ++p) {
        shift[p] = bit_lo + p * SORT_RADIX_BITS;
        int wdt = bit_hi - shift[p]; if (wdt > SORT_RADIX_BITS) wdt = SORT_RADIX_BITS;
        mask[p] = (1u << wdt) - 1u;
    }
    // run-length accumulation: a digit that repeats costs one shared atomic per run, so the
    // all-equal high digits of small keys do not serialise on a single bin.  Branch free: the flush
    // of a finished run is one PREDICATED atomic (a branch here diverges on every random digit and
    // tripled the instruction count of this kernel)
    uint32_t last[NPASS], cnt[NPASS];
#pragma unroll
    for (int p = 0; p < NPASS; ++p) { last[p] = 0; cnt[p] = 0; }
    auto take = [&](uint64_t w) {
#pragma unroll
        for (int p = 0; p < NPASS; ++p) {
            const uint32_t d = digit_of(w, shift[p], mask[p]);
            const bool same = d == last[p];
            if (!same && cnt[p]) atomicAdd(&sh[p * SORT_RADIX + last[p]], cnt[p]);
            cnt[p] = same ? cnt[p] + 1 : 1;
            last[p] = d;
        }
    };

    // two words per 128-bit load, four loads in flight per thread; the tail (and an unaligned
    // input) word by word
    const bool vec = (reinterpret_cast<uintptr_t>(in) & 15u) == 0;
    const int64_t n2 = vec ? (n >> 1) : 0;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    constexpr int UNR = 4;
    const ulonglong2* __restrict__ in2 = reinterpret_cast<const ulonglong2*>(in);
    int64_t q0 = gid;
    for (; q0 + (UNR - 1) * stride < n2; q0 += stride * UNR) {
        ulonglong2 w[UNR];
#pragma unroll
        for (int u = 0; u < UNR; ++u) w[u] = __ldg(in2 + q0 + u * stride);
#pragma unroll
        for (int u = 0; u < UNR; ++u) { take(w[u].x); take(w[u].y); }
    }
    for (; q0 < n2; q0 += stride) { const ulonglong2 w = __ldg(in2 + q0); take(w.x); take(w.y); }
    for (int64_t i = (n2 << 1) + gid; i < n; i += stride) take(__ldg(in + i));
#pragma unroll
    for (int p = 0; p < NPASS; ++p) if (cnt[p]) atomicAdd(&sh[p * SORT_RADIX + last[p]], cnt[p]);
    __syncthreads();
    for (int i = threadIdx.x; i < NPASS * SORT_RADIX; i += blockDim.x)
        if (sh[i]) atomicAdd(&ghist[i], sh[i]);
}

// ---- exclusive scan of each digit histogram + the ping-pong plan -------------------------------
__global__ void __launch_bounds__(SORT_RADIX) k_sort_plan(uint32_t* __restrict__ hist, int npass,
                                                         int64_t n, const uint64_t* in,
                                                         uint64_t* x, uint64_t* y,
                                                         SortPlan* __restrict__ plan)
{
    __shared__ uint32_t warp_tot[SORT_RADIX / 32];
    __shared__ int skip_s[SORT_MAX_PASSES];
    const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
    for (int p = 0; p < npass; ++p) {
        uint32_t c = hist[p * SORT_RADIX + tid];
        int trivial = __syncthreads_or(c == (uint32_t)n);
        uint32_t inc = c;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { uint32_t v = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += v; }
        if (lane == 31) warp_tot[wrp] = inc;
        __syncthreads();
        uint32_t off = 0;
        for (int w = 0; w < wrp; ++w) off += warp_tot[w];
        hist[p * SORT_RADIX + tid] = off + inc - c;
        if (tid == 0) skip_s[p] = trivial;
        __syncthreads();
    }
    if (tid == 0) {
        // ping-pong x, y so that the LAST executed pass writes x (the caller's output buffer: no
        // copy afterwards); when y aliases the input the first pass must write x instead
        int exec = 0;
        for (int p = 0; p < npass; ++p) exec += skip_s[p] ? 0 : 1;
        bool to_x = (y == in) ? true : ((exec & 1) != 0);
        const uint64_t* cur = in;
        for (int p = 0; p < npass; ++p) {
            plan->skip[p] = skip_s[p];
            if (skip_s[p]) { plan->src[p] = nullptr; plan->dst[p] = nullptr; continue; }
            uint64_t* d = to_x ? x : y;
            to_x = !to_x;
            plan->src[p] = cur; plan->dst[p] = d; cur = d;
        }
        plan->result = cur;
    }
}

// ---- TMA 1-D bulk copy + mbarrier (PTX; SASS: UBLKCP / SYNCS) ---------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_1d(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// ---- one onesweep pass -----------------------------------------------------------------------
struct PassSmem {
    uint64_t* staging; uint32_t *whist, *thist, *toff_s, *gbase_s, *warp_tot;
};

// the body for one tile; FULL = the tile holds SORT_TILE words (every tile but the last): the
// "is this element inside the tile" tests are compiled out of it
template <bool FULL>
__device__ __forceinline__ void sort_pass_tile(const PassSmem& sm, int tile_n, uint32_t tile,
                                               int shift, uint32_t mask, uint32_t* __restrict__ status,
                                               const uint32_t* __restrict__ bases, uint64_t* __restrict__ dst)
{
    constexpr int WARPS = SORT_THREADS / 32;
    const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
    const int wbase = wrp * 32 * SORT_IPT;
    // the digit of every key of this thread, once, four to a register; the keys themselves stay in
    // the staged tile until the scatter (16 x 64 bit in registers through the ranking would spill)
    uint32_t dig4[SORT_IPT / 4];
#pragma unroll
    for (int i = 0; i < SORT_IPT / 4; ++i) dig4[i] = 0;
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) dig4[i >> 2] |= digit_of(sm.staging[wbase + i * 32 + lane], shift, mask) << (8 * (i & 3));
    auto dig = [&](int i) { return (dig4[i >> 2] >> (8 * (i & 3))) & 0xffu; };

    // the tile's digit counts first (shared-memory atomics), published BEFORE the ranking: the
    // successors' look-back then finds an aggregate while this tile is still ranking (deriving the
    // counts from the ranking's warp histograms instead saves the atomics but publishes late: 2.11
    // against 1.78 ms for the 2^26-word sort)
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i)
        if (FULL || (wbase + i * 32 + lane) < tile_n) atomicAdd(&sm.thist[dig(i)], 1u);
    __syncthreads();
    const uint32_t count = sm.thist[tid];
    volatile uint32_t* st = status + (size_t)tile * SORT_RADIX + tid;
    *st = (tile == 0 ? FLAG_INCL : FLAG_AGG) | count;
    {   // tile-level exclusive scan of the counts
        uint32_t inc = count;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { uint32_t v = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += v; }
        if (lane == 31) sm.warp_tot[wrp] = inc;
        __syncthreads();
        uint32_t off = 0;
        for (int w = 0; w < wrp; ++w) off += sm.warp_tot[w];
        sm.toff_s[tid] = off + inc - count;
    }

    // per-warp stable ranking with digit ballots; two ranks (< 4096 each) to a register
    uint32_t* wh = sm.whist + wrp * SORT_RADIX;
    const uint32_t lt_mask = (1u << lane) - 1u;
    uint32_t rank2[SORT_IPT / 2];
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {
        const bool valid = FULL || (wbase + i * 32 + lane) < tile_n;
        const uint32_t d = dig(i);
        const uint32_t peers = warp_match_digit<FULL>(d, valid);
        // the highest peer owns the warp-private counter of its digit for this round
        const int leader = 31 - __clz(peers);
        uint32_t base = 0;
        if (valid && lane == leader) { base = wh[d]; wh[d] = base + __popc(peers); }
        base = __shfl_sync(0xffffffffu, base, leader);
        __syncwarp();
        const uint32_t r = base + __popc(peers & lt_mask);
        if (i & 1) rank2[i >> 1] |= r << 16; else rank2[i >> 1] = r;
    }
    __syncthreads();

    // digit d (thread d): exclusive scan of the warp-private counts over the warps; then the
    // decoupled look-back over the predecessor tiles of this digit (their aggregates were
    // published before their ranking, so this rarely waits)
    {
        // (the digit's offset inside the tile is folded in: the scatter then needs one lookup per key)
        uint32_t run = sm.toff_s[tid];
#pragma unroll
        for (int w = 0; w < WARPS; ++w) { uint32_t c = sm.whist[w * SORT_RADIX + tid]; sm.whist[w * SORT_RADIX + tid] = run; run += c; }
        uint32_t excl = 0;
        if (tile > 0) {
            // eight predecessors per round trip to L2 (independent loads), consumed in order
            constexpr int LOOK = 8;
            int64_t look = (int64_t)tile - 1;
            bool done = false;
            while (!done) {
                uint32_t v[LOOK];
#pragma unroll
                for (int q = 0; q < LOOK; ++q) {
                    const int64_t idx = look - q;
                    v[q] = idx >= 0 ? *(volatile uint32_t*)(status + (size_t)idx * SORT_RADIX + tid) : (2u << 30);   // past tile 0: an empty inclusive word
                }
                int used = 0;
#pragma unroll
                for (int q = 0; q < LOOK; ++q) {
                    if (!done && used == q) {
                        const uint32_t f = v[q] >> 30;
                        if (f != 0) {
                            excl += v[q] & VALUE_MASK;
                            ++used;
                            if (f == 2) done = true;
                        }
                    }
                }
                look -= used;
            }
            *st = FLAG_INCL | (excl + count);
        }
        sm.gbase_s[tid] = bases[tid] + excl - sm.toff_s[tid];    // modulo 2^32; dst index = gbase + slot
    }
    // every thread takes its keys out of the staged tile, then the tile is rewritten in digit order
    uint64_t key[SORT_IPT];
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) key[i] = sm.staging[wbase + i * 32 + lane];
    __syncthreads();

    // scatter inside shared memory, then write coalesced runs
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {
        if (FULL || (wbase + i * 32 + lane) < tile_n) {
            const uint32_t d = dig(i);
            const uint32_t r = (i & 1) ? (rank2[i >> 1] >> 16) : (rank2[i >> 1] & 0xffffu);
            sm.staging[wh[d] + r] = key[i];
        }
    }
    __syncthreads();
    if (FULL) {
#pragma unroll 4
        for (int q = tid; q < SORT_TILE; q += SORT_THREADS) {
            const uint64_t w = sm.staging[q];
            dst[(uint32_t)(sm.gbase_s[digit_of(w, shift, mask)] + (uint32_t)q)] = w;
        }
    } else {
        for (int q = tid; q < tile_n; q += SORT_THREADS) {
            const uint64_t w = sm.staging[q];
            dst[(uint32_t)(sm.gbase_s[digit_of(w, shift, mask)] + (uint32_t)q)] = w;
        }
    }
}

__global__ void __launch_bounds__(SORT_THREADS, 4) k_sort_pass(const SortPlan* __restrict__ plan,
                                                            int p, int64_t n, int shift,
                                                            uint32_t mask,
                                                            uint32_t* __restrict__ tile_ctr,
                                                            uint32_t* __restrict__ status,
                                                            const uint32_t* __restrict__ bases)
{
    constexpr int WARPS = SORT_THREADS / 32;
    __shared__ __align__(128) uint64_t staging[SORT_TILE];
    __shared__ uint32_t whist[WARPS * SORT_RADIX];
    __shared__ uint32_t thist[SORT_RADIX];
    __shared__ uint32_t toff_s[SORT_RADIX];
    __shared__ uint32_t gbase_s[SORT_RADIX];
    __shared__ uint32_t warp_tot[SORT_RADIX / 32];
    __shared__ __align__(8) uint64_t bar;
    __shared__ uint32_t tile_s;

    if (plan->skip[p]) return;                      // uniform over the grid
    const uint64_t* __restrict__ src = plan->src[p];
    uint64_t* __restrict__ dst = plan->dst[p];

    const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
    if (tid == 0) { tile_s = atomicAdd(&tile_ctr[p], 1u); mbar_init(&bar, 1); }
    for (int i = tid; i < WARPS * SORT_RADIX; i += SORT_THREADS) whist[i] = 0;
    thist[tid] = 0;
    __syncthreads();
    const uint32_t tile = tile_s;
    const int64_t tile_base = (int64_t)tile * SORT_TILE;
    const int tile_n = (int)((n - tile_base) < (int64_t)SORT_TILE ? (n - tile_base) : (int64_t)SORT_TILE);

    // stage the tile, then take it in warp-striped order: item i of lane l in warp w is element
    // w*32*IPT + i*32 + l of the tile (so ranks follow the input order = stability)
    const bool bulk = (tile_n == SORT_TILE) && ((reinterpret_cast<uintptr_t>(src + tile_base) & 15u) == 0);
    if (bulk) {
        if (tid == 0) {
            mbar_expect_tx(&bar, SORT_TILE * 8u);
            tma_load_1d(staging, src + tile_base, SORT_TILE * 8u, &bar);
        }
        mbar_wait(&bar, 0);
    } else {
        // ragged or unaligned tile: plain coalesced loads into the same staging buffer
        for (int e = tid; e < SORT_TILE; e += SORT_THREADS) staging[e] = e < tile_n ? __ldg(src + tile_base + e) : ~0ull;
        __syncthreads();
    }
    (void)lane; (void)wrp;
    PassSmem sm{staging, whist, thist, toff_s, gbase_s, warp_tot};
    if (tile_n == SORT_TILE) sort_pass_tile<true>(sm, tile_n, tile, shift, mask, status, bases, dst);
    else                     sort_pass_tile<false>(sm, tile_n, tile, shift, mask, status, bases, dst);
}

__global__ void k_sort_copy_result(const SortPlan* __restrict__ plan, uint64_t* __restrict__ out, int64_t n)
{
    const uint64_t* __restrict__ r = plan->result;
    if (r == out) return;
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) out[i] = r[i];
}

__global__ void k_sort_plan_identity(SortPlan* plan, const uint64_t* in) { plan->result = in; }

// ---- segmented sort of SMALL segments, entirely in shared memory ------------------------------
// One CTA per instance (svf_simulate's presort when every instance has at most SEG_SORT_MAX
// requests): keys (Eq. 1 / Eq. 2 / o / a) are computed from the trace, packed as (key << 32) + id,
// sorted by stable LSD radix passes over the significant key bytes only (an OR-reduction of the
// keys tells how many), ping-pong between two shared-memory buffers with the same warp-ballot
// ranking as k_sort_pass, and the priority order leaves the chip once: order[] (id at rank),
// rank[] (rank of id) and, if wanted, the (s, o, id, a) records in priority order.  HBM traffic:
// 12-13 B read + 8 B (24 B with records) written per request, against 8 + 16 B per executed pass
// of the device-wide sort.
template <int SORT_THREADS, int IPT>
__global__ void __launch_bounds__(SORT_THREADS) k_seg_sort(SegSortArgs A)
{
    static_assert(SORT_THREADS == 128 || SORT_THREADS == 256, "seg_pass: one or two digits per thread in the scans");
    constexpr int WARPS = SORT_THREADS / 32;
    extern __shared__ __align__(16) uint64_t seg_buf[];       // [2][cap]
    __shared__ uint32_t whist[WARPS * SORT_RADIX];
    __shared__ uint32_t toff_s[SORT_RADIX];
    __shared__ uint32_t warp_tot[WARPS];
    __shared__ uint32_t kor_s;
    const int tid = threadIdx.x;
    const int cap = A.cap;
    const int32_t* __restrict__ s = A.s;
    const int32_t* __restrict__ o = A.o;
    const int32_t* __restrict__ a = A.a;
    const int32_t* __restrict__ klen = A.okey ? A.okey : A.o;     // the length the SVF / SJF key sees
    for (int64_t j = blockIdx.x; j < A.I; j += gridDim.x) {
        const int64_t base = A.off[j], n64 = A.off[j + 1] - base;
        if (n64 <= 0 || n64 > cap || base < 0 || base + n64 > A.N) continue;   // the simulator reports the layout error
        const int n = (int)n64;
        // every policy of the call on this instance: the trace is read from HBM once (the later
        // policies hit L1 / L2) and the call pays one launch tail instead of one per policy
        for (int q = 0; q < A.n_policies; ++q) {
            const int policy = A.policy[q];
            uint32_t* __restrict__ order = A.order[q];
            uint32_t* __restrict__ rank = A.rank[q];
            int4* __restrict__ req = A.req[q];
            if (policy == SVF_FCFS) {
                // key = arrival and the input IS in (arrival, id) order (an instance whose arrivals
                // decrease is rejected by the simulator): the priority order is the identity
                for (int p = tid; p < n; p += SORT_THREADS) {
                    order[base + p] = (uint32_t)p;
                    rank[base + p] = (uint32_t)p;
                    if (req) req[base + p] = make_int4(s[base + p], o[base + p], p, a[base + p]);
                }
                continue;
            }
            if (tid == 0) kor_s = 0;
            __syncthreads();
            uint64_t* buf0 = seg_buf;
            uint64_t* buf1 = seg_buf + cap;
            uint32_t kor = 0;
            for (int i = tid; i < n; i += SORT_THREADS) {
                const uint32_t b = policy == SVF_SVF_1BIT ? (uint32_t)A.bit[base + i] : 0u;
                const uint32_t key = (uint32_t)priority_key(policy, s[base + i], klen[base + i], 0, b, A.O0, A.O1);
                buf0[i] = ((uint64_t)key << 32) | (uint32_t)i;
                kor |= key;
            }
            kor = __reduce_or_sync(0xffffffffu, kor);
            if ((tid & 31) == 0 && kor) atomicOr(&kor_s, kor);
            __syncthreads();
            const uint32_t kall = kor_s;
            const int bits = kall ? 32 - __clz(kall) : 0;
            const int npass = (bits + SORT_RADIX_BITS - 1) / SORT_RADIX_BITS;
            const int ipt = (n + SORT_THREADS - 1) / SORT_THREADS;
            for (int p = 0; p < npass; ++p) {
                seg_pass<SORT_THREADS, IPT>(buf0, buf1, n, ipt, 32 + p * SORT_RADIX_BITS, whist, toff_s, warp_tot);
                uint64_t* t = buf0; buf0 = buf1; buf1 = t;
            }
            for (int p = tid; p < n; p += SORT_THREADS) {
                const uint32_t id = (uint32_t)buf0[p];
                order[base + p] = id;
                rank[base + id] = (uint32_t)p;
                if (req) req[base + p] = make_int4(s[base + id], o[base + id], (int)id, a[base + id]);
            }
            __syncthreads();
        }
    }
}

}  // namespace

// SMs of the CURRENT device, asked every time (an attribute query, no device work): nothing is
// cached per process, so threads driving different devices each get their own count; 148 (B200)
// when there is no device, so that the host-side size computations still work there.
int sm_count()
{
    int dev = 0, v = 0;
    if (cudaGetDevice(&dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0)
        return v;
    return 148;
}

static size_t sort_status_bytes(int64_t n, int bit_lo, int bit_hi)
{
    int64_t tiles = ceil_div(n > 0 ? n : 1, SORT_TILE);
    return align_up((size_t)sort_num_passes(bit_lo, bit_hi) * (size_t)tiles * SORT_RADIX * sizeof(uint32_t), 256);
}

size_t sort_ws_bytes(int64_t n, int bit_lo, int bit_hi)
{
    size_t b = 0;
    b += align_up(sizeof(SortPlan), 256);
    b += align_up(sizeof(uint32_t) * SORT_MAX_PASSES * SORT_RADIX, 256);
    b += align_up(sizeof(uint32_t) * SORT_MAX_PASSES, 256);
    b += sort_status_bytes(n, bit_lo, bit_hi);
    return b;
}

void sort_ws_carve(SortWs* w, void* base, int64_t n, int bit_lo, int bit_hi)
{
    char* p = (char*)base;
    w->plan = (SortPlan*)p;       p += align_up(sizeof(SortPlan), 256);
    w->hist = (uint32_t*)p;       p += align_up(sizeof(uint32_t) * SORT_MAX_PASSES * SORT_RADIX, 256);
    w->tile_ctr = (uint32_t*)p;   p += align_up(sizeof(uint32_t) * SORT_MAX_PASSES, 256);
    w->status = (uint32_t*)p;
    w->status_bytes = sort_status_bytes(n, bit_lo, bit_hi);
}

int sort_u64(const SortWs& w, const uint64_t* in, uint64_t* x, uint64_t* y, int64_t n, int bit_lo,
             int bit_hi, cudaStream_t st, int64_t* launches)
{
    if (n <= 0) {
        k_sort_plan_identity<<<1, 1, 0, st>>>(w.plan, in);
        ++*launches;
        return (int)cudaGetLastError();
    }
    const int npass = sort_num_passes(bit_lo, bit_hi);
    // hist, tile counters and look-back words are contiguous: one memset
    size_t zero_bytes = (size_t)((char*)w.status - (char*)w.hist) + w.status_bytes;
    cudaError_t e = cudaMemsetAsync(w.hist, 0, zero_bytes, st);
    if (e != cudaSuccess) return (int)e;

    const int hthreads = 512;
    int64_t hblocks = ceil_div(n, (int64_t)hthreads * 8);
    int64_t hmax = (int64_t)sm_count() * 4;
    if (hblocks > hmax) hblocks = hmax;
    if (hblocks < 1) hblocks = 1;
    switch (npass) {
#define SVF_HIST_CASE(NP) case NP: k_sort_hist<NP><<<(unsigned)hblocks, hthreads, 0, st>>>(in, n, bit_lo, bit_hi, w.hist); break;
        SVF_HIST_CASE(1) SVF_HIST_CASE(2) SVF_HIST_CASE(3) SVF_HIST_CASE(4)
        SVF_HIST_CASE(5) SVF_HIST_CASE(6) SVF_HIST_CASE(7) SVF_HIST_CASE(8)
#undef SVF_HIST_CASE
    default: return (int)cudaErrorInvalidValue;
    }
    ++*launches;
    k_sort_plan<<<1, SORT_RADIX, 0, st>>>(w.hist, npass, n, in, x, y, w.plan);
    ++*launches;
    const int64_t tiles = ceil_div(n, SORT_TILE);
    for (int p = 0; p < npass; ++p) {
        int shift = bit_lo + p * SORT_RADIX_BITS;
        int wdt = bit_hi - shift; if (wdt > SORT_RADIX_BITS) wdt = SORT_RADIX_BITS;
        k_sort_pass<<<(unsigned)tiles, SORT_THREADS, 0, st>>>(w.plan, p, n, shift, (1u << wdt) - 1u, w.tile_ctr,
                                                              w.status + (size_t)p * tiles * SORT_RADIX,
                                                              w.hist + p * SORT_RADIX);
        ++*launches;
    }
    return (int)cudaGetLastError();
}

int seg_sort_keys(const SegSortArgs& A, int64_t max_instance, cudaStream_t st, int64_t* launches)
{
    if (A.I <= 0 || A.N <= 0 || A.n_policies <= 0) return 0;
    if (max_instance > SEG_SORT_MAX || A.n_policies > SEG_SORT_MAX_POLICIES) return (int)cudaErrorInvalidValue;
    SegSortArgs B = A;
    B.cap = (int)((max_instance > 0 ? max_instance : 1) + 1) / 2 * 2;
    const size_t smem = (size_t)2 * B.cap * sizeof(uint64_t);
    // items per thread sized to the largest instance (registers: occupancy of small segments)
#define SVF_SEG_LAUNCH(T, IPT)                                                                          \
    do {                                                                                                \
        cudaFuncSetAttribute(k_seg_sort<T, IPT>, cudaFuncAttributeMaxDynamicSharedMemorySize,           \
                             2 * SEG_SORT_MAX * (int)sizeof(uint64_t));   /* per device: set every time */ \
        int per_sm = 0;                                                                                 \
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_seg_sort<T, IPT>, T, smem)         \
                != cudaSuccess || per_sm < 1)                                                           \
            per_sm = 1;                                                                                 \
        int64_t grid = (int64_t)per_sm * sm_count();                                                    \
        if (grid > B.I) grid = B.I;                                                                     \
        k_seg_sort<T, IPT><<<(unsigned)grid, T, smem, st>>>(B);                                         \
    } while (0)
    // instances of at most 1024 requests: CTAs of four warps (half the per-pass overhead of the
    // histogram reset and the digit scans, barriers over four warps, twice the CTAs per SM)
    if (B.cap <= 8 * 128) SVF_SEG_LAUNCH(128, 8);
    else if (B.cap <= 8 * 256) SVF_SEG_LAUNCH(256, 8);
    else SVF_SEG_LAUNCH(256, 16);
#undef SVF_SEG_LAUNCH
    ++*launches;
    return (int)cudaGetLastError();
}

int sort_result_to(const SortWs& w, uint64_t* out, int64_t n, cudaStream_t st, int64_t* launches)
{
    if (n <= 0) return 0;
    int64_t blocks = ceil_div(n, 256 * 4);
    int64_t bmax = (int64_t)sm_count() * 8;
    if (blocks > bmax) blocks = bmax;
    k_sort_copy_result<<<(unsigned)blocks, 256, 0, st>>>(w.plan, out, n);
    ++*launches;
    return (int)cudaGetLastError();
}

}  // namespace svf
