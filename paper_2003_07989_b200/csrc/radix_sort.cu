// radix_sort.cu -- onesweep LSD radix sort of 64-bit records on a bit range, written by hand for
// sm_100a (no CUB/Thrust).  One histogram kernel over all digits (or a producer kernel that counts them while it
// writes the records), then one kernel per digit that scans the digit's histogram, ranks a tile in shared memory, resolves its global offsets with a decoupled look-back chained
// scan over (tile, bin) status words, and scatters coalesced runs.  Stable, so records that enter
// in increasing combinatorial index leave each pass in increasing index within equal digits: the
// index bits never have to be sorted.
#include "radix_sort.cuh"
#include <mutex>

namespace {

#ifndef RIPS_SORT_THREADS
#define RIPS_SORT_THREADS 256
#define RIPS_SORT_IPT 20
#define RIPS_SORT_MIN_BLOCKS 3
#define RIPS_SORT_RANK_BATCH 2
#endif
constexpr int SORT_THREADS = RIPS_SORT_THREADS;   // >= RIPS_SORT_MAX_BINS: one thread per bin for the scans and the look-back
constexpr int SORT_IPT = RIPS_SORT_IPT;
constexpr int SORT_MIN_BLOCKS = RIPS_SORT_MIN_BLOCKS;
#ifndef RIPS_SORT_LB_BATCH
#define RIPS_SORT_LB_BATCH 8
#endif
constexpr int SORT_LB_BATCH = RIPS_SORT_LB_BATCH;     // predecessor tiles read per look-back step
constexpr int SORT_RANK_BATCH = RIPS_SORT_RANK_BATCH;   // records ranked per pipelined batch (divides SORT_IPT)
constexpr int SORT_TILE = SORT_THREADS * SORT_IPT;
constexpr int SORT_WARPS = SORT_THREADS / 32;

constexpr int HIST_THREADS = 512;
constexpr int HIST_IPT = 16;

// ----------------------------------------------------------------------------------------------
// Histogram of every digit of the plan in one read of the records.
// hist: [npasses][RIPS_SORT_MAX_BINS] u64, zeroed by the caller.
// ----------------------------------------------------------------------------------------------
struct PlanDev {
    int npasses;
    int shift[RIPS_SORT_MAX_PASSES];
    int bits[RIPS_SORT_MAX_PASSES];
};

__global__ void __launch_bounds__(HIST_THREADS) sort_histogram_kernel(const u64* __restrict__ in, i64 n, const u64* __restrict__ n_dev,
                                                                      PlanDev plan, u64* __restrict__ hist)
{
    if (n_dev) n = min(n, (i64)__ldg(n_dev)); // the record count lives on the device: n is its upper bound
    extern __shared__ u32 sh_hist[]; // [npasses][MAX_BINS]
    const int total_bins = plan.npasses * RIPS_SORT_MAX_BINS;
    for (int i = threadIdx.x; i < total_bins; i += HIST_THREADS) sh_hist[i] = 0;
    __syncthreads();
    const i64 chunk = (i64)HIST_THREADS * HIST_IPT;
    for (i64 base = (i64)blockIdx.x * chunk; base < n; base += (i64)gridDim.x * chunk) {
        u64 k[HIST_IPT];
#pragma unroll
        for (int i = 0; i < HIST_IPT; ++i) {
            i64 idx = base + (i64)i * HIST_THREADS + threadIdx.x;
            k[i] = idx < n ? __ldg(in + idx) : 0;
        }
#pragma unroll
        for (int i = 0; i < HIST_IPT; ++i) {
            i64 idx = base + (i64)i * HIST_THREADS + threadIdx.x;
            if (idx < n) {
                for (int p = 0; p < plan.npasses; ++p) {
                    u32 d = (u32)(k[i] >> plan.shift[p]) & ((1u << plan.bits[p]) - 1u);
                    atomicAdd(&sh_hist[p * RIPS_SORT_MAX_BINS + d], 1u);
                }
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < total_bins; i += HIST_THREADS) {
        u32 c = sh_hist[i];
        if (c) atomicAdd((unsigned long long*)&hist[i], (unsigned long long)c);
    }
}

// ----------------------------------------------------------------------------------------------
// One onesweep pass.  Per tile: (1) warp-striped coalesced load; (2) rank inside each warp with
// match.any on the digit (one MATCH per record instead of a ballot per bit) and a per-warp
// histogram in shared memory; (3) per bin, scan over the warps, publish the tile's count for the
// look-back at once, scan over the bins; (4) records placed in tile-sorted order in shared memory;
// (5) decoupled look-back per bin; (6) scatter, consecutive threads writing consecutive slots.
// ----------------------------------------------------------------------------------------------
// BALLOT: how the lanes that share a digit find each other.  One MATCH per record costs ~2 cycles per DISTINCT digit in
// the warp; one ballot per digit bit costs the same whatever the digits.  MATCH wins while a warp's 32 records share a
// few digits (keys of neighbouring simplices of dimension >= 2, cofacet vertices: 0.27 / 0.24 against 0.30 / 0.31 ms
// per pass at cfg 2), ballots win when they are all different (keys of the edges: 1.15 against 1.50 ms per pass on a
// random matrix of 20000 points).  Two instantiations rather than a branch: with both in one kernel the MATCH path
// lost 9 % (measured).  The caller says which passes are of the second kind (sort_u64's ballot_passes).
template <bool BALLOT>
__global__ void __launch_bounds__(SORT_THREADS, SORT_MIN_BLOCKS)
onesweep_pass_kernel(const u64* __restrict__ in, u64* __restrict__ out, i64 n, const u64* __restrict__ n_dev, int shift, int bits,
                     const u64* __restrict__ hist_raw, u64* status, u32* ticket, int pf_dist)
{
    if (n_dev) n = min(n, (i64)__ldg(n_dev)); // launched for the upper bound: the tiles past the count leave at once
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nbins = 1 << bits;
    const u32 mask = (u32)nbins - 1u;
    u64* stage = reinterpret_cast<u64*>(smem_raw);                       // [SORT_TILE]
    u64* goff = stage + SORT_TILE;                                        // [MAX_BINS]
    u32* whist = reinterpret_cast<u32*>(goff + RIPS_SORT_MAX_BINS);       // [SORT_WARPS][MAX_BINS]
    u32* bin_start = whist + SORT_WARPS * RIPS_SORT_MAX_BINS;             // [MAX_BINS]
    __shared__ u32 s_tile;
    __shared__ u32 s_wsum[8];
    __shared__ u64 s_gsum[RIPS_SORT_MAX_BINS / 32];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u); // tiles numbered in the order they start: every predecessor is resident or done
    u32* wh = whist + warp * RIPS_SORT_MAX_BINS;
#pragma unroll
    for (int i = lane; i < RIPS_SORT_MAX_BINS; i += 32) wh[i] = 0;
    // first slot of every bin in the output = exclusive scan of the digit's histogram (raw counts, complete before this
    // pass starts), done by every tile for itself while its records are on their way: one kernel launch less per sort
    // than a separate scan, and nothing of it lies on the tile's critical path
    u64 g_cnt = 0, g_incl = 0;
    if (tid < RIPS_SORT_MAX_BINS) {
        g_cnt = __ldg(hist_raw + tid);
        g_incl = g_cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u64 t = __shfl_up_sync(RIPS_FULL_MASK, g_incl, o);
            if (lane >= o) g_incl += t;
        }
        if (lane == 31) s_gsum[warp] = g_incl;
    }
    __syncthreads();
    u64 g_base = 0; // records whose digit is smaller than `tid`
    if (tid < RIPS_SORT_MAX_BINS) {
#pragma unroll
        for (int w = 0; w < RIPS_SORT_MAX_BINS / 32; ++w) g_base += (w < warp) ? s_gsum[w] : 0ull;
        g_base += g_incl - g_cnt;
    }
    const i64 tile = s_tile;
    const i64 base = tile * SORT_TILE;
    if (base >= n) return; // (uniform; only with a device-side count)
    const int count = (int)min((i64)SORT_TILE, n - base);

    // L2 prefetch of the tile that is pf_dist tickets ahead (one bulk instruction): a CTA has loads in flight only
    // during its short load phase, so without it DRAM reads come in bursts; with it the later loads hit L2.
    if (tid == 0 && pf_dist > 0) {
        const i64 pbase = (tile + pf_dist) * SORT_TILE;
        if (pbase < n) {
            const u32 bytes = (u32)(min((i64)SORT_TILE, n - pbase) * 8) & ~15u;
            const u64* src = in + pbase;
            if (bytes && ((unsigned long long)src & 15ull) == 0)
                asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
        }
    }

    // ---- (1) load: item i of lane l of warp w is record base + w*32*IPT + i*32 + l
    u64 key[SORT_IPT];
    const i64 wbase = base + (i64)warp * (32 * SORT_IPT) + lane;
    if (count == SORT_TILE) {
#pragma unroll
        for (int i = 0; i < SORT_IPT; ++i) key[i] = __ldcs(in + wbase + i * 32);
    } else {
#pragma unroll
        for (int i = 0; i < SORT_IPT; ++i) {
            i64 idx = wbase + i * 32;
            key[i] = idx < n ? __ldcs(in + idx) : ~0ull; // padding: last bin, last inside the tile, never written
        }
    }

    // ---- (2) rank inside the warp.  Three pipelined phases instead of one latency chain per record:
    // all MATCHes, then one shared-memory atomic per digit group and round (the rounds of a warp
    // reach its histogram in program order, so the value returned is the count of the earlier
    // rounds), then the broadcasts.
    u32 rank[SORT_IPT];
    const u32 lt_mask = (1u << lane) - 1u;
#pragma unroll
    for (int h = 0; h < SORT_IPT; h += SORT_RANK_BATCH) {
#pragma unroll
        for (int i = h; i < h + SORT_RANK_BATCH; ++i) {
            const u32 d = (u32)(key[i] >> shift) & mask;
            if (BALLOT) {
                u32 peers = RIPS_FULL_MASK;
                for (int b = 0; b < bits; ++b) {
                    const bool one = (d >> b) & 1u;
                    const u32 v = __ballot_sync(RIPS_FULL_MASK, one);
                    peers &= one ? v : ~v;
                }
                rank[i] = peers;
            } else
                rank[i] = __match_any_sync(RIPS_FULL_MASK, d);
        }
        u32 old[SORT_RANK_BATCH];
#pragma unroll
        for (int i = h; i < h + SORT_RANK_BATCH; ++i) {
            const u32 d = (u32)(key[i] >> shift) & mask;
            old[i - h] = 0;
            if (lane == __ffs(rank[i]) - 1) old[i - h] = atomicAdd(&wh[d], (u32)__popc(rank[i]));
            __syncwarp();
        }
#pragma unroll
        for (int i = h; i < h + SORT_RANK_BATCH; ++i) {
            const u32 peers = rank[i];
            rank[i] = __shfl_sync(RIPS_FULL_MASK, old[i - h], __ffs(peers) - 1) + __popc(peers & lt_mask);
        }
    }
    __syncthreads();

    // ---- (3) per bin: exclusive scan over the warps; publish; exclusive scan over the bins
    const int n_pad = SORT_TILE - count;
    u32 my_count = 0; // valid records of bin `tid` in this tile
    if (tid < RIPS_SORT_MAX_BINS) {
        u32 run = 0;
        if (tid < nbins) {
#pragma unroll
            for (int w = 0; w < SORT_WARPS; ++w) {
                u32 c = whist[w * RIPS_SORT_MAX_BINS + tid];
                whist[w * RIPS_SORT_MAX_BINS + tid] = run;
                run += c;
            }
            my_count = (tid == nbins - 1) ? run - (u32)n_pad : run;
            stress_jitter((u32)tile * 31u + (u32)tid);
            st_volatile_u64(status + tile * nbins + tid, (tile == 0 ? LB_FLAG_INC : LB_FLAG_AGG) | (u64)my_count);
        }
        // block scan of `run` over the first MAX_BINS threads (8 warps)
        u32 incl = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            u32 t = __shfl_up_sync(RIPS_FULL_MASK, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) s_wsum[warp] = incl;
        asm volatile("bar.sync 1, %0;" ::"n"(RIPS_SORT_MAX_BINS));
        u32 woff = 0;
#pragma unroll
        for (int w = 0; w < RIPS_SORT_MAX_BINS / 32; ++w) woff += (w < warp) ? s_wsum[w] : 0u;
        bin_start[tid] = woff + incl - run;
    }
    __syncthreads();

    // ---- (4) place the records in tile-sorted order in shared memory
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {
        const u32 d = (u32)(key[i] >> shift) & mask;
        stage[bin_start[d] + wh[d] + rank[i]] = key[i];
    }

    // ---- (5) decoupled look-back, one thread per bin.  The tiles in flight finish their ranking at
    // about the same time, so the nearest inclusive prefix is usually many tiles back; LB_BATCH
    // predecessors are read at once (independent loads) so that the walk costs one L2 round trip per
    // batch instead of one per tile.
    if (tid < nbins) {
        u64 excl = 0;
        if (tile > 0) {
            i64 t = tile - 1;
            const u64* sp = status + t * nbins + tid; // status word of tile t and this bin; one tile back = -nbins words
            while (true) {
                // wait (one word, with a back-off) until the nearest tile not yet summed is published; the
                // tiles before it are older and almost always published already, so they are read as a batch
                u64 s0 = ld_volatile_u64(sp);
                while ((s0 >> 62) == 0) {
                    __nanosleep(40);
                    s0 = ld_volatile_u64(sp);
                }
                excl += s0 & LB_VALUE_MASK;
                sp -= nbins;
                --t;
                if ((s0 >> 62) == 2 || t < 0) break;
                if (t >= SORT_LB_BATCH) { // the whole batch lies at tiles >= 1: no bound checks inside
                    u64 sv[SORT_LB_BATCH];
                    const u64* q = sp;
#pragma unroll
                    for (int b = 0; b < SORT_LB_BATCH; ++b) {
                        sv[b] = ld_volatile_u64(q);
                        q -= nbins;
                    }
                    bool fin = false;
#pragma unroll
                    for (int b = 0; b < SORT_LB_BATCH; ++b) {
                        const u32 flag = (u32)(sv[b] >> 62);
                        if (flag == 0) break; // not published yet: wait for this tile
                        excl += sv[b] & LB_VALUE_MASK;
                        sp -= nbins;
                        --t;
                        if (flag == 2) { fin = true; break; }
                    }
                    if (fin) break;
                }
            }
            stress_jitter((u32)tile * 17u + (u32)tid);
            st_volatile_u64(status + tile * nbins + tid, LB_FLAG_INC | (excl + (u64)my_count));
        }
        goff[tid] = g_base + excl - (u64)bin_start[tid];
    }
    __syncthreads();

    // ---- (6) scatter: consecutive threads write consecutive slots of a bin's run
    if (count == SORT_TILE) {
#pragma unroll
        for (int i = 0; i < SORT_IPT; ++i) {
            const int p = tid + i * SORT_THREADS;
            const u64 k = stage[p];
            out[goff[(u32)(k >> shift) & mask] + (u64)p] = k;
        }
    } else {
        for (int p = tid; p < count; p += SORT_THREADS) {
            const u64 k = stage[p];
            out[goff[(u32)(k >> shift) & mask] + (u64)p] = k;
        }
    }
}

size_t pass_smem_bytes(int)
{
    const size_t nb = RIPS_SORT_MAX_BINS;
    return (size_t)SORT_TILE * 8 + nb * 8 + (size_t)SORT_WARPS * nb * 4 + nb * 4;
}

struct ScratchLayout {
    size_t hist_off, ticket_off, status_off[RIPS_SORT_MAX_PASSES], total;
};
ScratchLayout scratch_layout(i64 n, const SortPlan& plan)
{
    ScratchLayout L;
    L.hist_off = 0;
    size_t hist_bytes = (size_t)RIPS_SORT_MAX_PASSES * RIPS_SORT_MAX_BINS * 8;
    L.ticket_off = hist_bytes;
    i64 tiles = (n + SORT_TILE - 1) / SORT_TILE;
    if (tiles < 1) tiles = 1;
    size_t at = L.ticket_off + 256;
    for (int p = 0; p < RIPS_SORT_MAX_PASSES; ++p) { // every pass has its status words: one memset clears them all
        L.status_off[p] = at;
        if (p < plan.npasses) at += (size_t)tiles * ((size_t)1 << plan.bits[p]) * 8;
    }
    L.total = at;
    return L;
}

} // namespace

SortPlan sort_make_plan(int lo_bit, int hi_bit)
{
    SortPlan p;
    p.tile_items = SORT_TILE;
    int total = hi_bit - lo_bit;
    if (total < 1) total = 1;
    int np = (total + 7) / 8; // digits of at most 8 bits (RIPS_SORT_MAX_BINS = 256)
    if (np > RIPS_SORT_MAX_PASSES) np = RIPS_SORT_MAX_PASSES; // callers never ask for more than 64 bits
    p.npasses = np;
    // 8-bit digits from the bottom, the last one takes what is left: a producer kernel that accumulates the
    // histograms (FusedHist) then takes digit r of a field as byte r of it, with no shift or mask tables
    int at = lo_bit;
    for (int i = 0; i < np; ++i) {
        int w = (hi_bit - at) < 8 ? (hi_bit - at) : 8;
        if (w < 1) w = 1;
        p.shift[i] = at;
        p.bits[i] = w;
        at += w;
    }
    return p;
}

size_t sort_scratch_bytes(i64 n, const SortPlan& plan) { return scratch_layout(n, plan).total; }

u64* sort_hist_ptr(void* scratch) { return (u64*)scratch; }

// ---------------------------------------------------------------------------------------------------------------
// Static scratch for callers that cannot allocate (rips_sort_u64_static, include/rips.h): the sort's histograms,
// tickets and look-back status words in a file-scope device array instead of a cudaMalloc'ed buffer.  Every GPU that
// loads the library holds these RIPS_SORT_STATIC_BYTES until the process exits.  In HOST code the array's name is a
// host-side stand-in, not a device address: the address the kernels get comes from cudaGetSymbolAddress, asked once
// per device with that device current.  All calls share the array (it keeps the last call's contents: sort_u64 clears
// the histograms, the tickets and, before every pass, the status words it is about to use), so calls that overlap on
// the GPU race.
// ---------------------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_sort_static_scratch[RIPS_SORT_STATIC_BYTES];

cudaError_t sort_static_scratch(void** ptr, size_t* bytes)
{
    static std::mutex mu;
    static void* addr[RIPS_SORT_STATIC_MAX_DEVICES] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= RIPS_SORT_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_sort_static_scratch); // the current device's copy of the array
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        addr[dev] = p;
    }
    *ptr = addr[dev];
    *bytes = sizeof(g_sort_static_scratch);
    return cudaSuccess;
}

cudaError_t sort_prepare_fused(void* scratch, i64 n, const SortPlan& plan, cudaStream_t stream)
{
    return cudaMemsetAsync(scratch, 0, scratch_layout(n, plan).total, stream);
}

cudaError_t sort_u64(u64* a, u64* b, i64 n, const SortPlan& plan, void* scratch, cudaStream_t stream, u64** result,
                     SortTimes* times, i64* launches, bool hist_ready, u32 ballot_passes, const u64* n_dev)
{
    *result = a;
    int sms = 148;
    {
        int dev = 0;
        if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    }
    auto rec = [&](int i) {
        if (!times || !times->enabled) return;
        if (times->external) cudaEventRecordWithFlags(times->ev[i], stream, cudaEventRecordExternal);
        else cudaEventRecord(times->ev[i], stream);
    };
    rec(0);
    if (n <= 1) {
        rec(1);
        rec(2);
        return cudaSuccess;
    }
    {   // per call (cheap) rather than once per process: the attribute is per device
        cudaError_t e = cudaFuncSetAttribute(onesweep_pass_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pass_smem_bytes(8));
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(onesweep_pass_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pass_smem_bytes(8));
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(sort_histogram_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 RIPS_SORT_MAX_PASSES * RIPS_SORT_MAX_BINS * 4);
        if (e != cudaSuccess) return e;
    }
    const int pf_dist = sms; // tiles ahead of the L2 prefetch: one wave (swept 0 .. 12 waves in round 1)
    ScratchLayout L = scratch_layout(n, plan);
    unsigned char* sc = (unsigned char*)scratch;
    u64* hist = (u64*)(sc + L.hist_off);
    u32* ticket = (u32*)(sc + L.ticket_off);
    const i64 tiles = (n + SORT_TILE - 1) / SORT_TILE;

    cudaError_t e = cudaSuccess;
    if (!hist_ready) e = cudaMemsetAsync(sc, 0, L.total, stream); // histograms, tickets, status words of every pass (else sort_prepare_fused did it before the producer ran)
    if (e != cudaSuccess) return e;
    PlanDev pd;
    pd.npasses = plan.npasses;
    for (int p = 0; p < RIPS_SORT_MAX_PASSES; ++p) { pd.shift[p] = p < plan.npasses ? plan.shift[p] : 0; pd.bits[p] = p < plan.npasses ? plan.bits[p] : 1; }
    {
        i64 chunk = (i64)HIST_THREADS * HIST_IPT;
        i64 blocks = (n + chunk - 1) / chunk;
        if (blocks > (i64)sms * 4) blocks = (i64)sms * 4;
        if (!hist_ready) {
            sort_histogram_kernel<<<(unsigned)blocks, HIST_THREADS, plan.npasses * RIPS_SORT_MAX_BINS * 4, stream>>>(a, n, n_dev, pd, hist);
            if (launches) *launches += 1;
        }
    }
    rec(1);
    u64* src = a;
    u64* dst = b;
    for (int p = 0; p < plan.npasses; ++p) {
        if ((ballot_passes >> p) & 1u)
            onesweep_pass_kernel<true><<<(unsigned)tiles, SORT_THREADS, pass_smem_bytes(plan.bits[p]), stream>>>(
                src, dst, n, n_dev, plan.shift[p], plan.bits[p], hist + (size_t)p * RIPS_SORT_MAX_BINS, (u64*)(sc + L.status_off[p]), ticket + p, pf_dist);
        else
            onesweep_pass_kernel<false><<<(unsigned)tiles, SORT_THREADS, pass_smem_bytes(plan.bits[p]), stream>>>(
                src, dst, n, n_dev, plan.shift[p], plan.bits[p], hist + (size_t)p * RIPS_SORT_MAX_BINS, (u64*)(sc + L.status_off[p]), ticket + p, pf_dist);
        if (launches) *launches += 1;
        u64* t = src; src = dst; dst = t;
    }
    rec(2);
    *result = src;
    return cudaGetLastError();
}
