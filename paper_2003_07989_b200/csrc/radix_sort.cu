// radix_sort.cu -- onesweep LSD radix sort of 64-bit records on a bit range, written by hand for
// sm_100a (no CUB/Thrust).  One histogram kernel over all digits, then one kernel per digit that
// ranks a tile in shared memory, resolves its global offsets with a decoupled look-back chained
// scan over (tile, bin) status words, and scatters coalesced runs.  Stable, so records that enter
// in increasing combinatorial index leave each pass in increasing index within equal digits: the
// index bits never have to be sorted.
#include "radix_sort.cuh"

namespace {

constexpr int SORT_THREADS = 512;
constexpr int SORT_IPT = 16;
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

__global__ void __launch_bounds__(HIST_THREADS) sort_histogram_kernel(const u64* __restrict__ in, i64 n, PlanDev plan,
                                                                      u64* __restrict__ hist)
{
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

// Exclusive scan over the bins of each digit, in place: hist[p][b] = number of records whose
// digit p is smaller than b.  One block per pass.
__global__ void sort_scan_bins_kernel(u64* hist)
{
    __shared__ u64 s[RIPS_SORT_MAX_BINS];
    u64* h = hist + (size_t)blockIdx.x * RIPS_SORT_MAX_BINS;
    for (int i = threadIdx.x; i < RIPS_SORT_MAX_BINS; i += blockDim.x) s[i] = h[i];
    __syncthreads();
    if (threadIdx.x == 0) {
        u64 run = 0;
        for (int i = 0; i < RIPS_SORT_MAX_BINS; ++i) { u64 c = s[i]; s[i] = run; run += c; }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < RIPS_SORT_MAX_BINS; i += blockDim.x) h[i] = s[i];
}

// ----------------------------------------------------------------------------------------------
// One onesweep pass.
// ----------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(SORT_THREADS) onesweep_pass_kernel(const u64* __restrict__ in, u64* __restrict__ out, i64 n,
                                                                    int shift, int bits, const u64* __restrict__ global_base,
                                                                    u64* status, u32* ticket)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int nbins = 1 << bits;
    const u32 mask = (u32)nbins - 1u;
    u64* stage = reinterpret_cast<u64*>(smem_raw);                       // [SORT_TILE]
    u64* goff = stage + SORT_TILE;                                        // [nbins]
    u32* whist = reinterpret_cast<u32*>(goff + nbins);                    // [SORT_WARPS][nbins]
    u32* bin_start = whist + SORT_WARPS * nbins;                          // [nbins]
    u32* bin_count = bin_start + nbins;                                   // [nbins] valid records per bin
    __shared__ u32 s_tile;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    for (int i = tid; i < SORT_WARPS * nbins; i += SORT_THREADS) whist[i] = 0;
    __syncthreads();
    const i64 tile = s_tile;
    const i64 base = tile * SORT_TILE;
    const int count = (int)min((i64)SORT_TILE, n - base);

    // ---- load, warp-striped: item i of lane l of warp w is record base + w*32*IPT + i*32 + l
    u64 key[SORT_IPT];
    const i64 wbase = base + (i64)warp * (32 * SORT_IPT) + lane;
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {
        i64 idx = wbase + i * 32;
        key[i] = idx < n ? __ldg(in + idx) : ~0ull; // padding sorts last inside the tile and is never written
    }

    // ---- rank inside the warp: records with the same digit are found with one ballot per bit
    u32 rank[SORT_IPT];
    u32* wh = whist + warp * nbins;
    const u32 lt_mask = (1u << lane) - 1u;
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {
        const u32 d = (u32)(key[i] >> shift) & mask;
        u32 peers = RIPS_FULL_MASK;
        for (int b = 0; b < bits; ++b) {
            const bool bit = (d >> b) & 1u;
            const u32 bal = __ballot_sync(RIPS_FULL_MASK, bit);
            peers &= bit ? bal : ~bal;
        }
        const int leader = __ffs(peers) - 1;
        u32 old = 0;
        if (lane == leader) old = wh[d];
        old = __shfl_sync(RIPS_FULL_MASK, old, leader);
        if (lane == leader) wh[d] = old + __popc(peers);
        rank[i] = old + __popc(peers & lt_mask);
        __syncwarp();
    }
    __syncthreads();

    // ---- per bin: exclusive scan over the warps; publish the tile's count for the look-back
    const int n_pad = SORT_TILE - count;
    for (int b = tid; b < nbins; b += SORT_THREADS) {
        u32 run = 0;
#pragma unroll
        for (int w = 0; w < SORT_WARPS; ++w) {
            u32 c = whist[w * nbins + b];
            whist[w * nbins + b] = run;
            run += c;
        }
        bin_start[b] = run; // padded count for now; scanned below
        u32 valid = (b == nbins - 1) ? run - (u32)n_pad : run;
        bin_count[b] = valid;
        st_volatile_u64(status + tile * nbins + b, (tile == 0 ? LB_FLAG_INC : LB_FLAG_AGG) | (u64)valid);
    }
    __syncthreads();

    // ---- exclusive scan over the bins (warp 0): bin_start[b] = first slot of bin b in the tile
    if (warp == 0) {
        const int per = nbins >> 5; // nbins is a power of two >= 32 (bits >= 5 enforced by the plan) or handled below
        if (per >= 1) {
            u32 sum = 0;
            for (int j = 0; j < per; ++j) sum += bin_start[lane * per + j];
            u32 incl = sum;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                u32 t = __shfl_up_sync(RIPS_FULL_MASK, incl, o);
                if (lane >= o) incl += t;
            }
            u32 run = incl - sum;
            for (int j = 0; j < per; ++j) {
                u32 c = bin_start[lane * per + j];
                bin_start[lane * per + j] = run;
                run += c;
            }
        } else if (lane == 0) {
            u32 run = 0;
            for (int j = 0; j < nbins; ++j) { u32 c = bin_start[j]; bin_start[j] = run; run += c; }
        }
    }
    __syncthreads();

    // ---- place the records in tile-sorted order in shared memory
#pragma unroll
    for (int i = 0; i < SORT_IPT; ++i) {
        const u32 d = (u32)(key[i] >> shift) & mask;
        stage[bin_start[d] + wh[d] + rank[i]] = key[i];
    }

    // ---- decoupled look-back, one thread per bin
    for (int b = tid; b < nbins; b += SORT_THREADS) {
        u64 excl = 0;
        if (tile > 0) {
            i64 t = tile - 1;
            for (;;) {
                u64 s = ld_volatile_u64(status + t * nbins + b);
                u64 flag = s >> 62;
                if (flag == 0) continue;
                excl += s & LB_VALUE_MASK;
                if (flag == 2) break;
                --t;
            }
            st_volatile_u64(status + tile * nbins + b, LB_FLAG_INC | (excl + (u64)bin_count[b]));
        }
        goff[b] = __ldg(global_base + b) + excl - (u64)bin_start[b];
    }
    __syncthreads();

    // ---- scatter: consecutive threads write consecutive slots of a bin's run
    for (int p = tid; p < count; p += SORT_THREADS) {
        const u64 k = stage[p];
        const u32 d = (u32)(k >> shift) & mask;
        out[goff[d] + (u64)p] = k;
    }
}

size_t pass_smem_bytes(int bits)
{
    size_t nbins = (size_t)1 << bits;
    return (size_t)SORT_TILE * 8 + nbins * 8 + (size_t)SORT_WARPS * nbins * 4 + nbins * 4 * 2;
}

struct ScratchLayout {
    size_t hist_off, ticket_off, status_off, total;
};
ScratchLayout scratch_layout(i64 n, const SortPlan& plan)
{
    ScratchLayout L;
    L.hist_off = 0;
    size_t hist_bytes = (size_t)RIPS_SORT_MAX_PASSES * RIPS_SORT_MAX_BINS * 8;
    L.ticket_off = hist_bytes;
    L.status_off = L.ticket_off + 256;
    int maxbits = 1;
    for (int p = 0; p < plan.npasses; ++p) maxbits = plan.bits[p] > maxbits ? plan.bits[p] : maxbits;
    i64 tiles = (n + SORT_TILE - 1) / SORT_TILE;
    if (tiles < 1) tiles = 1;
    L.total = L.status_off + (size_t)tiles * ((size_t)1 << maxbits) * 8;
    return L;
}

} // namespace

SortPlan sort_make_plan(int lo_bit, int hi_bit)
{
    SortPlan p;
    p.tile_items = SORT_TILE;
    int total = hi_bit - lo_bit;
    if (total < 1) total = 1;
    int p8 = (total + 7) / 8, p9 = (total + 8) / 9;
    int np = p9 < p8 ? p9 : p8;
    if (np > RIPS_SORT_MAX_PASSES) np = RIPS_SORT_MAX_PASSES; // callers never ask for more than 64 bits
    p.npasses = np;
    int basew = total / np, extra = total % np, at = lo_bit;
    for (int i = 0; i < np; ++i) {
        int w = basew + (i < extra ? 1 : 0);
        p.shift[i] = at;
        p.bits[i] = w;
        at += w;
    }
    return p;
}

size_t sort_scratch_bytes(i64 n, const SortPlan& plan) { return scratch_layout(n, plan).total; }

cudaError_t sort_u64(u64* a, u64* b, i64 n, const SortPlan& plan, void* scratch, cudaStream_t stream, u64** result,
                     SortTimes* times, i64* launches)
{
    *result = a;
    if (times && times->enabled) cudaEventRecord(times->ev[0], stream);
    if (n <= 1) {
        if (times && times->enabled) { cudaEventRecord(times->ev[1], stream); cudaEventRecord(times->ev[2], stream); }
        return cudaSuccess;
    }
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(onesweep_pass_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                             (int)pass_smem_bytes(9));
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(sort_histogram_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 RIPS_SORT_MAX_PASSES * RIPS_SORT_MAX_BINS * 4);
        if (e != cudaSuccess) return e;
        attr_set = true;
    }
    ScratchLayout L = scratch_layout(n, plan);
    unsigned char* sc = (unsigned char*)scratch;
    u64* hist = (u64*)(sc + L.hist_off);
    u32* ticket = (u32*)(sc + L.ticket_off);
    u64* status = (u64*)(sc + L.status_off);
    const i64 tiles = (n + SORT_TILE - 1) / SORT_TILE;

    cudaError_t e = cudaMemsetAsync(sc, 0, L.status_off, stream);
    if (e != cudaSuccess) return e;
    PlanDev pd;
    pd.npasses = plan.npasses;
    for (int p = 0; p < RIPS_SORT_MAX_PASSES; ++p) { pd.shift[p] = p < plan.npasses ? plan.shift[p] : 0; pd.bits[p] = p < plan.npasses ? plan.bits[p] : 1; }
    {
        i64 chunk = (i64)HIST_THREADS * HIST_IPT;
        i64 blocks = (n + chunk - 1) / chunk;
        if (blocks > 148 * 4) blocks = 148 * 4;
        sort_histogram_kernel<<<(unsigned)blocks, HIST_THREADS, plan.npasses * RIPS_SORT_MAX_BINS * 4, stream>>>(a, n, pd, hist);
        sort_scan_bins_kernel<<<plan.npasses, 256, 0, stream>>>(hist);
        if (launches) *launches += 2;
    }
    if (times && times->enabled) cudaEventRecord(times->ev[1], stream);
    u64* src = a;
    u64* dst = b;
    for (int p = 0; p < plan.npasses; ++p) {
        size_t status_bytes = (size_t)tiles * ((size_t)1 << plan.bits[p]) * 8;
        e = cudaMemsetAsync(status, 0, status_bytes, stream);
        if (e != cudaSuccess) return e;
        onesweep_pass_kernel<<<(unsigned)tiles, SORT_THREADS, pass_smem_bytes(plan.bits[p]), stream>>>(
            src, dst, n, plan.shift[p], plan.bits[p], hist + (size_t)p * RIPS_SORT_MAX_BINS, status, ticket + p);
        if (launches) *launches += 1;
        u64* t = src; src = dst; dst = t;
    }
    if (times && times->enabled) cudaEventRecord(times->ev[2], stream);
    *result = src;
    return cudaGetLastError();
}
