// stage1.cu -- steps a3-a5: enumerate + diameter + threshold + clearing + ordered compaction.
// Algorithm 7 "filter-columns-kernel" and the count of Algorithm 8, redesigned:
// the paper launches one thread per candidate with a binary-search decode and leaves
// sentinels in place for the sort to sink; here a warp walks 32 consecutive indices at a time
// (lane = lowest vertex, so the reads of the distance keys are coalesced and the upper vertices
// are warp-uniform), decodes once per lane per tile and then steps with the colex successor, and
// survivors are compacted in increasing index with a decoupled look-back, so only survivors are
// ever written or sorted.
#include "kernels.cuh"

namespace {

constexpr int S1_THREADS = 256;
constexpr int S1_IPT = 16;
constexpr int S1_WARPS = S1_THREADS / 32;
constexpr int S1_WCHUNK = 32 * S1_IPT;        // candidates per warp per tile
constexpr int S1_TILE = S1_THREADS * S1_IPT;  // candidates per tile

__device__ __forceinline__ bool in_sorted(const u64* __restrict__ a, i64 n, int shift, u64 x)
{
    i64 lo = 0, hi = n;
    while (lo < hi) {
        i64 mid = lo + ((hi - lo) >> 1);
        if ((__ldg(a + mid) >> shift) < x) lo = mid + 1;
        else hi = mid;
    }
    return lo < n && (__ldg(a + lo) >> shift) == x;
}

template <int M>
__global__ void __launch_bounds__(S1_THREADS) stage1_kernel(const Stage1Params p)
{
    __shared__ u64 stage[S1_WARPS][S1_WCHUNK];
    __shared__ u32 s_wcount[S1_WARPS];
    __shared__ u32 s_tile;
    __shared__ u64 s_tile_excl;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(p.ticket, 1u);
    __syncthreads();
    const i64 tile = s_tile;
    const u32* __restrict__ K = p.K;
    const u32 lt_mask = (1u << lane) - 1u;

    u64 idx = (u64)tile * S1_TILE + (u64)warp * S1_WCHUNK + lane;
    int v[M];
    u32 row[M]; // row[j] = v[j](v[j]-1)/2 for j >= 1
    u32 uk1 = 0xffffffffu, uk2 = 0xffffffffu;
    if (idx < p.total) {
        decode_simplex<M>(p.bt, idx, p.n, v);
#pragma unroll
        for (int j = 1; j < M; ++j) row[j] = (u32)v[j] * (u32)(v[j] - 1) >> 1;
#pragma unroll
        for (int a = 3; a < M; ++a)
#pragma unroll
            for (int b = 2; b < a; ++b) uk2 = min(uk2, __ldg(K + row[a] + v[b]));
        uk1 = uk2;
#pragma unroll
        for (int a = 2; a < M; ++a) uk1 = min(uk1, __ldg(K + row[a] + v[1]));
    } else {
#pragma unroll
        for (int j = 0; j < M; ++j) { v[j] = j; row[j] = 0; }
    }

    u32 wcount = 0, n_over = 0, n_clr = 0;
#pragma unroll 1
    for (int it = 0; it < S1_IPT; ++it) {
        bool keep = false;
        u32 key = 0;
        if (idx < p.total) {
            key = uk1;
#pragma unroll
            for (int j = 1; j < M; ++j) key = min(key, __ldg(K + row[j] + v[0]));
            if (key >= p.thr_key) {
                bool clr;
                if (p.clear.bitmap) clr = (__ldg(p.clear.bitmap + (idx >> 5)) >> (idx & 31)) & 1u;
                else
                    clr = in_sorted(p.clear.layer1, p.clear.n1, p.clear.shift1, idx) ||
                          in_sorted(p.clear.layer2, p.clear.n2, 0, idx);
                keep = !clr;
                n_clr += clr;
            } else
                ++n_over;
        }
        const u32 bal = __ballot_sync(RIPS_FULL_MASK, keep);
        if (keep) stage[warp][wcount + __popc(bal & lt_mask)] = ((u64)key << p.cbits) | idx;
        wcount += __popc(bal);

        // ---- colex successor, 32 steps at once
        idx += 32;
        if (idx < p.total) {
            v[0] += 32;
            int maxlvl = 0;
            while (v[0] >= v[1]) {
                v[0] -= v[1];
                bool done = false;
#pragma unroll
                for (int j = 1; j < M; ++j) {
                    if (!done) {
                        bool blocked = false;
                        if (j < M - 1) blocked = (v[j] + 1 == v[j + 1]);
                        if (blocked) v[j] = j;
                        else { v[j] += 1; done = true; maxlvl = max(maxlvl, j); }
                    }
                }
            }
            if (maxlvl > 0) {
#pragma unroll
                for (int j = 1; j < M; ++j) row[j] = (u32)v[j] * (u32)(v[j] - 1) >> 1;
                if (maxlvl >= 2) {
                    uk2 = 0xffffffffu;
#pragma unroll
                    for (int a = 3; a < M; ++a)
#pragma unroll
                        for (int b = 2; b < a; ++b) uk2 = min(uk2, __ldg(K + row[a] + v[b]));
                }
                uk1 = uk2;
#pragma unroll
                for (int a = 2; a < M; ++a) uk1 = min(uk1, __ldg(K + row[a] + v[1]));
            }
        }
    }

    // ---- counters (one atomic per warp and counter)
    n_over = warp_sum_u32(n_over);
    n_clr = warp_sum_u32(n_clr);
    if (lane == 0) {
        s_wcount[warp] = wcount;
        if (n_over) atomicAdd((unsigned long long*)&p.counters[1], (unsigned long long)n_over);
        if (n_clr) atomicAdd((unsigned long long*)&p.counters[2], (unsigned long long)n_clr);
    }
    __syncthreads();
    u32 wexcl = 0, ttotal = 0;
#pragma unroll
    for (int w = 0; w < S1_WARPS; ++w) {
        u32 c = s_wcount[w];
        if (w < warp) wexcl += c;
        ttotal += c;
    }
    if (p.out == nullptr) { // count-only pass
        if (tid == 0 && ttotal) atomicAdd((unsigned long long*)&p.counters[0], (unsigned long long)ttotal);
        return;
    }
    if (warp == 0) {
        u64 excl = lookback_exclusive(p.status, tile, (u64)ttotal);
        if (lane == 0) {
            s_tile_excl = excl;
            if (ttotal) atomicAdd((unsigned long long*)&p.counters[0], (unsigned long long)ttotal);
        }
    }
    __syncthreads();
    u64* dst = p.out + s_tile_excl + wexcl;
    for (u32 i = lane; i < wcount; i += 32) dst[i] = stage[warp][i];
}

__global__ void clear_bitmap_kernel(u32* bitmap, const u64* __restrict__ rows, i64 n_rows, int shift)
{
    i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_rows) {
        u64 t = __ldg(rows + i) >> shift;
        atomicOr(bitmap + (t >> 5), 1u << (t & 31));
    }
}

} // namespace

i64 stage1_tiles(u64 total) { return (i64)((total + S1_TILE - 1) / S1_TILE); }

cudaError_t launch_stage1(int M, const Stage1Params& p, cudaStream_t st)
{
    i64 tiles = stage1_tiles(p.total);
    if (tiles == 0) return cudaSuccess;
    if (tiles > 0x7fffffffLL) return cudaErrorInvalidValue;
    unsigned g = (unsigned)tiles;
    switch (M) {
    case 2: stage1_kernel<2><<<g, S1_THREADS, 0, st>>>(p); break;
    case 3: stage1_kernel<3><<<g, S1_THREADS, 0, st>>>(p); break;
    case 4: stage1_kernel<4><<<g, S1_THREADS, 0, st>>>(p); break;
    case 5: stage1_kernel<5><<<g, S1_THREADS, 0, st>>>(p); break;
    case 6: stage1_kernel<6><<<g, S1_THREADS, 0, st>>>(p); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_clear_bitmap(u32* bitmap, const u64* rows, i64 n_rows, int shift, cudaStream_t st)
{
    if (n_rows == 0) return cudaSuccess;
    i64 blocks = (n_rows + 255) / 256;
    clear_bitmap_kernel<<<(unsigned)blocks, 256, 0, st>>>(bitmap, rows, n_rows, shift);
    return cudaGetLastError();
}
