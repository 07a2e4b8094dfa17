// stage1.cu -- steps a3-a5: enumerate + diameter + threshold + clearing + ordered compaction.
// Algorithm 7 "filter-columns-kernel" and the count of Algorithm 8, redesigned:
// the paper launches one thread per candidate with a binary-search decode and leaves
// sentinels in place for the sort to sink.  Here a warp walks 32 consecutive indices at a time
// (lane = consecutive lowest vertex, so the reads of the key matrix are coalesced), each lane
// decodes once per tile (closed-form estimate + exact fix-up) and then steps with the colex
// successor; survivors are compacted in increasing index with a decoupled look-back, so only
// survivors are ever written or sorted; and the digit histogram of the sort that follows is
// accumulated on the way out, which spares that sort its own read of the records.
#include "kernels.cuh"

namespace {

constexpr int S1_THREADS = 256;
constexpr int S1_IPT = 16;
constexpr int S1_WARPS = S1_THREADS / 32;
constexpr int S1_WCHUNK = 32 * S1_IPT;        // candidates per warp per tile
constexpr int S1_TILE = S1_THREADS * S1_IPT;  // candidates per tile
constexpr int S1_BLOCKS_PER_SM = 5;

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
__device__ __forceinline__ u64 pack_vertices(const int (&v)[M], int vbits)
{
    u64 w = 0;
#pragma unroll
    for (int j = M - 1; j >= 0; --j) w = (w << vbits) | (u64)(u32)v[j];
    return w;
}

// min over the edges among v[lo..M-1] that touch v[lo] ... helpers for the cached upper keys
template <int M, typename KT>
__device__ __forceinline__ u32 upper_keys_from(const KT* __restrict__ Kf, int n, const int (&v)[M], int lo)
{ // min key+1 over all edges (a, b) with lo <= b < a < M
    u32 m = 0xffffffffu;
#pragma unroll
    for (int a = 1; a < M; ++a)
#pragma unroll
        for (int b = 0; b < a; ++b)
            if (b >= lo) m = min(m, (u32)__ldg(Kf + v[a] * n + v[b]));
    return m;
}

template <int M, typename KT>
__global__ void __launch_bounds__(S1_THREADS) stage1_kernel(const Stage1Params p)
{
    __shared__ u64 stage[S1_WARPS][S1_WCHUNK];
    __shared__ u32 s_hist[4][256];
    __shared__ u32 s_wcount[S1_WARPS];
    __shared__ u32 s_tile;
    __shared__ u64 s_tile_excl;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const KT* __restrict__ Kf = reinterpret_cast<const KT*>(p.Kf);
    const int n = p.n;
    const u32 lt_mask = (1u << lane) - 1u;
    const u32 thr1 = p.thr_key + 1u; // keys in Kf are shifted by one
    const bool fused = p.fh.hist != nullptr && p.out != nullptr;
    if (fused)
        for (int i = tid; i < 4 * 256; i += S1_THREADS) (&s_hist[0][0])[i] = 0;
    u64 n_over = 0, n_clr = 0;

    for (;;) {
        __syncthreads(); // previous tile's staging and s_tile are no longer in use
        if (tid == 0) s_tile = atomicAdd(p.ticket, 1u);
        __syncthreads();
        const i64 tile = s_tile;
        if (tile >= p.tiles) break;

        const u64 wbase = (u64)tile * S1_TILE + (u64)warp * S1_WCHUNK; // multiple of 32
        const u64 idx0 = wbase + lane;
        int iters = 0; // iterations in which this lane holds a real candidate
        if (idx0 < p.total) {
            u64 left = (p.total - idx0 + 31) >> 5;
            iters = left < (u64)S1_IPT ? (int)left : S1_IPT;
        }
        int v[M];
        u32 up1 = 0xffffffffu, up2 = 0xffffffffu; // min key+1 over edges among v[1..], among v[2..]
        u64 low = 0;
        if (iters > 0) {
            decode_simplex_fast<M>(p.bt, idx0, n, v);
            if (M > 2) up2 = upper_keys_from<M, KT>(Kf, n, v, 2);
            up1 = up2;
#pragma unroll
            for (int a = 2; a < M; ++a) up1 = min(up1, (u32)__ldg(Kf + v[a] * n + v[1]));
            low = pack_vertices<M>(v, p.vbits);
        } else {
#pragma unroll
            for (int j = 0; j < M; ++j) v[j] = j;
        }

        u32 wcount = 0;
#pragma unroll 1
        for (int it = 0; it < S1_IPT; ++it) {
            bool keep = false;
            u32 key1 = 0;
            if (it < iters) {
                key1 = up1;
#pragma unroll
                for (int j = 1; j < M; ++j) key1 = min(key1, (u32)__ldg(Kf + v[j] * n + v[0]));
                if (key1 >= thr1) {
                    bool clr;
                    const u64 idx = idx0 + (u64)it * 32;
                    if (p.clear.bitmap) clr = (__ldg(p.clear.bitmap + (idx >> 5)) >> lane) & 1u; // idx & 31 == lane
                    else
                        clr = in_sorted(p.clear.layer1, p.clear.n1, p.clear.shift1, idx) ||
                              in_sorted(p.clear.layer2, p.clear.n2, 0, idx);
                    keep = !clr;
                    n_clr += clr;
                } else
                    ++n_over;
            }
            const u32 bal = __ballot_sync(RIPS_FULL_MASK, keep);
            if (keep) {
                const u64 rec = ((u64)(key1 - 1u) << p.lowbits) | low;
                stage[warp][wcount + __popc(bal & lt_mask)] = rec;
                if (fused) {
#pragma unroll
                    for (int q = 0; q < 4; ++q)
                        if (q < p.fh.npasses)
                            atomicAdd(&s_hist[q][(u32)(rec >> p.fh.shift[q]) & ((1u << p.fh.bits[q]) - 1u)], 1u);
                }
            }
            wcount += __popc(bal);

            // ---- colex successor, 32 steps at once
            if (it + 1 < iters) {
                v[0] += 32;
                low += 32;
                if (v[0] >= v[1]) {
                    bool upper = false;
                    do {
                        v[0] -= v[1];
                        v[1] += 1;
                        if (M > 2) {
                            if (v[1] == v[M > 2 ? 2 : 1]) { // carry into the upper vertices (rare)
                                upper = true;
                                v[1] = 1;
#pragma unroll
                                for (int j = 2; j < M; ++j) {
                                    v[j] += 1;
                                    if (j + 1 < M && v[j] == v[j + 1 < M ? j + 1 : j]) v[j] = j;
                                    else break;
                                }
                            }
                        }
                    } while (v[0] >= v[1]);
                    if (M > 2 && upper) up2 = upper_keys_from<M, KT>(Kf, n, v, 2);
                    up1 = up2;
#pragma unroll
                    for (int a = 2; a < M; ++a) up1 = min(up1, (u32)__ldg(Kf + v[a] * n + v[1]));
                    low = pack_vertices<M>(v, p.vbits);
                }
            }
        }

        // ---- ordered compaction
        if (lane == 0) s_wcount[warp] = wcount;
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
            continue;
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
        for (u32 i = lane; i < wcount; i += 32) __stcs(dst + i, stage[warp][i]);
    }

    // ---- counters and the fused histogram: once per block
    n_over = warp_sum_u64(n_over);
    n_clr = warp_sum_u64(n_clr);
    if (lane == 0) {
        if (n_over) atomicAdd((unsigned long long*)&p.counters[1], (unsigned long long)n_over);
        if (n_clr) atomicAdd((unsigned long long*)&p.counters[2], (unsigned long long)n_clr);
    }
    if (fused) {
        // the loop's closing __syncthreads has made every shared atomic visible
        for (int i = tid; i < p.fh.npasses * 256; i += S1_THREADS) {
            u32 c = (&s_hist[0][0])[i];
            if (c) atomicAdd((unsigned long long*)&p.fh.hist[i], (unsigned long long)c);
        }
    }
}

__global__ void clear_bitmap_kernel(u32* bitmap, const u64* __restrict__ rows, i64 n_rows, int shift)
{
    i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_rows) {
        u64 t = __ldg(rows + i) >> shift;
        atomicOr(bitmap + (t >> 5), 1u << (t & 31));
    }
}

template <int M, typename KT>
cudaError_t launch_stage1_t(const Stage1Params& p, cudaStream_t st)
{
    i64 g = p.tiles < (i64)148 * S1_BLOCKS_PER_SM ? p.tiles : (i64)148 * S1_BLOCKS_PER_SM;
    stage1_kernel<M, KT><<<(unsigned)g, S1_THREADS, 0, st>>>(p);
    return cudaGetLastError();
}

} // namespace

i64 stage1_tiles(u64 total) { return (i64)((total + S1_TILE - 1) / S1_TILE); }

cudaError_t launch_stage1(int M, int kf_u16, const Stage1Params& p, cudaStream_t st)
{
    if (p.tiles == 0) return cudaSuccess;
    if (p.tiles > 0x7fffffffLL) return cudaErrorInvalidValue;
#define S1_CASE(MM)                                                                          \
    case MM: return kf_u16 ? launch_stage1_t<MM, unsigned short>(p, st) : launch_stage1_t<MM, u32>(p, st);
    switch (M) {
        S1_CASE(2) S1_CASE(3) S1_CASE(4) S1_CASE(5) S1_CASE(6)
    default: return cudaErrorInvalidValue;
    }
#undef S1_CASE
}

cudaError_t launch_clear_bitmap(u32* bitmap, const u64* rows, i64 n_rows, int shift, cudaStream_t st)
{
    if (n_rows == 0) return cudaSuccess;
    i64 blocks = (n_rows + 255) / 256;
    clear_bitmap_kernel<<<(unsigned)blocks, 256, 0, st>>>(bitmap, rows, n_rows, shift);
    return cudaGetLastError();
}
