// stage1.cu -- steps a3-a5: enumerate + diameter + threshold + clearing + ordered compaction.
// Algorithm 7 "filter-columns-kernel" and the count of Algorithm 8, redesigned:
// the paper launches one thread per candidate with a binary-search decode and leaves
// sentinels in place for the sort to sink.  Here a warp walks a chunk of consecutive indices row by
// row (see the kernel), decodes once per chunk (closed-form estimate + exact fix-up), survivors
// are compacted in increasing index with a decoupled look-back, so only survivors are ever written
// or sorted, and the digit histogram of the sort that follows is accumulated on the way out, which
// spares that sort its own read of the records.
#include "kernels.cuh"

namespace {

constexpr int S1_THREADS = 256;
constexpr int S1_WARPS = S1_THREADS / 32;
constexpr int S1_CHUNK = 512;                 // candidates per warp chunk = unit of the look-back chain
constexpr int S1_BLOCKS_PER_SM = 6;
constexpr int S1_MAX_FUSED = 3;               // digits of the following sort histogrammed on the way out

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

// A warp owns a chunk of S1_CHUNK consecutive combinatorial indices and walks it row by row: a
// row fixes the vertices v[M-1] > ... > v[1] (warp-uniform: their mutual keys, the row pointers
// into Kf and the upper part of the record are computed once per row) and the lanes take
// consecutive lowest vertices v[0], so every read of the key matrix is coalesced and no lane
// ever carries on its own.  The warp's survivors are staged in shared memory in index order and
// written out after a warp-level decoupled look-back over the chunks (no block-wide barrier).
template <int M, typename KT>
__global__ void __launch_bounds__(S1_THREADS) stage1_kernel(const Stage1Params p)
{
    __shared__ u64 stage[S1_WARPS][S1_CHUNK];
    __shared__ u32 s_hist[S1_MAX_FUSED][256];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const KT* __restrict__ Kf = reinterpret_cast<const KT*>(p.Kf);
    const int n = p.n, vbits = p.vbits, lowbits = p.lowbits;
    const u32 lt_mask = (1u << lane) - 1u;
    const u32 thr1 = p.thr_key + 1u; // keys in Kf are shifted by one
    const bool write = p.out != nullptr;
    const int nfused = (write && p.fh.hist != nullptr) ? p.fh.npasses : 0;
    int fsh[S1_MAX_FUSED];
    u32 fmk[S1_MAX_FUSED];
#pragma unroll
    for (int q = 0; q < S1_MAX_FUSED; ++q) {
        fsh[q] = q < nfused ? p.fh.shift[q] : 0;
        fmk[q] = q < nfused ? (1u << p.fh.bits[q]) - 1u : 0u;
    }
    if (nfused) {
        for (int i = tid; i < S1_MAX_FUSED * 256; i += S1_THREADS) (&s_hist[0][0])[i] = 0;
        __syncthreads();
    }
    u32 n_over = 0, n_clr = 0;
    u64 n_kept = 0;
    u64* const wstage = stage[warp];

    for (;;) {
        u32 chunk = 0;
        if (lane == 0) chunk = atomicAdd(p.ticket, 1u);
        chunk = __shfl_sync(RIPS_FULL_MASK, chunk, 0);
        if ((i64)chunk >= p.tiles) break;

        u64 idx = (u64)chunk * S1_CHUNK;
        int rem = (p.total - idx) < (u64)S1_CHUNK ? (int)(p.total - idx) : S1_CHUNK;
        int v[M];
        decode_simplex_fast<M>(p.bt, idx, n, v); // warp-uniform
        int v0 = v[0];
        u32 wcount = 0;
        bool new_upper = true;
        u32 up2 = 0xffffffffu;

        while (rem > 0) {
            // ---- per row: keys among v[1..M-1], upper part of the record
            if (M > 2 && new_upper) {
                up2 = 0xffffffffu;
#pragma unroll
                for (int a = 3; a < M; ++a)
#pragma unroll
                    for (int b = 2; b < a; ++b) up2 = min(up2, (u32)__ldg(Kf + v[a] * n + v[b]));
                new_upper = false;
            }
            u32 up1 = up2;
#pragma unroll
            for (int a = 2; a < M; ++a) up1 = min(up1, (u32)__ldg(Kf + v[a] * n + v[1]));
            u64 lowbase = 0;
#pragma unroll
            for (int j = M - 1; j >= 1; --j) lowbase = (lowbase << vbits) | (u64)(u32)v[j];
            lowbase <<= vbits;
            const int row_len = min(v[1] - v0, rem);

            for (int off = lane; off - lane < row_len; off += 32) {
                const bool valid = off < row_len;
                const int x = v0 + off;
                bool keep = false;
                u32 key1 = up1;
                if (valid) {
#pragma unroll
                    for (int j = 1; j < M; ++j) key1 = min(key1, (u32)__ldg(Kf + v[j] * n + x));
                    if (key1 >= thr1) {
                        const u64 ci = idx + (u64)off;
                        bool clr;
                        if (p.clear.bitmap) clr = (__ldg(p.clear.bitmap + (ci >> 5)) >> (ci & 31)) & 1u;
                        else
                            clr = in_sorted(p.clear.layer1, p.clear.n1, p.clear.shift1, ci) ||
                                  in_sorted(p.clear.layer2, p.clear.n2, 0, ci);
                        keep = !clr;
                        n_clr += clr;
                    } else
                        ++n_over;
                }
                const u32 bal = __ballot_sync(RIPS_FULL_MASK, keep);
                if (keep && write) {
                    const u64 rec = ((u64)(key1 - 1u) << lowbits) | lowbase | (u64)(u32)x;
                    wstage[wcount + __popc(bal & lt_mask)] = rec;
#pragma unroll
                    for (int q = 0; q < S1_MAX_FUSED; ++q)
                        if (q < nfused) atomicAdd(&s_hist[q][(u32)(rec >> fsh[q]) & fmk[q]], 1u);
                }
                wcount += __popc(bal);
            }
            idx += (u64)row_len;
            rem -= row_len;
            // ---- next row (colex successor of (v[M-1..1]))
            v0 = 0;
            v[1] += 1;
            if (M > 2) {
                if (v[1] == v[M > 2 ? 2 : 1]) {
                    new_upper = true;
                    v[1] = 1;
#pragma unroll
                    for (int j = 2; j < M; ++j) {
                        v[j] += 1;
                        if (j + 1 < M && v[j] == v[j + 1 < M ? j + 1 : j]) v[j] = j;
                        else break;
                    }
                }
            }
        }

        n_kept += wcount;
        if (!write) continue; // count-only pass
        // ---- ordered compaction: warp-level look-back over the chunks
        const u64 excl = lookback_exclusive(p.status, (i64)chunk, (u64)wcount);
        __syncwarp();
        u64* dst = p.out + excl;
        for (u32 i = lane; i < wcount; i += 32) __stcs(dst + i, wstage[i]);
        __syncwarp();
    }

    // ---- counters and the fused histogram: once per block
    n_over = warp_sum_u32(n_over);
    n_clr = warp_sum_u32(n_clr);
    if (lane == 0) {
        if (n_kept) atomicAdd((unsigned long long*)&p.counters[0], (unsigned long long)n_kept);
        if (n_over) atomicAdd((unsigned long long*)&p.counters[1], (unsigned long long)n_over);
        if (n_clr) atomicAdd((unsigned long long*)&p.counters[2], (unsigned long long)n_clr);
    }
    if (nfused) {
        __syncthreads();
        for (int i = tid; i < nfused * 256; i += S1_THREADS) {
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
    i64 g = (p.tiles + S1_WARPS - 1) / S1_WARPS;
    if (g > (i64)148 * S1_BLOCKS_PER_SM) g = (i64)148 * S1_BLOCKS_PER_SM;
    stage1_kernel<M, KT><<<(unsigned)g, S1_THREADS, 0, st>>>(p);
    return cudaGetLastError();
}

} // namespace

i64 stage1_tiles(u64 total) { return (i64)((total + S1_CHUNK - 1) / S1_CHUNK); } // warp chunks

cudaError_t launch_stage1(int M, int kf_u16, const Stage1Params& p, cudaStream_t st)
{
    if (p.tiles == 0) return cudaSuccess;
    if (p.tiles > 0xffffffffLL) return cudaErrorInvalidValue;
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
