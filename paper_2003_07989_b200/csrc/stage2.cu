// stage2.cu -- steps a7-a8 (+ the unpack / merge / lookup kernels of a10).
// Algorithm 3 "finding apparent pairs" via the Apparent Pairs Lemma
// (Lemma 7): for a column s, scan the cofacets t = s + {v} for v = n-1 .. 0
// (decreasing cidx, Remark 2 PAPER.md:95); the first with diam(t) = diam(s) is the oldest cofacet;
// (s,t) is apparent iff no facet of t that precedes s in increasing-cidx order (Algorithm 6,
// PAPER.md:439-469) has the same diameter.  The facets of t that precede s are exactly those that
// drop a vertex w of s with w > v, so no facet index is ever computed.
// Diameters are compared as dense ranks ("keys", see common.cuh): equality of keys is equality of
// the fp32 diameters.
#include "kernels.cuh"

namespace {

constexpr int S2_THREADS = 256;
constexpr int S2_IPT = 4;
constexpr int S2_WARPS = S2_THREADS / 32;
constexpr int S2_WCHUNK = 32 * S2_IPT;
constexpr int S2_TILE = S2_THREADS * S2_IPT;

// One column.  Returns 0 = not apparent, 1 = apparent (then *pair = packed pair record).
template <int M>
__device__ __forceinline__ int apparent_column(const u32* __restrict__ K, const BinomTable& bt, int n, u32 key_s, u64 cidx_s,
                                               u64* pair)
{
    int s[M];
    u32 row[M];
    decode_simplex<M>(bt, cidx_s, n, s);
#pragma unroll
    for (int j = 0; j < M; ++j) row[j] = (u32)s[j] * (u32)(s[j] - 1) >> 1;

    int fv = -1, fseg = 0;
    // segments of the scan: seg = number of vertices of s below v
#pragma unroll
    for (int seg = M; seg >= 0; --seg) {
        if (fv < 0) {
            const int hi = (seg == M) ? n - 1 : s[seg < M ? seg : 0] - 1;
            const int lo = (seg == 0) ? 0 : s[seg > 0 ? seg - 1 : 0] + 1;
            for (int v = hi; v >= lo; --v) {
                const u32 rv = (u32)v * (u32)(v - 1) >> 1;
                bool ok = true;
#pragma unroll
                for (int j = 0; j < M; ++j) {
                    if (ok) {
                        const u32 kk = (j >= seg) ? __ldg(K + row[j] + v) : __ldg(K + rv + s[j]);
                        ok = kk >= key_s;
                    }
                }
                if (ok) { fv = v; fseg = seg; break; }
            }
        }
    }
    if (fv < 0) return 0;

    // facets of t that come before s in increasing cidx: drop w = s[j], j >= fseg (w > v)
    bool apparent = true;
    if (fseg < M) {
        u32 vk[M];
        const u32 rv = (u32)fv * (u32)(fv - 1) >> 1;
#pragma unroll
        for (int a = 0; a < M; ++a) vk[a] = (a >= fseg) ? __ldg(K + row[a] + fv) : __ldg(K + rv + s[a]);
        u32 pk[M][M];
#pragma unroll
        for (int a = 1; a < M; ++a)
#pragma unroll
            for (int b = 0; b < a; ++b) pk[a][b] = __ldg(K + row[a] + s[b]);
#pragma unroll
        for (int j = 0; j < M; ++j) {
            if (j >= fseg) {
                u32 mn = 0xffffffffu;
#pragma unroll
                for (int a = 0; a < M; ++a) {
                    if (a != j) {
                        mn = min(mn, vk[a]);
#pragma unroll
                        for (int b = 0; b < a; ++b)
                            if (b != j) mn = min(mn, pk[a][b]);
                    }
                }
                if (mn == key_s) apparent = false;
            }
        }
    }
    if (!apparent) return 0;
    u64 t = bt(fv, fseg + 1);
#pragma unroll
    for (int i = 0; i < M; ++i) t += (i < fseg) ? bt(s[i], i + 1) : bt(s[i], i + 2);
    *pair = (t << RIPS_PAIR_POS_BITS) | (u64)fseg;
    return 1;
}

template <int M>
__global__ void __launch_bounds__(S2_THREADS) stage2_kernel(const Stage2Params p)
{
    __shared__ u64 st_app[S2_WARPS][S2_WCHUNK];
    __shared__ u64 st_non[S2_WARPS][S2_WCHUNK];
    __shared__ u32 s_wapp[S2_WARPS], s_wnon[S2_WARPS];
    __shared__ u32 s_tile;
    __shared__ u64 s_excl_app, s_excl_non;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(p.ticket, 1u);
    __syncthreads();
    const i64 tile = s_tile;
    const u32 lt_mask = (1u << lane) - 1u;
    const u64 cmask = (p.cbits >= 64) ? ~0ull : ((1ull << p.cbits) - 1ull);

    u32 capp = 0, cnon = 0;
    i64 ci = tile * S2_TILE + (i64)warp * S2_WCHUNK + lane;
#pragma unroll 1
    for (int it = 0; it < S2_IPT; ++it, ci += 32) {
        int res = -1;
        u64 rec = 0, pair = 0;
        if (ci < p.len) {
            rec = __ldg(p.cols + ci);
            res = apparent_column<M>(p.K, p.bt, p.n, (u32)(rec >> p.cbits), rec & cmask, &pair);
        }
        const u32 ba = __ballot_sync(RIPS_FULL_MASK, res == 1);
        const u32 bn = __ballot_sync(RIPS_FULL_MASK, res == 0);
        if (res == 1) st_app[warp][capp + __popc(ba & lt_mask)] = pair;
        if (res == 0) st_non[warp][cnon + __popc(bn & lt_mask)] = rec;
        capp += __popc(ba);
        cnon += __popc(bn);
    }
    if (lane == 0) { s_wapp[warp] = capp; s_wnon[warp] = cnon; }
    __syncthreads();
    u32 ea = 0, en = 0, ta = 0, tn = 0;
#pragma unroll
    for (int w = 0; w < S2_WARPS; ++w) {
        u32 a = s_wapp[w], b = s_wnon[w];
        if (w < warp) { ea += a; en += b; }
        ta += a;
        tn += b;
    }
    if (warp == 0) {
        u64 e = lookback_exclusive(p.status_app, tile, (u64)ta);
        if (lane == 0) { s_excl_app = e; if (ta) atomicAdd((unsigned long long*)&p.counters[0], (unsigned long long)ta); }
    } else if (warp == 1) {
        u64 e = lookback_exclusive(p.status_non, tile, (u64)tn);
        if (lane == 0) { s_excl_non = e; if (tn) atomicAdd((unsigned long long*)&p.counters[1], (unsigned long long)tn); }
    }
    __syncthreads();
    u64* da = p.app_out + s_excl_app + ea;
    for (u32 i = lane; i < capp; i += 32) da[i] = st_app[warp][i];
    u64* dn = p.non_out + s_excl_non + en;
    for (u32 i = lane; i < cnon; i += 32) dn[i] = st_non[warp][i];
}

// ---------------------------------------------------------------------------------------------
// Unpack kernels: the packed records are the library's working form; the C ABI exposes the
// paper's (diameter, cidx) and (t, s) arrays, produced here on demand.
// ---------------------------------------------------------------------------------------------
__global__ void unpack_columns_kernel(const u64* __restrict__ cols, i64 len, int cbits, const float* __restrict__ values,
                                      float* __restrict__ diam, u64* __restrict__ cidx)
{
    i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= len) return;
    const u64 cmask = (1ull << cbits) - 1ull;
    u64 r = __ldg(cols + i);
    diam[i] = __ldg(values + (r >> cbits));
    cidx[i] = r & cmask;
}

// s = t minus its vertex at position j (M = vertices of s, t has M+1)
template <int M>
__device__ __forceinline__ u64 pair_s_of(const BinomTable& bt, int n, u64 rec)
{
    int tv[M + 1];
    const int j = (int)(rec & ((1u << RIPS_PAIR_POS_BITS) - 1u));
    decode_simplex<M + 1>(bt, rec >> RIPS_PAIR_POS_BITS, n, tv);
    u64 s = 0;
#pragma unroll
    for (int i = 0; i <= M; ++i) {
        if (i < j) s += bt(tv[i], i + 1);
        else if (i > j) s += bt(tv[i], i);
    }
    return s;
}

template <int M>
__global__ void unpack_pairs_kernel(const u64* __restrict__ pairs, i64 len, BinomTable bt, int n, u64* __restrict__ t,
                                    u64* __restrict__ s)
{
    i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= len) return;
    u64 r = __ldg(pairs + i);
    t[i] = r >> RIPS_PAIR_POS_BITS;
    s[i] = pair_s_of<M>(bt, n, r);
}

__device__ __forceinline__ i64 lower_bound_shifted(const u64* __restrict__ a, i64 n, int shift, u64 x)
{
    i64 lo = 0, hi = n;
    while (lo < hi) {
        i64 mid = lo + ((hi - lo) >> 1);
        if ((__ldg(a + mid) >> shift) < x) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

// Merge of layer 1 (packed apparent pairs, ascending t) and layer 2 (reduced pivots, ascending t):
// the rows are distinct, so element i of layer 1 lands at i + #{layer-2 rows below it} and vice versa.
template <int M>
__global__ void merge_pivots_kernel(const u64* __restrict__ pairs, i64 n1, BinomTable bt, int n, const u64* __restrict__ red_t,
                                    const u64* __restrict__ red_s, i64 n2, u64* __restrict__ t, u64* __restrict__ s)
{
    i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n1) {
        u64 r = __ldg(pairs + i);
        u64 tt = r >> RIPS_PAIR_POS_BITS;
        i64 pos = i + lower_bound_shifted(red_t, n2, 0, tt);
        t[pos] = tt;
        s[pos] = pair_s_of<M>(bt, n, r);
    } else if (i < n1 + n2) {
        i64 k = i - n1;
        u64 tt = __ldg(red_t + k);
        i64 pos = k + lower_bound_shifted(pairs, n1, RIPS_PAIR_POS_BITS, tt);
        t[pos] = tt;
        s[pos] = __ldg(red_s + k);
    }
}

// a10: two-layer lookup: binary search of the sorted apparent array, then of the
// (small, sorted) array of pivots found by the reduction.
template <int M>
__global__ void pivot_lookup_kernel(const u64* __restrict__ pairs, i64 n1, BinomTable bt, int n, const u64* __restrict__ red_t,
                                    const u64* __restrict__ red_s, i64 n2, const u64* __restrict__ query, i64 m,
                                    i64* __restrict__ s_out)
{
    i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    const u64 q = __ldg(query + i);
    i64 r = -1;
    i64 p1 = lower_bound_shifted(pairs, n1, RIPS_PAIR_POS_BITS, q);
    if (p1 < n1 && (__ldg(pairs + p1) >> RIPS_PAIR_POS_BITS) == q) r = (i64)pair_s_of<M>(bt, n, __ldg(pairs + p1));
    else {
        i64 p2 = lower_bound_shifted(red_t, n2, 0, q);
        if (p2 < n2 && __ldg(red_t + p2) == q) r = (i64)__ldg(red_s + p2);
    }
    s_out[i] = r;
}

} // namespace

i64 stage2_tiles(i64 len) { return (len + S2_TILE - 1) / S2_TILE; }

#define RIPS_DISPATCH_M(M, CALL)                      \
    switch (M) {                                      \
    case 1: { constexpr int MM = 1; CALL; } break;    \
    case 2: { constexpr int MM = 2; CALL; } break;    \
    case 3: { constexpr int MM = 3; CALL; } break;    \
    case 4: { constexpr int MM = 4; CALL; } break;    \
    case 5: { constexpr int MM = 5; CALL; } break;    \
    case 6: { constexpr int MM = 6; CALL; } break;    \
    default: return cudaErrorInvalidValue;            \
    }

cudaError_t launch_stage2(int M, const Stage2Params& p, cudaStream_t st)
{
    i64 tiles = stage2_tiles(p.len);
    if (tiles == 0) return cudaSuccess;
    if (M < 2) return cudaErrorInvalidValue;
    unsigned g = (unsigned)tiles;
    RIPS_DISPATCH_M(M, (stage2_kernel<(MM < 2 ? 2 : MM)><<<g, S2_THREADS, 0, st>>>(p)));
    return cudaGetLastError();
}

cudaError_t launch_unpack_columns(const u64* cols, i64 len, int cbits, const float* values, float* diam, u64* cidx,
                                  cudaStream_t st)
{
    if (len == 0) return cudaSuccess;
    unpack_columns_kernel<<<(unsigned)((len + 255) / 256), 256, 0, st>>>(cols, len, cbits, values, diam, cidx);
    return cudaGetLastError();
}

cudaError_t launch_unpack_pairs(int M, const u64* pairs, i64 len, BinomTable bt, int n, u64* t, u64* s, cudaStream_t st)
{
    if (len == 0) return cudaSuccess;
    unsigned g = (unsigned)((len + 255) / 256);
    RIPS_DISPATCH_M(M, (unpack_pairs_kernel<MM><<<g, 256, 0, st>>>(pairs, len, bt, n, t, s)));
    return cudaGetLastError();
}

cudaError_t launch_merge_pivots(int M, const u64* pairs, i64 n1, BinomTable bt, int n, const u64* red_t, const u64* red_s,
                                i64 n2, u64* t, u64* s, cudaStream_t st)
{
    if (n1 + n2 == 0) return cudaSuccess;
    unsigned g = (unsigned)((n1 + n2 + 255) / 256);
    RIPS_DISPATCH_M(M, (merge_pivots_kernel<MM><<<g, 256, 0, st>>>(pairs, n1, bt, n, red_t, red_s, n2, t, s)));
    return cudaGetLastError();
}

cudaError_t launch_pivot_lookup(int M, const u64* pairs, i64 n1, BinomTable bt, int n, const u64* red_t, const u64* red_s,
                                i64 n2, const u64* query, i64 m, i64* s_out, cudaStream_t st)
{
    if (m == 0) return cudaSuccess;
    unsigned g = (unsigned)((m + 255) / 256);
    RIPS_DISPATCH_M(M, (pivot_lookup_kernel<MM><<<g, 256, 0, st>>>(pairs, n1, bt, n, red_t, red_s, n2, query, m, s_out)));
    return cudaGetLastError();
}
