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

constexpr int S2_THREADS = 512;
constexpr int S2_BLOCKS_PER_SM = 2;

// One column.  `rec` = packed column record.  Returns the packed pair record if the column is
// apparent, else ~0.  Kf and B may live in shared or in global memory (generic pointers).
template <int M, typename KT>
__device__ __forceinline__ u64 apparent_column(const KT* Kf, const u64* B, int bstride, int n, int vbits, int lowbits, u64 rec)
{
    const u32 key_s1 = (u32)(rec >> lowbits) + 1u; // Kf holds key+1
    const u32 vmask = (1u << vbits) - 1u;
    int s[M];
    const KT* row[M];
#pragma unroll
    for (int j = 0; j < M; ++j) {
        s[j] = (int)((u32)(rec >> (j * vbits)) & vmask);
        row[j] = Kf + s[j] * n;
    }
    // scan of the cofacets s + {v}, v = n-1 .. 0 (decreasing cidx): the first whose new edges all have
    // key >= key(s) has diam(t) = diam(s) and is the oldest such cofacet.  v in s reads the zero
    // diagonal and fails by itself.
    int v = n - 1;
    for (; v >= 1; v -= 2) {
        u32 m0 = 0xffffffffu, m1 = 0xffffffffu;
#pragma unroll
        for (int j = 0; j < M; ++j) {
            m0 = min(m0, (u32)row[j][v]);
            m1 = min(m1, (u32)row[j][v - 1]);
        }
        if (m0 >= key_s1) break;
        if (m1 >= key_s1) { v -= 1; break; }
    }
    if (v == 0) { // n odd leaves vertex 0 to the pair loop's tail
        u32 m0 = 0xffffffffu;
#pragma unroll
        for (int j = 0; j < M; ++j) m0 = min(m0, (u32)row[j][0]);
        if (m0 < key_s1) v = -1;
    }
    if (v < 0) return ~0ull;

    // facets of t that precede s in increasing cidx (Algorithm 6) are those dropping a vertex w of s
    // with w > v; s is the youngest facet iff none of them has the diameter of s
    int fseg = 0;
#pragma unroll
    for (int j = 0; j < M; ++j) fseg += (s[j] < v) ? 1 : 0;
    if (fseg < M) {
        u32 vk[M];
#pragma unroll
        for (int a = 0; a < M; ++a) vk[a] = (u32)row[a][v];
        u32 pk[M][M];
#pragma unroll
        for (int a = 1; a < M; ++a)
#pragma unroll
            for (int b = 0; b < a; ++b) pk[a][b] = (u32)row[a][s[b]];
        bool apparent = true;
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
                if (mn == key_s1) apparent = false;
            }
        }
        if (!apparent) return ~0ull;
    }
    u64 t = B[(fseg + 1) * bstride + v];
#pragma unroll
    for (int i = 0; i < M; ++i) t += B[((i < fseg) ? i + 1 : i + 2) * bstride + s[i]];
    return (t << RIPS_PAIR_POS_BITS) | (u64)fseg;
}

// a7: a pure map over the columns.  Column i writes its pair record to app_out[i], or the sentinel
// (rows << 3, rows = C(n, d+2), larger than every real row index) when it is not apparent, and the
// warp writes one word of the non-apparent bitmap.  The pair sort then sinks the few sentinels to
// the end (the paper's own device, used here where ~99 % survive), and
// compact_nonapparent_kernel gathers the non-apparent columns in coboundary order from the bitmap.
template <int M, typename KT>
__global__ void __launch_bounds__(S2_THREADS, S2_BLOCKS_PER_SM) stage2_kernel(const Stage2Params p, int k_in_smem, int b_in_smem,
                                                                              u64 sentinel, u32* __restrict__ nonmask)
{
    extern __shared__ __align__(16) unsigned char smem2[];
    const int tid = threadIdx.x, lane = tid & 31;
    const int n = p.n, bstride = p.bt.stride;
    size_t off = 0;
    const u64* B = p.bt.B;
    if (b_in_smem) {
        u64* sb = reinterpret_cast<u64*>(smem2);
        const int cnt = (p.kmax + 1) * bstride;
        for (int i = tid; i < cnt; i += S2_THREADS) sb[i] = __ldg(p.bt.B + i);
        B = sb;
        off = ((size_t)cnt * 8 + 15) & ~(size_t)15;
    }
    const KT* Kf = reinterpret_cast<const KT*>(p.Kf);
    if (k_in_smem) {
        KT* sk = reinterpret_cast<KT*>(smem2 + off);
        const uint4* src = reinterpret_cast<const uint4*>(p.Kf);
        const int cnt16 = (int)(((size_t)n * n * sizeof(KT) + 15) / 16); // the buffer is padded to 16 bytes
        uint4* dst = reinterpret_cast<uint4*>(sk);
        for (int i = tid; i < cnt16; i += S2_THREADS) dst[i] = __ldg(src + i);
        Kf = sk;
    }
    __syncthreads();

    u64 n_app = 0;
    const i64 stride = (i64)gridDim.x * S2_THREADS;
    // whole warps stay in the loop so the ballot is complete; len is padded per warp
    for (i64 ci = (i64)blockIdx.x * S2_THREADS + tid; (ci - lane) < p.len; ci += stride) {
        u64 pair = ~0ull;
        const bool valid = ci < p.len;
        if (valid) {
            const u64 rec = __ldcs(p.cols + ci);
            pair = apparent_column<M, KT>(Kf, B, bstride, n, p.vbits, p.lowbits, rec);
        }
        const bool is_app = pair != ~0ull;
        const u32 bal_non = __ballot_sync(RIPS_FULL_MASK, valid && !is_app);
        if (valid) {
            p.app_out[ci] = is_app ? pair : sentinel;
            n_app += is_app;
        }
        if (lane == 0) nonmask[ci >> 5] = bal_non;
    }
    n_app = warp_sum_u64(n_app);
    if (lane == 0 && n_app) atomicAdd((unsigned long long*)&p.counters[0], (unsigned long long)n_app);
}

// a8: the non-apparent columns in coboundary order from the bitmap stage2_kernel
// wrote: single-pass scan of the popcounts with a decoupled look-back, then an ordered gather.
constexpr int CN_THREADS = 256;
constexpr int CN_WPT = 8;                       // bitmap words per thread
constexpr int CN_TILE = CN_THREADS * CN_WPT;    // words per tile

__global__ void __launch_bounds__(CN_THREADS) compact_nonapparent_kernel(const u32* __restrict__ nonmask, i64 n_words,
                                                                         const u64* __restrict__ cols, u64* __restrict__ non_out,
                                                                         u64* status, u32* ticket, u64* counter)
{
    __shared__ u32 s_wsum[CN_THREADS / 32];
    __shared__ u32 s_tile;
    __shared__ u64 s_excl;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const i64 tile = s_tile;
    const i64 w0 = tile * CN_TILE + (i64)tid * CN_WPT; // blocked: thread owns CN_WPT consecutive words
    u32 word[CN_WPT];
    u32 cnt = 0;
#pragma unroll
    for (int i = 0; i < CN_WPT; ++i) {
        word[i] = (w0 + i < n_words) ? __ldg(nonmask + w0 + i) : 0u;
        cnt += __popc(word[i]);
    }
    u32 incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        u32 t = __shfl_up_sync(RIPS_FULL_MASK, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_wsum[warp] = incl;
    __syncthreads();
    u32 wexcl = 0, ttotal = 0;
#pragma unroll
    for (int w = 0; w < CN_THREADS / 32; ++w) {
        u32 c = s_wsum[w];
        if (w < warp) wexcl += c;
        ttotal += c;
    }
    if (warp == 0) {
        u64 e = lookback_exclusive(status, tile, (u64)ttotal);
        if (lane == 0) {
            s_excl = e;
            if (ttotal) atomicAdd((unsigned long long*)counter, (unsigned long long)ttotal);
        }
    }
    __syncthreads();
    u64 pos = s_excl + wexcl + (incl - cnt);
#pragma unroll
    for (int i = 0; i < CN_WPT; ++i) {
        u32 w = word[i];
        while (w) {
            const int b = __ffs(w) - 1;
            w &= w - 1;
            non_out[pos++] = __ldg(cols + ((w0 + i) << 5) + b);
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Unpack kernels: the packed records are the library's working form; the C ABI exposes the
// paper's (diameter, cidx) and (t, s) arrays, produced here on demand.
// ---------------------------------------------------------------------------------------------
template <int M>
__global__ void unpack_columns_kernel(const u64* __restrict__ cols, i64 len, int vbits, BinomTable bt,
                                      const float* __restrict__ values, float* __restrict__ diam, u64* __restrict__ cidx)
{
    i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= len) return;
    const u32 vmask = (1u << vbits) - 1u;
    u64 r = __ldg(cols + i);
    diam[i] = __ldg(values + (r >> (M * vbits)));
    u64 c = 0;
#pragma unroll
    for (int j = 0; j < M; ++j) c += bt((int)((u32)(r >> (j * vbits)) & vmask), j + 1); // Eq. 2
    cidx[i] = c;
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

i64 stage2_tiles(i64 len) { return (len + CN_TILE * 32 - 1) / ((i64)CN_TILE * 32); } // tiles of the compaction

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

namespace {
template <int M, typename KT>
cudaError_t launch_stage2_t(const Stage2Params& p, u64 sentinel, u32* nonmask, cudaStream_t st)
{
    // shared memory: binomial table and key matrix when they fit (two blocks per SM)
    const size_t budget = 110 * 1024;
    const size_t bbytes = (((size_t)(p.kmax + 1) * p.bt.stride * 8) + 15) & ~(size_t)15;
    const size_t kbytes = (((size_t)p.n * p.n * sizeof(KT)) + 15) & ~(size_t)15;
    const int b_in = bbytes <= 48 * 1024;
    const int k_in = (b_in ? bbytes : 0) + kbytes <= budget;
    const size_t smem = (b_in ? bbytes : 0) + (k_in ? kbytes : 0);
    cudaError_t e = cudaFuncSetAttribute(stage2_kernel<M, KT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)budget);
    if (e != cudaSuccess) return e;
    i64 blocks = (p.len + S2_THREADS - 1) / S2_THREADS;
    const i64 cap = (i64)148 * S2_BLOCKS_PER_SM;
    if (blocks > cap) blocks = cap;
    stage2_kernel<M, KT><<<(unsigned)blocks, S2_THREADS, smem, st>>>(p, k_in, b_in, sentinel, nonmask);
    return cudaGetLastError();
}
} // namespace

cudaError_t launch_stage2(int M, int kf_u16, const Stage2Params& p, u64 sentinel, u32* nonmask, cudaStream_t st)
{
    if (p.len == 0) return cudaSuccess;
    if (M < 2) return cudaErrorInvalidValue;
    cudaError_t e = cudaErrorInvalidValue;
    if (kf_u16) { RIPS_DISPATCH_M(M, (e = launch_stage2_t<(MM < 2 ? 2 : MM), unsigned short>(p, sentinel, nonmask, st))); }
    else { RIPS_DISPATCH_M(M, (e = launch_stage2_t<(MM < 2 ? 2 : MM), u32>(p, sentinel, nonmask, st))); }
    return e;
}

cudaError_t launch_compact_nonapparent(const u32* nonmask, i64 len, const u64* cols, u64* non_out, u64* status, u32* ticket,
                                       u64* counter, cudaStream_t st)
{
    if (len == 0) return cudaSuccess;
    const i64 n_words = (len + 31) / 32;
    const i64 tiles = (n_words + CN_TILE - 1) / CN_TILE;
    compact_nonapparent_kernel<<<(unsigned)tiles, CN_THREADS, 0, st>>>(nonmask, n_words, cols, non_out, status, ticket, counter);
    return cudaGetLastError();
}

cudaError_t launch_unpack_columns(int M, const u64* cols, i64 len, int vbits, BinomTable bt, const float* values,
                                  float* diam, u64* cidx, cudaStream_t st)
{
    if (len == 0) return cudaSuccess;
    unsigned g = (unsigned)((len + 255) / 256);
    RIPS_DISPATCH_M(M, (unpack_columns_kernel<MM><<<g, 256, 0, st>>>(cols, len, vbits, bt, values, diam, cidx)));
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
