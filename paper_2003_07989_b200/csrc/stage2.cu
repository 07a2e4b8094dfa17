// stage2.cu -- the pair store (steps a8-a10) and the unpack kernels behind the C ABI's accessors.
//
// The apparent test itself (a7) runs inside the fused kernel of stage1.cu.  What stage 2 does on
// the device is: one stable partition of the pair slots by the cofacet vertex v (radix_sort.cu),
// after which the REGULAR pairs are sorted by cidx(t) (apparent.cuh); full sorts of the two small
// lists the fused kernel appended out of order (irregular pairs by cidx(t), non-apparent columns
// by (key, vertices) = coboundary order).  The pair store then has
// three sorted layers, each looked up by binary search:
//   regular    (v << tbits) | cidx(t)      s = t minus its top vertex v:  cidx(s) = cidx(t) - C(v, M+1)
//   irregular  (cidx(t) << 3) | j          s = t minus its vertex at position j
//   reduced    t[], s[]                    pivots found by the reduction of the non-apparent columns
#include "kernels.cuh"

namespace {

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

__device__ __forceinline__ i64 lower_bound_field_in(const u64* __restrict__ a, i64 lo, i64 hi, int shift, u64 mask, u64 x)
{
    while (lo < hi) {
        i64 mid = lo + ((hi - lo) >> 1);
        if (((__ldg(a + mid) >> shift) & mask) < x) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ i64 lower_bound_field(const u64* __restrict__ a, i64 n, int shift, u64 mask, u64 x)
{
    i64 lo = 0, hi = n;
    while (lo < hi) {
        i64 mid = lo + ((hi - lo) >> 1);
        if (((__ldg(a + mid) >> shift) & mask) < x) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

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

// Apparent pairs ascending by t: merge of the regular and the irregular layer.  Rows are distinct,
// so element i of one layer lands at i + #{rows of the other layer below it}.
constexpr int MA_THREADS = 256, MA_ITEMS = 8; // rows per block: MA_THREADS * MA_ITEMS
template <int M>
__global__ void __launch_bounds__(MA_THREADS) merge_apparent_kernel(PairLayers L, BinomTable bt, int n, u64* __restrict__ t, u64* __restrict__ s)
{
    const u64 tmask = (L.tbits >= 64) ? ~0ull : ((1ull << L.tbits) - 1ull);
    const i64 b0 = (i64)blockIdx.x * (MA_THREADS * MA_ITEMS);
    // the regular rows of a block are ascending, so their places in the irregular layer lie between those of the
    // block's first and last row: two searches through the whole layer per block of 2048 rows (their ~20 dependent
    // loads each were the kernel's run time when every row, and then every 256 rows, made them), the others through
    // that window
    __shared__ i64 s_win[2];
    if (b0 < L.n_reg && (threadIdx.x == 0 || threadIdx.x == 32)) {
        const i64 b1 = (b0 + MA_THREADS * MA_ITEMS - 1 < L.n_reg) ? b0 + MA_THREADS * MA_ITEMS - 1 : L.n_reg - 1;
        const u64 tb = __ldg(L.reg + (threadIdx.x == 0 ? b0 : b1)) & tmask;
        s_win[threadIdx.x == 0 ? 0 : 1] = lower_bound_field(L.irr, L.n_irr, RIPS_PAIR_POS_BITS, ~0ull, tb);
    }
    __syncthreads();
#pragma unroll 4
    for (int it = 0; it < MA_ITEMS; ++it) {
        const i64 i = b0 + (i64)it * MA_THREADS + threadIdx.x;
        if (i < L.n_reg) {
            const u64 r = __ldg(L.reg + i);
            const u64 tt = r & tmask;
            const int v = (int)(r >> L.tbits);
            const i64 pos = i + lower_bound_field_in(L.irr, s_win[0], s_win[1], RIPS_PAIR_POS_BITS, ~0ull, tt);
            t[pos] = tt;
            s[pos] = tt - bt(v, M + 1);
        } else if (i < L.n_reg + L.n_irr) {
            const i64 k = i - L.n_reg;
            const u64 r = __ldg(L.irr + k);
            const u64 tt = r >> RIPS_PAIR_POS_BITS;
            const i64 pos = k + lower_bound_field(L.reg, L.n_reg, 0, tmask, tt);
            t[pos] = tt;
            s[pos] = pair_s_of<M>(bt, n, r);
        }
    }
}

// merge of two (t, s) arrays with distinct t, both ascending (the first one the long one: the same windowed search
// as merge_apparent_kernel)
__global__ void __launch_bounds__(MA_THREADS) merge_ts_kernel(const u64* __restrict__ t1, const u64* __restrict__ s1, i64 n1,
                                                            const u64* __restrict__ t2, const u64* __restrict__ s2, i64 n2,
                                                            u64* __restrict__ t, u64* __restrict__ s)
{
    const i64 b0 = (i64)blockIdx.x * (MA_THREADS * MA_ITEMS);
    __shared__ i64 s_win[2];
    if (b0 < n1 && (threadIdx.x == 0 || threadIdx.x == 32)) {
        const i64 b1 = (b0 + MA_THREADS * MA_ITEMS - 1 < n1) ? b0 + MA_THREADS * MA_ITEMS - 1 : n1 - 1;
        s_win[threadIdx.x == 0 ? 0 : 1] = lower_bound_field(t2, n2, 0, ~0ull, __ldg(t1 + (threadIdx.x == 0 ? b0 : b1)));
    }
    __syncthreads();
#pragma unroll 4
    for (int it = 0; it < MA_ITEMS; ++it) {
        const i64 i = b0 + (i64)it * MA_THREADS + threadIdx.x;
        if (i < n1) {
            const u64 tt = __ldg(t1 + i);
            const i64 pos = i + lower_bound_field_in(t2, s_win[0], s_win[1], 0, ~0ull, tt);
            t[pos] = tt;
            s[pos] = __ldg(s1 + i);
        } else if (i < n1 + n2) {
            const i64 k = i - n1;
            const u64 tt = __ldg(t2 + k);
            const i64 pos = k + lower_bound_field(t1, n1, 0, ~0ull, tt);
            t[pos] = tt;
            s[pos] = __ldg(s2 + k);
        }
    }
}

// a10: lookup through the layers
template <int M>
__global__ void pivot_lookup_kernel(PairLayers L, BinomTable bt, int n, const u64* __restrict__ red_t,
                                    const u64* __restrict__ red_s, i64 n2, const u64* __restrict__ query, i64 m,
                                    i64* __restrict__ s_out)
{
    i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= m) return;
    const u64 q = __ldg(query + i);
    const u64 tmask = (L.tbits >= 64) ? ~0ull : ((1ull << L.tbits) - 1ull);
    i64 r = -1;
    i64 p1 = lower_bound_field(L.reg, L.n_reg, 0, tmask, q);
    if (p1 < L.n_reg && (__ldg(L.reg + p1) & tmask) == q) {
        r = (i64)(q - bt((int)(__ldg(L.reg + p1) >> L.tbits), M + 1));
    } else {
        i64 p2 = lower_bound_field(L.irr, L.n_irr, RIPS_PAIR_POS_BITS, ~0ull, q);
        if (p2 < L.n_irr && (__ldg(L.irr + p2) >> RIPS_PAIR_POS_BITS) == q) r = (i64)pair_s_of<M>(bt, n, __ldg(L.irr + p2));
        else {
            i64 p3 = lower_bound_field(red_t, n2, 0, ~0ull, q);
            if (p3 < n2 && __ldg(red_t + p3) == q) r = (i64)__ldg(red_s + p3);
        }
    }
    s_out[i] = r;
}

} // namespace

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

cudaError_t launch_unpack_columns(int M, const u64* cols, i64 len, int vbits, BinomTable bt, const float* values,
                                  float* diam, u64* cidx, cudaStream_t st)
{
    if (len == 0) return cudaSuccess;
    unsigned g = (unsigned)((len + 255) / 256);
    RIPS_DISPATCH_M(M, (unpack_columns_kernel<MM><<<g, 256, 0, st>>>(cols, len, vbits, bt, values, diam, cidx)));
    return cudaGetLastError();
}

cudaError_t launch_merge_apparent(int M, const PairLayers& L, BinomTable bt, int n, u64* t, u64* s, cudaStream_t st)
{
    const i64 tot = L.n_reg + L.n_irr;
    if (tot == 0) return cudaSuccess;
    unsigned g = (unsigned)((tot + MA_THREADS * MA_ITEMS - 1) / (MA_THREADS * MA_ITEMS));
    RIPS_DISPATCH_M(M, (merge_apparent_kernel<MM><<<g, MA_THREADS, 0, st>>>(L, bt, n, t, s)));
    return cudaGetLastError();
}

cudaError_t launch_merge_ts(const u64* t1, const u64* s1, i64 n1, const u64* t2, const u64* s2, i64 n2, u64* t, u64* s,
                            cudaStream_t st)
{
    if (n1 + n2 == 0) return cudaSuccess;
    unsigned g = (unsigned)((n1 + n2 + MA_THREADS * MA_ITEMS - 1) / (MA_THREADS * MA_ITEMS));
    merge_ts_kernel<<<g, MA_THREADS, 0, st>>>(t1, s1, n1, t2, s2, n2, t, s);
    return cudaGetLastError();
}

cudaError_t launch_pivot_lookup(int M, const PairLayers& L, BinomTable bt, int n, const u64* red_t, const u64* red_s,
                                i64 n2, const u64* query, i64 m, i64* s_out, cudaStream_t st)
{
    if (m == 0) return cudaSuccess;
    unsigned g = (unsigned)((m + 255) / 256);
    RIPS_DISPATCH_M(M, (pivot_lookup_kernel<MM><<<g, 256, 0, st>>>(L, bt, n, red_t, red_s, n2, query, m, s_out)));
    return cudaGetLastError();
}
