// common.cuh -- shared device/host helpers of the CUDA path (sm_100a only).
// Nothing here is shared with oracle/ (the oracle is plain C and has its own everything).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

typedef uint64_t u64;
typedef uint32_t u32;
typedef int64_t i64;

#define RIPS_FULL_MASK 0xffffffffu

// ---------------------------------------------------------------------------------------------
// Decoupled look-back (single-pass chained scan).  One 64-bit word per tile: flag in the top two
// bits (0 = not ready, 1 = tile aggregate, 2 = inclusive prefix), value in the low 62 bits, so flag
// and value are published by one store and need no fence between them.
// ---------------------------------------------------------------------------------------------
#define LB_FLAG_AGG (1ull << 62)
#define LB_FLAG_INC (2ull << 62)
#define LB_VALUE_MASK ((1ull << 62) - 1)

__device__ __forceinline__ u64 ld_volatile_u64(const u64* p)
{
    u64 v;
    asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_volatile_u64(u64* p, u64 v)
{
    asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Stress build (-DRIPS_STRESS, paper_2003_07989_b200/build.py build_stress): tiny tiles and pseudo-random delays in
// front of every publication of a chained scan and of the lock-free reduction, so that the orders in which tiles and
// columns publish are shuffled far beyond what a normal run produces (compute-sanitizer is not available on the pool).
#ifdef RIPS_STRESS
__device__ __forceinline__ void stress_jitter(u32 salt)
{
    u32 h = (salt * 2654435761u + blockIdx.x * 2246822519u + (u32)clock64()) * 3266489917u;
    __nanosleep((h >> 21) & 2047u);
}
#else
__device__ __forceinline__ void stress_jitter(u32) {}
#endif

__device__ __forceinline__ u64 warp_sum_u64(u64 v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(RIPS_FULL_MASK, v, o);
    return v;
}
__device__ __forceinline__ u32 warp_sum_u32(u32 v)
{
    return __reduce_add_sync(RIPS_FULL_MASK, v);
}

// Called by ONE full warp of the block.  Publishes this tile's aggregate, walks back over the
// predecessors 32 at a time and returns the exclusive prefix (sum of the aggregates of tiles
// 0..tile-1); then publishes the inclusive prefix.  Tiles must be numbered in the order they
// start (ticket counter), so every predecessor is resident or finished.
__device__ __forceinline__ u64 lookback_exclusive(u64* status, i64 tile, u64 aggregate)
{
    const int lane = threadIdx.x & 31;
    if (tile == 0) {
        if (lane == 0) st_volatile_u64(status, LB_FLAG_INC | aggregate);
        return 0;
    }
    stress_jitter((u32)tile);
    if (lane == 0) st_volatile_u64(status + tile, LB_FLAG_AGG | aggregate);
    u64 excl = 0;
    i64 look = tile - 1;
    for (;;) {
        i64 t = look - lane;
        u64 s = LB_FLAG_INC; // tiles before 0: inclusive prefix 0
        if (t >= 0) s = ld_volatile_u64(status + t);
        while (__any_sync(RIPS_FULL_MASK, (s >> 62) == 0)) {
            if (t >= 0 && (s >> 62) == 0) s = ld_volatile_u64(status + t);
        }
        unsigned inc = __ballot_sync(RIPS_FULL_MASK, (s >> 62) == 2);
        if (inc) {
            int first = __ffs(inc) - 1; // nearest predecessor that already holds an inclusive prefix
            excl += warp_sum_u64(lane <= first ? (s & LB_VALUE_MASK) : 0ull);
            break;
        }
        excl += warp_sum_u64(s & LB_VALUE_MASK);
        look -= 32;
    }
    stress_jitter((u32)tile + 77u);
    if (lane == 0) st_volatile_u64(status + tile, LB_FLAG_INC | (excl + aggregate));
    return excl;
}

// ---------------------------------------------------------------------------------------------
// Diameter KEYS.  key(e) = dense rank of the edge value in DESCENDING order (0 = the largest
// distance), so diam(simplex) = max value = MIN key, the coboundary order (diameter descending) is
// key ascending, and "diam <= threshold" is "key >= thr_key".
//   K  : u32, strict lower triangle, element (a > b) at a(a-1)/2 + b          (set-up, host reduction)
//   Kf : full symmetric n x n matrix of key+1 with a ZERO diagonal, u16 when every key+1 fits,
//        else u32.  The shift makes 0 smaller than every real entry, so a test "all edges from v
//        to the vertices of s have key >= key(s)" rejects v in s by itself, with no membership
//        logic, and rows are contiguous in the scanned vertex whichever of the two is larger.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ u32 dkey(const u32* __restrict__ K, int a, int b)
{
    int hi = max(a, b), lo = min(a, b);
    return __ldg(K + ((u32)hi * (u32)(hi - 1) >> 1) + lo);
}

// Binomial table, k-major: B[k * stride + v] = C(v, k), v in [0, n], k in [0, kmax], saturating.
struct BinomTable {
    const u64* B;
    int stride; // n + 1
    __device__ __forceinline__ u64 operator()(int v, int k) const { return __ldg(B + k * stride + v); }
};

// Largest v in [lo, hi] with C(v, k) <= x (exists because C(lo, k) <= x is guaranteed by callers).
__device__ __forceinline__ int binom_upper_vertex(const BinomTable& bt, u64 x, int k, int lo, int hi)
{
    const u64* row = bt.B + k * bt.stride;
    while (lo < hi) {
        int mid = (lo + hi + 1) >> 1;
        if (__ldg(row + mid) <= x) lo = mid;
        else hi = mid - 1;
    }
    return lo;
}

// Eq. 2 inverse: idx -> vertices v[M-1] > ... > v[0] of an (M-1)-simplex on n points.
template <int M>
__device__ __forceinline__ void decode_simplex(const BinomTable& bt, u64 idx, int n, int (&v)[M])
{
    int hi = n - 1;
#pragma unroll
    for (int k = M; k >= 1; --k) {
        int x = binom_upper_vertex(bt, idx, k, k - 1, hi);
        v[k - 1] = x;
        idx -= bt(x, k);
        hi = x - 1;
    }
}

// Same result as decode_simplex, but each binary search is replaced by the closed-form estimate
// v ~ (k! idx)^(1/k) + (k-1)/2 (from C(v,k) ~ (v-(k-1)/2)^k / k!) followed by an exact fix-up against
// the table, so the float arithmetic only decides how many fix-up steps run, never the result.
template <int M>
__device__ __forceinline__ void decode_simplex_fast(const BinomTable& bt, u64 idx, int n, int (&v)[M])
{
    int hi = n - 1;
#pragma unroll
    for (int k = M; k >= 1; --k) {
        int x;
        if (k == 1) {
            x = (int)idx;
        } else {
            float fact = 1.f;
#pragma unroll
            for (int i = 2; i <= k; ++i) fact *= (float)i;
            const float y = fact * (float)idx;
            float r;
            if (k == 2) r = sqrtf(y);
            else if (k == 4) r = sqrtf(sqrtf(y));
            else r = __powf(y, 1.0f / (float)k);
            x = (int)(r + 0.5f * (float)(k - 1));
            x = min(max(x, k - 1), hi);
            const u64* row = bt.B + k * bt.stride;
            while (x < hi && __ldg(row + x + 1) <= idx) ++x;
            while (x > k - 1 && __ldg(row + x) > idx) --x;
        }
        v[k - 1] = x;
        idx -= bt(x, k);
        hi = x - 1;
    }
}

static inline int bits_for(u64 max_value)
{ // number of bits needed to store values in [0, max_value]
    int b = 0;
    while (max_value) { ++b; max_value >>= 1; }
    return b ? b : 1;
}
