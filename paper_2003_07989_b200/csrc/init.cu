// init.cu -- set-up kernels of rips_init (steps a1-a2): validate and canonicalise the distance
// matrix, and replace every distance by the dense rank of its value in DESCENDING order (the
// "key").  Every diameter is one of the edge values (Eq. 1), so keys of 15-19 bits
// replace the fp32 diameters inside the kernels and inside the sort; the fp32 values come back
// through values[key].
#include "kernels.cuh"

namespace {

__global__ void prep_edges_kernel(float* __restrict__ dist, i64 E, u64* __restrict__ rec, int* bad, float threshold, u64* n_over)
{
    i64 e = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= E) return;
    float x = dist[e];
    if (x == 0.0f) x = 0.0f; // -0 -> +0 (the comparison is true for both zeros)
    if (!(x >= 0.0f) || isinf(x)) { atomicOr(bad, 1); x = 0.0f; }
    dist[e] = x;
    // every value above the threshold is ranked as ONE class (key 0, "value" +inf): no simplex that holds such an edge
    // is ever kept, so their order among themselves is never looked at, and the keys of a thresholded input need only
    // as many bits as it has admissible values (fewer sort passes; records that fit 64 bits for larger n)
    if (x > threshold) {
        x = __int_as_float(0x7f800000);
        atomicAdd((unsigned long long*)n_over, 1ull); // (the compiler aggregates this per warp)
    }
    // non-negative floats order like their bit patterns; invert so that ascending = value descending
    rec[e] = ((u64)(~__float_as_uint(x)) << 32) | (u64)e;
}

constexpr int RK_THREADS = 256;
constexpr int RK_IPT = 8;
constexpr int RK_WARPS = RK_THREADS / 32;
constexpr int RK_TILE = RK_THREADS * RK_IPT;

// Dense rank of the sorted edge values: head[i] = value differs from its predecessor; rank = number
// of heads at or before i, minus one.  Single pass, decoupled look-back over tiles.
__global__ void __launch_bounds__(RK_THREADS) rank_edges_kernel(const u64* __restrict__ rec, i64 E, u32* __restrict__ K,
                                                               float* __restrict__ values, u64* status, u32* ticket,
                                                               u64* n_distinct)
{
    __shared__ u32 s_wcount[RK_WARPS];
    __shared__ u32 s_tile;
    __shared__ u64 s_excl;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const i64 tile = s_tile;
    const i64 wbase = tile * RK_TILE + (i64)warp * (32 * RK_IPT);
    u32 heads[RK_IPT]; // ballot of the heads of each 32-wide step (same in every lane)
    u64 r[RK_IPT];
    u32 wcount = 0;
#pragma unroll
    for (int it = 0; it < RK_IPT; ++it) {
        i64 i = wbase + it * 32 + lane;
        bool head = false;
        r[it] = 0;
        if (i < E) {
            r[it] = __ldg(rec + i);
            head = (i == 0) || ((__ldg(rec + i - 1) >> 32) != (r[it] >> 32));
        }
        heads[it] = __ballot_sync(RIPS_FULL_MASK, head);
        wcount += __popc(heads[it]);
    }
    if (lane == 0) s_wcount[warp] = wcount;
    __syncthreads();
    u32 wexcl = 0, ttotal = 0;
#pragma unroll
    for (int w = 0; w < RK_WARPS; ++w) {
        u32 c = s_wcount[w];
        if (w < warp) wexcl += c;
        ttotal += c;
    }
    if (warp == 0) {
        u64 e = lookback_exclusive(status, tile, (u64)ttotal);
        if (lane == 0) {
            s_excl = e;
            if (ttotal) atomicAdd((unsigned long long*)n_distinct, (unsigned long long)ttotal);
        }
    }
    __syncthreads();
    u64 run = s_excl + wexcl; // heads before this warp's chunk
    const u32 le_mask = (lane == 31) ? RIPS_FULL_MASK : ((2u << lane) - 1u);
#pragma unroll
    for (int it = 0; it < RK_IPT; ++it) {
        i64 i = wbase + it * 32 + lane;
        if (i < E) {
            u32 rank = (u32)(run + __popc(heads[it] & le_mask)) - 1u;
            K[(u32)r[it]] = rank;
            if ((heads[it] >> lane) & 1u) values[rank] = __uint_as_float(~(u32)(r[it] >> 32));
        }
        run += __popc(heads[it]);
    }
}

// Kf[i*pitch + j] = key(i,j) + 1 for i != j, 0 on the diagonal (common.cuh); the pitch makes the rows
// of consecutive vertices fall into different shared-memory banks
template <typename KT>
__global__ void build_full_keys_kernel(const u32* __restrict__ K, int n, int pitch, KT* __restrict__ Kf)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
    if (j >= n) return;
    u32 x = 0;
    if (i != j) x = dkey(K, i, j) + 1u;
    Kf[(size_t)i * pitch + j] = (KT)x;
}

// Sf[i*spitch + b] = max of Kf[i][32b .. 32b+31]: the largest key+1 (the shortest edge) from vertex i into block b of 32
// vertices.  The fused kernels' warp scan for a cofacet of equal diameter reads these block maxima first and skips
// every block that cannot hold one (stage1.cu, summary_scan).  One warp per (row, block).
template <typename KT>
__global__ void build_block_max_kernel(const KT* __restrict__ Kf, int n, int pitch, KT* __restrict__ Sf, int spitch, int nb)
{
    const int b = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), i = blockIdx.y, lane = threadIdx.x & 31;
    if (b >= nb) return;
    const int j = b * 32 + lane;
    u32 x = 0;
    if (j < n) x = (u32)Kf[(size_t)i * pitch + j];
    x = __reduce_max_sync(RIPS_FULL_MASK, x);
    if (lane == 0) Sf[(size_t)i * spitch + b] = (KT)x;
}

} // namespace

cudaError_t launch_build_block_max(const void* Kf, int n, int pitch, void* Sf, int spitch, int kf_u16, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    const int nb = (n + 31) / 32;
    dim3 g((unsigned)((nb + 7) / 8), (unsigned)n);
    if (kf_u16) build_block_max_kernel<unsigned short><<<g, 256, 0, st>>>((const unsigned short*)Kf, n, pitch, (unsigned short*)Sf, spitch, nb);
    else build_block_max_kernel<u32><<<g, 256, 0, st>>>((const u32*)Kf, n, pitch, (u32*)Sf, spitch, nb);
    return cudaGetLastError();
}

cudaError_t launch_build_full_keys(const u32* K, int n, int pitch, void* Kf, int kf_u16, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    dim3 g((unsigned)((n + 255) / 256), (unsigned)n);
    if (kf_u16) build_full_keys_kernel<unsigned short><<<g, 256, 0, st>>>(K, n, pitch, (unsigned short*)Kf);
    else build_full_keys_kernel<u32><<<g, 256, 0, st>>>(K, n, pitch, (u32*)Kf);
    return cudaGetLastError();
}

cudaError_t launch_prep_edges(float* dist, i64 E, u64* rec, int* bad, float threshold, u64* n_over, cudaStream_t st)
{
    if (E == 0) return cudaSuccess;
    prep_edges_kernel<<<(unsigned)((E + 255) / 256), 256, 0, st>>>(dist, E, rec, bad, threshold, n_over);
    return cudaGetLastError();
}

i64 rank_edges_tiles(i64 E) { return (E + RK_TILE - 1) / RK_TILE; }

cudaError_t launch_rank_edges(const u64* rec_sorted, i64 E, u32* K, float* values, u64* status, u32* ticket,
                              u64* n_distinct, cudaStream_t st)
{
    if (E == 0) return cudaSuccess;
    rank_edges_kernel<<<(unsigned)rank_edges_tiles(E), RK_THREADS, 0, st>>>(rec_sorted, E, K, values, status, ticket,
                                                                           n_distinct);
    return cudaGetLastError();
}
