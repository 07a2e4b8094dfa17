// reduce.cu -- device part of the reduction of the non-apparent columns (not the hot path; SURVEY.md
// 8(f) item 1).  Algorithm 2 restricted to what is embarrassingly parallel: every
// non-apparent column is reduced against the APPARENT columns only,
//     R[j] <- D_j ;  while low(R[j]) is the row of an apparent pair (s', t):  R[j] <- R[j] + D_{s'}
// which needs nothing from the other non-apparent columns (an apparent column is reduced as it stands,
// PAPER.md:260, :297-299, and precedes every other facet of its row in the coboundary order).  At the
// paper-shaped workloads ~97 % of all column additions are of this kind.  One warp per column: the
// working column is an unsorted list of packed entries (key << tbits | cidx(t)) in shared memory, its
// pivot the largest entry (smallest diameter, then largest index: the first in filtration order,
// PAPER.md:77-79) of odd multiplicity (Z/2), found by a warp-wide max; rows are looked up in the
// sorted layers of the pair store by binary search.  The few conflicts between
// non-apparent columns that remain (equal pivots) are resolved serially on the host (reduce_host.cpp).
#include "apparent.cuh"
#include "kernels.cuh"

namespace {

constexpr int PR_WARPS = 4;
constexpr int PR_THREADS = PR_WARPS * 32;
constexpr int PR_CAP = 2048; // entries of a working column

__device__ __forceinline__ i64 lower_bound_field_d(const u64* __restrict__ a, i64 n, int shift, u64 mask, u64 x)
{
    i64 lo = 0, hi = n;
    while (lo < hi) {
        i64 mid = lo + ((hi - lo) >> 1);
        if (((__ldg(a + mid) >> shift) & mask) < x) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

// coboundary of s appended to the list (entries stored +1 so that 0 means "empty"); returns the new length,
// or -1 if the list is full
template <int M, typename KT>
__device__ __forceinline__ int push_coboundary(const PreReduceParams& p, const KT* __restrict__ Kf, const int (&s)[M], u64* list,
                                               int len, int lane)
{
    u32 key_s = 0xffffffffu;
#pragma unroll
    for (int a = 1; a < M; ++a)
#pragma unroll
        for (int b = 0; b < a; ++b) key_s = min(key_s, (u32)__ldg(Kf + s[a] * p.pitch + s[b]));
    const u32 thr1 = p.thr_key + 1u;
    for (int base = p.n - 1; base >= 0; base -= 32) {
        const int v = base - lane;
        bool ok = false;
        u64 e = 0;
        if (v >= 0) {
            u32 kt = key_s;
#pragma unroll
            for (int j = 0; j < M; ++j) kt = min(kt, (u32)__ldg(Kf + s[j] * p.pitch + v));
            // kt == 0: v is a vertex of s (zero diagonal); kt < thr1: the cofacet is above the threshold
            if (kt != 0 && kt >= thr1) {
                int fseg = 0;
#pragma unroll
                for (int j = 0; j < M; ++j) fseg += (s[j] < v) ? 1 : 0;
                e = (((u64)(kt - 1u) << p.tbits) | cofacet_index<M>(p.bt, s, v, fseg)) + 1ull;
                ok = true;
            }
        }
        const u32 bal = __ballot_sync(RIPS_FULL_MASK, ok);
        if (len + __popc(bal) > PR_CAP) return -1;
        if (ok) list[len + __popc(bal & ((1u << lane) - 1u))] = e;
        len += __popc(bal);
    }
    __syncwarp();
    return len;
}

template <int M, typename KT>
__global__ void __launch_bounds__(PR_THREADS) prereduce_kernel(const PreReduceParams p)
{
    extern __shared__ __align__(16) unsigned char smem_pr[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    u64* list = reinterpret_cast<u64*>(smem_pr) + (size_t)warp * PR_CAP;
    const KT* __restrict__ Kf = reinterpret_cast<const KT*>(p.Kf);
    const u64 tmask = (1ull << p.tbits) - 1ull;

    for (i64 col = (i64)blockIdx.x * PR_WARPS + warp; col < p.ncols; col += (i64)gridDim.x * PR_WARPS) {
        int s[M];
        unpack_vertices<M>(__ldg(p.cols + col), p.vbits, s);
        int len = push_coboundary<M, KT>(p, Kf, s, list, 0, lane);
        u64 result = 0; // 0: the column reduced to zero
        u32 adds = 0;
        for (;;) {
            // ---- pivot: the largest entry of odd multiplicity
            u64 piv = 0;
            for (;;) {
                u64 m = 0;
                for (int i = lane; i < len; i += 32) m = max(m, list[i]);
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(RIPS_FULL_MASK, m, o));
                if (m == 0) break;
                u32 cnt = 0;
                for (int i = lane; i < len; i += 32)
                    if (list[i] == m) { ++cnt; list[i] = 0; }
                cnt = __reduce_add_sync(RIPS_FULL_MASK, cnt);
                __syncwarp();
                if (cnt & 1u) { piv = m; break; }
            }
            if (piv == 0) { result = 0; break; }
            // ---- is the pivot's row the row of an apparent pair?  (all lanes search redundantly: uniform)
            const u64 t = (piv - 1ull) & tmask;
            bool hit = false;
            int s2[M];
            {
                i64 p1 = lower_bound_field_d(p.layers.reg, p.layers.n_reg, 0, tmask, t);
                if (p1 < p.layers.n_reg && (__ldg(p.layers.reg + p1) & tmask) == t) {
                    // s' = t minus its top vertex v
                    int tv[M + 1];
                    decode_simplex<M + 1>(p.bt, t, p.n, tv);
#pragma unroll
                    for (int j = 0; j < M; ++j) s2[j] = tv[j];
                    hit = true;
                } else {
                    i64 p2 = lower_bound_field_d(p.layers.irr, p.layers.n_irr, RIPS_PAIR_POS_BITS, ~0ull, t);
                    if (p2 < p.layers.n_irr && (__ldg(p.layers.irr + p2) >> RIPS_PAIR_POS_BITS) == t) {
                        const int jpos = (int)(__ldg(p.layers.irr + p2) & ((1u << RIPS_PAIR_POS_BITS) - 1u));
                        int tv[M + 1];
                        decode_simplex<M + 1>(p.bt, t, p.n, tv);
#pragma unroll
                        for (int j = 0; j < M; ++j) s2[j] = tv[j < jpos ? j : j + 1];
                        hit = true;
                    }
                }
            }
            if (!hit) { result = piv; break; } // a row no apparent pair owns: left to the host's conflict pass
            if (adds >= p.max_additions) { result = ~0ull; break; }
            // ---- R[j] <- R[j] + D_{s'}: the pivot itself goes back, D_{s'} holds it once more and they cancel
            if (len + 1 > PR_CAP) { result = ~0ull; break; }
            if (lane == 0) list[len] = piv;
            ++len;
            __syncwarp();
            int nl = push_coboundary<M, KT>(p, Kf, s2, list, len, lane);
            if (nl < 0) {
                // compact the list (drop the emptied slots) and try once more
                int w = 0;
                for (int base = 0; base < len; base += 32) {
                    const int i = base + lane;
                    const u64 e = i < len ? list[i] : 0;
                    const u32 bal = __ballot_sync(RIPS_FULL_MASK, e != 0);
                    __syncwarp();
                    if (e != 0) list[w + __popc(bal & ((1u << lane) - 1u))] = e;
                    w += __popc(bal);
                    __syncwarp();
                }
                len = w;
                nl = push_coboundary<M, KT>(p, Kf, s2, list, len, lane);
                if (nl < 0) { result = ~0ull; break; }
            }
            len = nl;
            ++adds;
        }
        if (lane == 0) {
            p.pivot_out[col] = result; // 0 zero column, ~0 deferred to the host, else (key << tbits | t) + 1
            p.adds_out[col] = adds;
        }
        __syncwarp();
    }
}

template <int M, typename KT>
cudaError_t launch_prereduce_t(const PreReduceParams& p, cudaStream_t st)
{
    const size_t smem = (size_t)PR_WARPS * PR_CAP * 8;
    auto kern = prereduce_kernel<M, KT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    i64 g = (p.ncols + PR_WARPS - 1) / PR_WARPS;
    if (g > 148 * 3 * 8) g = 148 * 3 * 8;
    kern<<<(unsigned)g, PR_THREADS, smem, st>>>(p);
    return cudaGetLastError();
}

} // namespace

cudaError_t launch_prereduce(int M, int kf_u16, const PreReduceParams& p, cudaStream_t st)
{
    if (p.ncols == 0) return cudaSuccess;
#define PR_CASE(MM)                                                                          \
    case MM: return kf_u16 ? launch_prereduce_t<MM, unsigned short>(p, st) : launch_prereduce_t<MM, u32>(p, st);
    switch (M) {
        PR_CASE(2) PR_CASE(3) PR_CASE(4) PR_CASE(5) PR_CASE(6)
    default: return cudaErrorInvalidValue;
    }
#undef PR_CASE
}
