// apparent.cuh -- device pieces of the Apparent Pairs Lemma test (Lemma 7, PAPER.md:283-293;
// Algorithm 3) shared by the fused enumerate kernel (stage1.cu) and the
// warp-cooperative tail it falls back to.
//
// For a column s (vertices s[M-1] > ... > s[0], key1 = key(s)+1 in the units of Kf):
//   * the cofacets t = s + {v} are scanned for v = n-1 .. 0 (decreasing cidx, Remark 2,
//     PAPER.md:95); diam(t) = diam(s) iff every new edge (v, s_j) has key >= key(s); the first such
//     v gives the oldest cofacet of equal diameter.  v in s reads Kf's zero diagonal and fails by
//     itself;
//   * the facets of t that precede s in increasing cidx (Algorithm 6) are exactly
//     those that drop a vertex w of s with w > v (colex order), so (s,t) is apparent iff none of
//     them has the diameter of s -- no facet index is ever formed.  If v exceeds every vertex of
//     s there is no such facet: the pair is apparent with no further work, and
//     cidx(t) = cidx(s) + C(v, M+1).  These are the REGULAR pairs (>99.9 % at the paper-shaped
//     workloads); since cidx(t) is then increasing in cidx(s) for fixed v and the ranges of
//     different v are disjoint and increasing, a stable partition by v of the regular pairs,
//     produced in cidx(s) order, IS their sort by cidx(t).
#pragma once
#include "common.cuh"

template <int M>
__device__ __forceinline__ void unpack_vertices(u64 rec, int vbits, int (&s)[M])
{
    const u32 vmask = (1u << vbits) - 1u;
#pragma unroll
    for (int j = 0; j < M; ++j) s[j] = (int)((u32)(rec >> (j * vbits)) & vmask);
}

// Facet test for a cofacet vertex v below the top of s.  fseg = number of vertices of s below v.
template <int M, typename KT>
__device__ __forceinline__ bool s_is_youngest_facet(const KT* Kf, int pitch, const int (&s)[M], u32 key1, int v, int fseg)
{
    u32 vk[M];
#pragma unroll
    for (int a = 0; a < M; ++a) vk[a] = (u32)Kf[s[a] * pitch + v];
    u32 pk[M][M];
#pragma unroll
    for (int a = 1; a < M; ++a)
#pragma unroll
        for (int b = 0; b < a; ++b) pk[a][b] = (u32)Kf[s[a] * pitch + s[b]];
    bool youngest = true;
#pragma unroll
    for (int j = 0; j < M; ++j) {
        if (j >= fseg) { // facet t - s[j], s[j] > v
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
            if (mn == key1) youngest = false;
        }
    }
    return youngest;
}

// cidx of t = s + {v}, v at position fseg (Eq. 2)
template <int M>
__device__ __forceinline__ u64 cofacet_index(const BinomTable& bt, const int (&s)[M], int v, int fseg)
{
    u64 t = bt(v, fseg + 1);
#pragma unroll
    for (int i = 0; i < M; ++i) t += bt(s[i], (i < fseg) ? i + 1 : i + 2);
    return t;
}
