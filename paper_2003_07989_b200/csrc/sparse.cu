// sparse.cu -- the sparse path: stage 1 for a threshold far below the enclosing radius,
// where the Rips complex is the flag complex of a sparse graph and walking all C(n, d+1) combinatorial indices
// (and holding a C(n, d+1)-bit clearing bitmap) is out of the question.  After the paper's sparse option
// (Algorithm 5: cofacets from the neighbour lists of the 1-skeleton; the
// filtration is built from the simplices one dimension down, the memory is sized by what is found):
//
//   neighbour lists   CSR of the admissible edges (key >= thr_key), every list ascending by vertex.
//   simplex lists     L_1 = the admissible edges; L_d = for every sigma in L_{d-1} (in index order) and every
//                     neighbour w of its top vertex with w > top(sigma) that is adjacent to all of sigma:
//                     sigma + {w}.  Every d-simplex of the complex is made exactly once (from the facet that lacks
//                     its top vertex); a stable partition by the top vertex w puts the list into increasing
//                     combinatorial index (colex order, Remark 2).  The lists hold ALL simplices,
//                     cleared or not: the next dimension is made from them.
//   sparse_apparent_kernel   one THREAD per simplex of L_d: diameter key, clearing by binary search in the sorted
//                     pivots of dimension d-1, and the apparent-pair test of Algorithm 3 with the cofacets taken,
//                     in decreasing vertex order, from the neighbour list of the simplex's vertex of smallest degree
//                     (a cofacet vertex is a common neighbour of all vertices).  It writes what the dense kernels
//                     write in slot mode, with the position in L_d in place of the combinatorial index as the slot:
//                     a column record or a sentinel, a pair slot, the two small lists, the counters -- so the sorts
//                     of stage 1 and all of stage 2 are the dense path's, unchanged.
#include "apparent.cuh"
#include "kernels.cuh"

namespace {

constexpr int SP_THREADS = 256;

// ---- CSR of the admissible edges
template <typename KT>
__global__ void csr_count_kernel(const KT* __restrict__ Kf, int n, int pitch, u32 thr1, u32* __restrict__ deg)
{
    const int v = blockIdx.x;
    u32 c = 0;
    for (int w = threadIdx.x; w < n; w += blockDim.x) c += ((u32)Kf[(size_t)v * pitch + w] >= thr1) ? 1u : 0u; // the zero diagonal fails
    c = warp_sum_u32(c);
    __shared__ u32 s[32];
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        u32 t = 0;
        for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += s[i];
        deg[v] = t;
    }
}

// off[v] = sum of deg[0..v), off[n] = total; one CTA (n <= 46340)
__global__ void csr_scan_kernel(const u32* __restrict__ deg, int n, u64* __restrict__ off)
{
    __shared__ u64 s_w[32];
    __shared__ u64 s_carry;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (int base = 0; base < n; base += blockDim.x) {
        const int i = base + tid;
        const u64 c = i < n ? (u64)deg[i] : 0ull;
        u64 incl = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u64 t = __shfl_up_sync(RIPS_FULL_MASK, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) s_w[warp] = incl;
        __syncthreads();
        u64 woff = 0, tot = 0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) {
            if (w < warp) woff += s_w[w];
            tot += s_w[w];
        }
        if (i < n) off[i] = s_carry + woff + incl - c;
        __syncthreads();
        if (tid == 0) s_carry += tot;
        __syncthreads();
    }
    if (tid == 0) off[n] = s_carry;
}

// adj[off[v] ..] = the neighbours of v, ascending; one warp per vertex
template <typename KT>
__global__ void csr_fill_kernel(const KT* __restrict__ Kf, int n, int pitch, u32 thr1, const u64* __restrict__ off, u32* __restrict__ adj)
{
    const int v = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (v >= n) return;
    u64 at = off[v];
    for (int base = 0; base < n; base += 32) {
        const int w = base + lane;
        const bool ok = w < n && (u32)Kf[(size_t)v * pitch + w] >= thr1;
        const u32 bal = __ballot_sync(RIPS_FULL_MASK, ok);
        if (ok) adj[at + __popc(bal & ((1u << lane) - 1u))] = (u32)w;
        at += __popc(bal);
    }
}

// first position in the ascending list a[0..len) whose entry exceeds x
__device__ __forceinline__ u32 upper_bound_u32(const u32* __restrict__ a, u32 len, u32 x)
{
    u32 lo = 0, hi = len;
    while (lo < hi) {
        const u32 mid = (lo + hi) >> 1;
        if (__ldg(a + mid) <= x) lo = mid + 1;
        else hi = mid;
    }
    return lo;
}

// ---- simplex lists.  MP = vertices of the simplices of the INPUT list (MP = 1: the vertices themselves).
// WRITE = false: cnt[i] = number of simplices made from input simplex i; WRITE = true: they are written at pos[i],
// in increasing w.  Records are vertex words (vertex j at bit j * vbits).
template <int MP, typename KT, bool WRITE>
__global__ void expand_kernel(const u64* __restrict__ in, i64 n_in, const KT* __restrict__ Kf, int pitch, u32 thr1, int vbits,
                              const u64* __restrict__ off, const u32* __restrict__ adj, u32* __restrict__ cnt,
                              const u64* __restrict__ pos, u64* __restrict__ out)
{
    const i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_in) return;
    int s[MP];
    u64 rec;
    if (MP == 1) { rec = (u64)i; s[0] = (int)i; }   // the list of vertices is implicit
    else { rec = __ldg(in + i); unpack_vertices<MP>(rec, vbits, s); }
    const int top = s[MP - 1];
    const u32* list = adj + off[top];
    const u32 len = (u32)(off[top + 1] - off[top]);
    u32 c = 0;
    u64 at = WRITE ? pos[i] : 0;
    for (u32 k = upper_bound_u32(list, len, (u32)top); k < len; ++k) {
        const int w = (int)__ldg(list + k);
        bool ok = true;
#pragma unroll
        for (int j = 0; j < MP - 1; ++j) ok = ok && ((u32)Kf[(size_t)w * pitch + s[j]] >= thr1);
        if (ok) {
            if (WRITE) out[at++] = rec | ((u64)(u32)w << (MP * vbits));
            ++c;
        }
    }
    if (!WRITE) cnt[i] = c;
}

// pos[i] = sum of cnt[0..i) (u64), total at pos[n]; tiles of 2048 with a decoupled look-back
__global__ void __launch_bounds__(SP_THREADS) scan_counts_kernel(const u32* __restrict__ cnt, i64 n, u64* __restrict__ pos, u64* status, u32* ticket)
{
    __shared__ u32 s_tile;
    __shared__ u64 s_w[SP_THREADS / 32];
    __shared__ u64 s_excl;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = atomicAdd(ticket, 1u);
    __syncthreads();
    const i64 tile = s_tile, base = tile * (SP_THREADS * 8) + (i64)tid * 8;
    u64 c[8], sum = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        c[k] = (base + k < n) ? (u64)cnt[base + k] : 0ull;
        sum += c[k];
    }
    u64 incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const u64 t = __shfl_up_sync(RIPS_FULL_MASK, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_w[warp] = incl;
    __syncthreads();
    u64 woff = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < SP_THREADS / 32; ++w) {
        if (w < warp) woff += s_w[w];
        tot += s_w[w];
    }
    if (warp == 0) {
        const u64 e = lookback_exclusive(status, tile, tot);
        if (lane == 0) s_excl = e;
    }
    __syncthreads();
    u64 run = s_excl + woff + incl - sum;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        if (base + k < n) pos[base + k] = run;
        run += c[k];
    }
    if (base <= n - 1 && n - 1 < base + 8) pos[n] = s_excl + woff + incl; // the thread that holds the last element
}

__device__ __forceinline__ bool in_sorted_field(const u64* __restrict__ a, i64 n, int shift, u64 mask, u64 x)
{
    i64 lo = 0, hi = n;
    while (lo < hi) {
        const i64 mid = lo + ((hi - lo) >> 1);
        if (((__ldg(a + mid) >> shift) & mask) < x) lo = mid + 1;
        else hi = mid;
    }
    return lo < n && ((__ldg(a + lo) >> shift) & mask) == x;
}

// ============================================================================== sparse_apparent_kernel
template <int M, typename KT>
__global__ void __launch_bounds__(SP_THREADS) sparse_apparent_kernel(const SparseParams p)
{
    const KT* __restrict__ Kf = reinterpret_cast<const KT*>(p.Kf);
    const i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    const u32 lt_mask = (1u << lane) - 1u;
    const bool valid = i < p.n_simp;
    int s[M];
    u64 verts = 0;
    if (valid) verts = __ldg(p.simp + i);
    unpack_vertices<M>(verts, p.vbits, s);
    bool keep = false, cleared = false;
    u32 key1 = 0xffffffffu;
    u64 ci = 0;
    if (valid) {
#pragma unroll
        for (int a = 1; a < M; ++a)
#pragma unroll
            for (int b = 0; b < a; ++b) key1 = min(key1, (u32)Kf[(size_t)s[a] * p.pitch + s[b]]);
#pragma unroll
        for (int j = 0; j < M; ++j) ci += p.bt(s[j], j + 1); // Eq. 2
        // a4: cleared iff the simplex is the death simplex of a pair of dimension d-1 (three sorted layers)
        cleared = in_sorted_field(p.c_reg, p.n_reg, 0, p.reg_mask, ci) || in_sorted_field(p.c_irr, p.n_irr, RIPS_PAIR_POS_BITS, ~0ull, ci) ||
                  in_sorted_field(p.c_red, p.n_red, 0, ~0ull, ci);
        keep = !cleared;
    }
    // ---- a7: cofacets s + {v}, v a common neighbour, in decreasing v: the neighbour list of the vertex of smallest degree
    int fv = -1;
    if (keep) {
        int jb = 0;
        u32 best = 0xffffffffu;
#pragma unroll
        for (int j = 0; j < M; ++j) {
            const u32 dg = (u32)(p.off[s[j] + 1] - p.off[s[j]]);
            if (dg < best) { best = dg; jb = j; }
        }
        int vb = s[0];
#pragma unroll
        for (int j = 1; j < M; ++j) vb = (j == jb) ? s[j] : vb;
        const u32* list = p.adj + p.off[vb];
        for (int k = (int)best - 1; k >= 0; --k) {
            const int v = (int)__ldg(list + k);
            u32 m = 0xffffffffu;
#pragma unroll
            for (int j = 0; j < M; ++j) m = min(m, (u32)Kf[(size_t)s[j] * p.pitch + v]); // a vertex of s reads the zero diagonal and fails
            if (m >= key1) { fv = v; break; }
        }
    }
    const bool found = fv >= 0;
    const bool regular = found && fv > s[M - 1];
    u64 prec = (u64)(u32)p.n << p.tbits;
    if (regular) prec = ((u64)(u32)fv << p.tbits) | (ci + p.bt(fv, M + 1));
    const u64 rec = keep ? (((u64)(key1 - 1u) << p.lowbits) | verts) : ((u64)p.sentinel_key << p.lowbits);
    bool is_irr = false, is_non = keep && !found;
    u64 irr_rec = 0;
    if (found && !regular) {
        int fseg = 0;
#pragma unroll
        for (int j = 0; j < M; ++j) fseg += (s[j] < fv) ? 1 : 0;
        if (s_is_youngest_facet<M, KT>(Kf, p.pitch, s, key1, fv, fseg)) {
            irr_rec = (cofacet_index<M>(p.bt, s, fv, fseg) << RIPS_PAIR_POS_BITS) | (u64)fseg;
            is_irr = true;
        } else
            is_non = true;
    }
    const u32 b_irr = __ballot_sync(RIPS_FULL_MASK, is_irr);
    if (b_irr) {
        u64 base = 0;
        if (lane == __ffs(b_irr) - 1) base = atomicAdd((unsigned long long*)(p.counters + S1C_IRREGULAR), (unsigned long long)__popc(b_irr));
        base = __shfl_sync(RIPS_FULL_MASK, base, __ffs(b_irr) - 1) + __popc(b_irr & lt_mask);
        if (is_irr && base < p.irr_cap) p.irr_out[base] = irr_rec;
    }
    const u32 b_non = __ballot_sync(RIPS_FULL_MASK, is_non);
    if (b_non) {
        u64 base = 0;
        if (lane == __ffs(b_non) - 1) base = atomicAdd((unsigned long long*)(p.counters + S1C_NONAPP), (unsigned long long)__popc(b_non));
        base = __shfl_sync(RIPS_FULL_MASK, base, __ffs(b_non) - 1) + __popc(b_non & lt_mask);
        if (is_non && base < p.non_cap) p.non_out[base] = rec;
    }
    if (valid) {
        p.cols_out[i] = rec;
        p.pairs_out[i] = prec;
    }
    const u32 b_keep = __ballot_sync(RIPS_FULL_MASK, keep), b_clr = __ballot_sync(RIPS_FULL_MASK, cleared), b_reg = __ballot_sync(RIPS_FULL_MASK, regular);
    if (lane == 0) {
        if (b_keep) atomicAdd((unsigned long long*)(p.counters + S1C_KEPT), (unsigned long long)__popc(b_keep));
        if (b_clr) atomicAdd((unsigned long long*)(p.counters + S1C_CLEARED), (unsigned long long)__popc(b_clr));
        if (b_reg) atomicAdd((unsigned long long*)(p.counters + S1C_REGULAR), (unsigned long long)__popc(b_reg));
    }
}

} // namespace

// =============================================================================================== launchers
i64 sparse_scan_tiles(i64 n) { return (n + SP_THREADS * 8 - 1) / (SP_THREADS * 8); }

cudaError_t launch_csr_count(const void* Kf, int kf_u16, int n, int pitch, u32 thr1, u32* deg, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    if (kf_u16) csr_count_kernel<unsigned short><<<n, 128, 0, st>>>((const unsigned short*)Kf, n, pitch, thr1, deg);
    else csr_count_kernel<u32><<<n, 128, 0, st>>>((const u32*)Kf, n, pitch, thr1, deg);
    return cudaGetLastError();
}
cudaError_t launch_csr_scan(const u32* deg, int n, u64* off, cudaStream_t st)
{
    csr_scan_kernel<<<1, 1024, 0, st>>>(deg, n, off);
    return cudaGetLastError();
}
cudaError_t launch_csr_fill(const void* Kf, int kf_u16, int n, int pitch, u32 thr1, const u64* off, u32* adj, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    const unsigned g = (unsigned)((n + 3) / 4);
    if (kf_u16) csr_fill_kernel<unsigned short><<<g, 128, 0, st>>>((const unsigned short*)Kf, n, pitch, thr1, off, adj);
    else csr_fill_kernel<u32><<<g, 128, 0, st>>>((const u32*)Kf, n, pitch, thr1, off, adj);
    return cudaGetLastError();
}
cudaError_t launch_scan_counts(const u32* cnt, i64 n, u64* pos, u64* status, u32* ticket, cudaStream_t st)
{
    if (n == 0) return cudaSuccess;
    scan_counts_kernel<<<(unsigned)sparse_scan_tiles(n), SP_THREADS, 0, st>>>(cnt, n, pos, status, ticket);
    return cudaGetLastError();
}

template <int MP, typename KT>
static cudaError_t launch_expand_t(const SparseExpand& e, bool write, cudaStream_t st)
{
    const unsigned g = (unsigned)((e.n_in + SP_THREADS - 1) / SP_THREADS);
    if (write) expand_kernel<MP, KT, true><<<g, SP_THREADS, 0, st>>>(e.in, e.n_in, (const KT*)e.Kf, e.pitch, e.thr1, e.vbits, e.off, e.adj, e.cnt, e.pos, e.out);
    else expand_kernel<MP, KT, false><<<g, SP_THREADS, 0, st>>>(e.in, e.n_in, (const KT*)e.Kf, e.pitch, e.thr1, e.vbits, e.off, e.adj, e.cnt, e.pos, e.out);
    return cudaGetLastError();
}
cudaError_t launch_expand(int MP, int kf_u16, const SparseExpand& e, bool write, cudaStream_t st)
{
    if (e.n_in == 0) return cudaSuccess;
#define SX_CASE(MM) case MM: return kf_u16 ? launch_expand_t<MM, unsigned short>(e, write, st) : launch_expand_t<MM, u32>(e, write, st);
    switch (MP) {
        SX_CASE(1) SX_CASE(2) SX_CASE(3) SX_CASE(4) SX_CASE(5)
    default: return cudaErrorInvalidValue;
    }
#undef SX_CASE
}

cudaError_t launch_sparse_apparent(int M, int kf_u16, const SparseParams& p, cudaStream_t st)
{
    if (p.n_simp == 0) return cudaSuccess;
    const unsigned g = (unsigned)((p.n_simp + SP_THREADS - 1) / SP_THREADS);
#define SA_CASE(MM)                                                                                     \
    case MM:                                                                                            \
        if (kf_u16) sparse_apparent_kernel<MM, unsigned short><<<g, SP_THREADS, 0, st>>>(p);            \
        else sparse_apparent_kernel<MM, u32><<<g, SP_THREADS, 0, st>>>(p);                              \
        break;
    switch (M) {
        SA_CASE(2) SA_CASE(3) SA_CASE(4) SA_CASE(5) SA_CASE(6)
    default: return cudaErrorInvalidValue;
    }
#undef SA_CASE
    return cudaGetLastError();
}
