// dim0.cu -- dimension 0 on the GPU (union-find over the edges in filtration order;
// the paper keeps it on the CPU).  Not the hot path; timed separately.
// Filter-Kruskal in one CTA: the sorted edge records of rips_init (value descending, cidx
// ascending) read backwards ARE the filtration order of the 1-simplices (diameter ascending,
// cidx descending).  Each round 1024 threads test 1024 edges against the current
// forest in parallel (read-mostly finds with path compression); the few edges whose endpoints are
// still in different components are compacted in order -- record and vertices into shared memory, so that
// no load from HBM sits on the serial path -- and merged serially by one thread, which
// is what makes the result independent of scheduling.  The loop stops after n-1 merges.
#include "kernels.cuh"

namespace {

constexpr int D0_THREADS = 1024;

__device__ __forceinline__ void edge_vertices(u32 e, int* a, int* b)
{
    int i = (int)((1.0 + sqrt(1.0 + 8.0 * (double)e)) * 0.5);
    while ((u64)i * (u64)(i - 1) / 2 > (u64)e) --i;
    while ((u64)(i + 1) * (u64)i / 2 <= (u64)e) ++i;
    *a = i;
    *b = (int)(e - (u32)((u64)i * (u64)(i - 1) / 2));
}

typedef unsigned short u16; // vertex numbers: n <= 46340 (rips_init)

__device__ __forceinline__ u32 find_root(volatile u16* parent, u32 x)
{
    u32 r = x;
    while (parent[r] != r) r = parent[r];
    // compression: every write stores an ancestor, so concurrent readers always see a valid forest
    while (parent[x] != r) { u32 nx = parent[x]; parent[x] = (u16)r; x = nx; }
    return r;
}

// SM: the union-find arrays (parent, largest vertex per root: 16 bits each, 4 bytes per vertex) live in shared memory
// (every n rips_init admits: 181 KB at n = 46340; as 32-bit words they left shared memory at n = 25000, and the kernel
// with its forest in HBM took 59 ms at n = 40000 instead of 14); else in the global scratch the caller passed.  The merges are serial, so their latency is
// the kernel's run time.
template <bool SM>
__global__ void __launch_bounds__(D0_THREADS) dim0_kernel(const u64* __restrict__ rec, i64 E, int n, u32 thr_inv,
                                                          u32* parent_maxv, Dim0Out out)
{
    extern __shared__ u32 s_uf[];
    if (SM) parent_maxv = s_uf;
    __shared__ u64 s_rec[D0_THREADS];  // the round's surviving edges in filtration order: record,
    __shared__ u32 s_ab[D0_THREADS];   // vertices (a << 16) | b (n <= 46340)
    __shared__ u32 s_wcount[D0_THREADS / 32];
    __shared__ i64 s_start;
    __shared__ u32 s_merges;
    volatile u16* parent = reinterpret_cast<volatile u16*>(parent_maxv);
    volatile u16* maxv = parent + n;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int i = tid; i < n; i += D0_THREADS) { parent[i] = (u16)i; maxv[i] = (u16)i; }
    if (tid == 0) {
        // first position whose value is <= threshold (records are value-descending = inverted bits ascending)
        i64 lo = 0, hi = E;
        while (lo < hi) {
            i64 mid = lo + ((hi - lo) >> 1);
            if ((u32)(rec[mid] >> 32) < thr_inv) lo = mid + 1;
            else hi = mid;
        }
        s_start = lo;
        s_merges = 0;
    }
    __syncthreads();
    const i64 start = s_start;
    for (i64 hi = E; hi > start; hi -= D0_THREADS) {
        const i64 i = hi - 1 - tid;
        bool cand = false;
        u64 r_mine = 0;
        int a_mine = 0, b_mine = 0;
        if (i >= start) {
            r_mine = rec[i];
            edge_vertices((u32)r_mine, &a_mine, &b_mine);
            cand = find_root(parent, a_mine) != find_root(parent, b_mine);
        }
        const u32 bal = __ballot_sync(RIPS_FULL_MASK, cand);
        if (lane == 0) s_wcount[warp] = __popc(bal);
        __syncthreads();
        u32 off = 0, tot = 0;
        for (int w = 0; w < D0_THREADS / 32; ++w) {
            u32 c = s_wcount[w];
            if (w < warp) off += c;
            tot += c;
        }
        if (cand) {
            const u32 slot = off + __popc(bal & ((1u << lane) - 1u));
            s_rec[slot] = r_mine;
            s_ab[slot] = ((u32)a_mine << 16) | (u32)b_mine;
        }
        __syncthreads();
        if (tid == 0) {
            u32 m = s_merges;
            for (u32 c = 0; c < tot && m < (u32)(n - 1); ++c) {
                const u64 r = s_rec[c];
                const u32 ab = s_ab[c];
                u32 ra = find_root(parent, ab >> 16), rb = find_root(parent, ab & 0xffffu);
                if (ra == rb) continue;
                // a component is born with its largest vertex (vertices enter in decreasing index,
                // PAPER.md:79); the younger component, the one with the smaller largest vertex, dies
                u32 dying = (maxv[ra] < maxv[rb]) ? ra : rb;
                u32 living = (dying == ra) ? rb : ra;
                out.pair_ts[m] = ((u64)(u32)r << 16) | (u64)maxv[dying];
                out.death[m] = __uint_as_float(~(u32)(r >> 32));
                parent[dying] = (u16)living;
                ++m;
            }
            s_merges = m;
        }
        __syncthreads();
        if (s_merges >= (u32)(n - 1)) break;
    }
    if (tid == 0) *out.n_pairs = s_merges;
}

} // namespace

cudaError_t launch_dim0(const u64* rec_sorted, i64 E, int n, u32 thr_bits_inv, u32* parent_maxv, Dim0Out out,
                        cudaStream_t st)
{
    const size_t bytes = ((size_t)n * 4 + 15) & ~(size_t)15;
    if (n <= 65535 && bytes <= 200 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(dim0_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e != cudaSuccess) return e;
        dim0_kernel<true><<<1, D0_THREADS, bytes, st>>>(rec_sorted, E, n, thr_bits_inv, parent_maxv, out);
    } else
        dim0_kernel<false><<<1, D0_THREADS, 0, st>>>(rec_sorted, E, n, thr_bits_inv, parent_maxv, out);
    return cudaGetLastError();
}
