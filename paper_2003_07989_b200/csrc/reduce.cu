// reduce.cu -- the reduction of the non-apparent columns on the device (not the hot
// path, timed separately).  The paper runs this "submatrix reduction" on the host (PAPER.md:244, :543,
// :549-561, Fig. 8-9); here it is four kernels:
//
//   prereduce_kernel   one WARP per column.  R[j] <- D_j ; while low(R[j]) is the row of an apparent pair
//                      (s', t): R[j] <- R[j] + D_{s'}.  An apparent column is reduced as it stands
//                       and precedes every other facet of its row in the coboundary
//                      order, so this needs nothing from the other non-apparent columns; at the paper-shaped
//                      workloads ~97 % of all column additions are of this kind.  The working column is an
//                      unsorted list of packed entries in shared memory, its pivot the largest entry of odd
//                      multiplicity (Z/2).  A column that ends on a row no apparent pair owns is PUBLISHED:
//                      its entries go to the arena (pivot first) and the pivot is its candidate.
//   claim_kernel       one thread per candidate: the second layer of the pair store, an
//                      open-addressing hash table row -> column, claimed with atomicMin on the column index.
//   worklist_kernel    the columns that lost their claim to an earlier column, or that the warp could not
//                      hold (more than PR_CAP entries, more than PR_MAX_ADDS additions), are flagged.
//   reduce_kernel      persistent CTAs take the flagged columns in coboundary order and run the standard
//                      reduction R_j <- R_j + R_i (Algorithm 1; by Lemma 3, PAPER.md:204,
//                      the same pairs as the oblivious Algorithm 2) with EXPLICIT reduced
//                      columns: sorted arrays of packed entries in a bump-allocated arena in HBM, immutable
//                      once published; column addition is a CTA-wide merge of two sorted arrays with equal
//                      entries cancelling (symmetric difference).  Columns are processed concurrently without
//                      locks: a column whose pivot row is free claims it with a compare-and-swap; if the row
//                      is owned by an EARLIER column, that column is added; if it is owned by a LATER column
//                      (which got there first), the earlier column takes the row and its worker goes on with
//                      the displaced column.  Only earlier columns are ever added to later ones, so the pairs
//                      are the unique ones of the reduction in coboundary order, whatever the schedule.
//
// Packed entry: ((key << tbits) | cidx(t)) + 1 -- never 0, so 0 can mark an empty slot; the pivot of a column,
// the cofacet that comes first in the filtration order (smallest diameter = largest key, then largest cidx,
// PAPER.md:77-79), is simply the largest entry.
#include "apparent.cuh"
#include "kernels.cuh"

namespace {

constexpr int PR_WARPS = 4;
constexpr int PR_THREADS = PR_WARPS * 32;
constexpr int PR_CAP = 2048;       // entries of a warp's working column
constexpr u32 PR_MAX_ADDS = 64;    // a warp that needs more leaves the column to reduce_kernel

constexpr int RD_THREADS = 256;
constexpr int RD_WARPS = RD_THREADS / 32;
constexpr int RD_IPT = 8;
constexpr int RD_TILE = RD_THREADS * RD_IPT;   // outputs per merge tile
constexpr u64 RD_BUF0 = 4096;                   // first capacity of a working buffer (entries)

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

__device__ __forceinline__ u64 ld_cg_u64(const u64* p)
{
    u64 v;
    asm volatile("ld.global.cg.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// ---- arena: bump allocation in units of 16 entries (128 bytes: no two columns share a cache line)
__device__ __forceinline__ u64 arena_alloc(const ReduceParams& p, u64 entries)
{
    const u64 need = (entries + 15ull) & ~15ull;
    const u64 off = atomicAdd((unsigned long long*)(p.counters + RDC_ARENA_TOP), (unsigned long long)need);
    if (off + need > p.arena_cap) {
        atomicOr((unsigned int*)p.error, RD_ERR_ARENA);
        return ~0ull;
    }
    return off;
}

// ---- the second layer of the pair store: row -> owning column
__device__ __forceinline__ u32 ht_hash(u64 t, u32 mask) { return (u32)((t * 0x9E3779B97F4A7C15ull) >> 24) & mask; }
__device__ __forceinline__ u32 ht_find_or_insert(const ReduceParams& p, u64 t)
{
    u32 s = ht_hash(t, p.ht_mask);
    for (u32 probes = 0;; ++probes) {
        if (probes > p.ht_mask) { atomicOr((unsigned int*)p.error, RD_ERR_PROTOCOL); return s; } // table full: cannot happen (capacity >= 2 x columns)
        u64 k = ld_volatile_u64(p.ht_keys + s);
        if (k == t) return s;
        if (k == ~0ull) {
            k = atomicCAS((unsigned long long*)(p.ht_keys + s), ~0ull, (unsigned long long)t);
            if (k == ~0ull || k == t) return s;
        }
        s = (s + 1) & p.ht_mask;
    }
}

// coboundary of s appended to the list (entries +1); returns the new length, or -1 if the list is full
template <int M, typename KT>
__device__ __forceinline__ int push_coboundary(const ReduceParams& p, const KT* __restrict__ Kf, const int (&s)[M], u64* list,
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

// ============================================================================== prereduce_kernel
template <int M, typename KT>
__global__ void __launch_bounds__(PR_THREADS) prereduce_kernel(const ReduceParams p)
{
    extern __shared__ __align__(16) unsigned char smem_pr[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    u64* list = reinterpret_cast<u64*>(smem_pr) + (size_t)warp * PR_CAP;
    const KT* __restrict__ Kf = reinterpret_cast<const KT*>(p.Kf);
    const u64 tmask = (1ull << p.tbits) - 1ull;
    u64 n_adds = 0;

    for (i64 col = (i64)blockIdx.x * PR_WARPS + warp; col < p.ncols; col += (i64)gridDim.x * PR_WARPS) {
        int s[M];
        unpack_vertices<M>(__ldg(p.cols + col), p.vbits, s);
        int len = push_coboundary<M, KT>(p, Kf, s, list, 0, lane);
        u64 result = 0; // 0: the column reduced to zero; ~0: left to reduce_kernel; else the candidate pivot
        u32 adds = 0;
        if (len < 0) result = ~0ull; // more cofacets than the warp's list holds
        while (len >= 0) {
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
            if (!hit) {
                // ---- a row no apparent pair owns: publish the column (pivot first, the rest unsorted) as this
                // column's candidate; whether another column wants the same row is settled by claim_kernel
                int live = 0;
                for (int base = 0; base < len; base += 32) {
                    const int i = base + lane;
                    const u64 e = i < len ? list[i] : 0;
                    const u32 bal = __ballot_sync(RIPS_FULL_MASK, e != 0);
                    __syncwarp();
                    if (e != 0) list[live + __popc(bal & ((1u << lane) - 1u))] = e;
                    live += __popc(bal);
                    __syncwarp();
                }
                u64 off = 0;
                if (lane == 0) off = arena_alloc(p, (u64)live + 1ull);
                off = __shfl_sync(RIPS_FULL_MASK, off, 0);
                if (off == ~0ull) { result = ~0ull; break; }
                u64* dst = p.arena + off;
                if (lane == 0) dst[0] = piv;
                for (int i = lane; i < live; i += 32) dst[1 + i] = list[i];
                __threadfence();
                __syncwarp();
                if (lane == 0) p.colref[col] = RD_REF(off, (u64)live + 1ull, 0);
                result = piv;
                break;
            }
            if (adds >= PR_MAX_ADDS) { result = ~0ull; break; }
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
            p.piv[col] = result; // 0 zero column, ~0 left to reduce_kernel, else the candidate pivot entry
            if (result != ~0ull) n_adds += adds; // a deferred column starts again from D_j
        }
        __syncwarp();
    }
    if (lane == 0 && n_adds) atomicAdd((unsigned long long*)(p.counters + RDC_ADDS), (unsigned long long)n_adds);
}

// ============================================================================== claim / worklist
__global__ void claim_kernel(const ReduceParams p)
{
    const i64 j = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= p.ncols) return;
    const u64 e = p.piv[j];
    if (e == 0 || e == ~0ull) return;
    const u64 tmask = (1ull << p.tbits) - 1ull;
    const u32 s = ht_find_or_insert(p, (e - 1ull) & tmask);
    atomicMin(p.ht_vals + s, (u32)j);
}

__global__ void worklist_kernel(const ReduceParams p)
{
    const i64 j = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= p.ncols) return;
    const u64 e = p.piv[j];
    unsigned char todo = 0;
    if (e == ~0ull) todo = 1;
    else if (e != 0) {
        const u64 tmask = (1ull << p.tbits) - 1ull;
        const u32 s = ht_find_or_insert(p, (e - 1ull) & tmask);
        todo = (p.ht_vals[s] != (u32)j) ? 1 : 0; // an earlier column claimed the same row
    }
    p.todo[j] = todo;
    if (todo) atomicAdd((unsigned long long*)(p.counters + RDC_TODO), 1ull);
}

// ============================================================================== reduce_kernel
constexpr int ACC_CAP = 2048;          // entries the shared-memory accumulator keeps before it is flushed to a run
constexpr int ACC_BUF = 2 * ACC_CAP;   // capacity of each of its two buffers (accumulator + one addition)
constexpr int X_SMEM_MAX = ACC_CAP;    // additions up to this size go through the accumulator
struct RdShared {
    u64* acc[2];      // the accumulator's two buffers (shared memory)
    int acc_sel, acc_pos, acc_len;
    u64* x;           // result of the last block_coboundary_sorted / block_sort_column (shared memory)
    u64 bc_u64[4];
    i64 bc_i64[4];
    int bc_int[8];
    u32 wsum[RD_WARPS];
    u32 cnt;
    int sv[RIPS_MAX_M];
};

// bitonic sort of sb[0..npow2), descending; empty slots (0) end up last
__device__ void block_sort_desc(u64* sb, int npow2)
{
    const int tid = threadIdx.x;
    for (int k = 2; k <= npow2; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int i = tid; i < npow2; i += RD_THREADS) {
                const int ixj = i ^ j;
                if (ixj > i) {
                    const u64 a = sb[i], b = sb[ixj];
                    const bool desc = (i & k) == 0;
                    if (desc ? (a < b) : (a > b)) { sb[i] = b; sb[ixj] = a; }
                }
            }
            __syncthreads();
        }
    }
}

// sb[0..cnt) (distinct entries) sorted descending.  Small counts by ranking (every thread counts the entries
// larger than its own: one barrier instead of the ~log^2 of a bitonic network); sh.x = where the result is.
__device__ void block_sort_distinct(u64* sb, int cnt, RdShared& sh)
{
    const int tid = threadIdx.x;
    if (cnt <= 1024) {
        u64* out = sb + 2048;
        for (int i = tid; i < cnt; i += RD_THREADS) {
            const u64 x = sb[i];
            int r = 0;
            for (int j = 0; j < cnt; ++j) r += (sb[j] > x) ? 1 : 0;
            out[r] = x;
        }
        if (tid == 0) sh.x = out;
        __syncthreads();
        return;
    }
    int np2 = 32;
    while (np2 < cnt) np2 <<= 1;
    for (int i = cnt + tid; i < np2; i += RD_THREADS) sb[i] = 0;
    __syncthreads();
    block_sort_desc(sb, np2);
    if (tid == 0) sh.x = sb;
    __syncthreads();
}

// the coboundary of the simplex sh.sv (entries +1) sorted descending, in shared memory at sh.x; returns the count
template <int M, typename KT>
__device__ int block_coboundary_sorted(const ReduceParams& p, const KT* __restrict__ Kf, RdShared& sh, u64* sb)
{
    const int tid = threadIdx.x;
    int s[M];
#pragma unroll
    for (int j = 0; j < M; ++j) s[j] = sh.sv[j];
    __syncthreads(); // sb may still be read as the previous addition
    if (tid == 0) sh.cnt = 0;
    __syncthreads();
    u32 key_s = 0xffffffffu;
#pragma unroll
    for (int a = 1; a < M; ++a)
#pragma unroll
        for (int b = 0; b < a; ++b) key_s = min(key_s, (u32)__ldg(Kf + s[a] * p.pitch + s[b]));
    const u32 thr1 = p.thr_key + 1u;
    for (int v = p.n - 1 - tid; v >= 0; v -= RD_THREADS) {
        u32 kt = key_s;
#pragma unroll
        for (int j = 0; j < M; ++j) kt = min(kt, (u32)__ldg(Kf + s[j] * p.pitch + v));
        if (kt != 0 && kt >= thr1) {
            int fseg = 0;
#pragma unroll
            for (int j = 0; j < M; ++j) fseg += (s[j] < v) ? 1 : 0;
            const u64 e = (((u64)(kt - 1u) << p.tbits) | cofacet_index<M>(p.bt, s, v, fseg)) + 1ull;
            const u32 pos = atomicAdd(&sh.cnt, 1u);
            if (pos < (u32)p.sort_cap) sb[pos] = e;
        }
    }
    __syncthreads();
    const int cnt = (int)sh.cnt;
    if (cnt > p.sort_cap) {
        if (tid == 0) atomicOr((unsigned int*)p.error, RD_ERR_SORTCAP);
        return -1;
    }
    block_sort_distinct(sb, cnt, sh);
    return cnt;
}

// A published but unsorted column (prereduce_kernel's, at most PR_CAP entries) as a sorted array of DISTINCT entries
// in shared memory at sh.x; returns its length.  The warp's list is a multiset (entries of even multiplicity
// cancel only once they are the largest), so after sorting every run of equal entries is reduced to its parity.
__device__ int block_sort_column(const ReduceParams& p, const u64* src, int len, u64* sb, RdShared& sh)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    int np2 = 32;
    while (np2 < len) np2 <<= 1;
    __syncthreads(); // sb may still be read as the previous addition
    for (int i = tid; i < np2; i += RD_THREADS) sb[i] = i < len ? ld_cg_u64(src + i) : 0ull;
    __syncthreads();
    block_sort_desc(sb, np2);
    u64* out_buf = sb + 2048;
    int out = 0;
    for (int base = 0; base < len; base += RD_THREADS) {
        const int i = base + tid;
        bool keep = false;
        u64 x = 0;
        if (i < len) {
            x = sb[i];
            if (i == 0 || sb[i - 1] != x) { // first of its run: survives iff the run is odd
                int r = 1;
                while (i + r < len && sb[i + r] == x) ++r;
                keep = (r & 1) != 0;
            }
        }
        const u32 bal = __ballot_sync(RIPS_FULL_MASK, keep);
        if (lane == 0) sh.wsum[warp] = __popc(bal);
        __syncthreads();
        u32 woff = 0, total = 0;
#pragma unroll
        for (int w = 0; w < RD_WARPS; ++w) {
            const u32 c = sh.wsum[w];
            if (w < warp) woff += c;
            total += c;
        }
        if (keep) out_buf[out + woff + __popc(bal & ((1u << lane) - 1u))] = x;
        out += (int)total;
        __syncthreads();
    }
    if (tid == 0) sh.x = out_buf;
    __syncthreads();
    return out;
}

// The accumulator: the newest part of the working column, a sorted run in SHARED memory.  acc <- acc xor X for a
// sorted X in shared memory (|acc| <= ACC_CAP, |X| <= X_SMEM_MAX): merge-path split per thread, up to
// ACC_BUF / RD_THREADS outputs per thread, survivors compacted into the other buffer.
__device__ void acc_merge(RdShared& sh, const u64* X, int xl)
{
    constexpr int IPT = ACC_BUF / RD_THREADS;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    __syncthreads();
    const u64* A = sh.acc[sh.acc_sel] + sh.acc_pos;
    u64* out = sh.acc[1 - sh.acc_sel];
    const int na = sh.acc_len - sh.acc_pos, nb = xl, tot = na + nb;
    const int per = (tot + RD_THREADS - 1) / RD_THREADS;
    const int d0 = min(tid * per, tot), d1 = min(d0 + per, tot);
    int lo = max(0, d0 - nb), hi = min(d0, na);
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (A[mid] >= X[d0 - 1 - mid]) lo = mid + 1;
        else hi = mid;
    }
    int i = lo, j = d0 - lo;
    u64 item[IPT];
    int nlive = 0;
#pragma unroll
    for (int k = 0; k < IPT; ++k) {
        item[k] = 0ull;
        if (d0 + k < d1) {
            const bool take_a = (j >= nb) || (i < na && A[i] >= X[j]);
            u64 x;
            bool dead;
            if (take_a) { x = A[i]; dead = (j < nb) && (X[j] == x); ++i; }
            else { x = X[j]; dead = (i > 0) && (A[i - 1] == x); ++j; }
            if (!dead) { item[k] = x; ++nlive; }
        }
    }
    u32 incl = (u32)nlive;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const u32 t = __shfl_up_sync(RIPS_FULL_MASK, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) sh.wsum[warp] = incl;
    __syncthreads();
    u32 woff = 0, total = 0;
#pragma unroll
    for (int w = 0; w < RD_WARPS; ++w) {
        const u32 c = sh.wsum[w];
        if (w < warp) woff += c;
        total += c;
    }
    u32 pos = woff + incl - (u32)nlive;
#pragma unroll
    for (int k = 0; k < IPT; ++k)
        if (item[k] != 0ull) out[pos++] = item[k];
    __syncthreads();
    if (tid == 0) { sh.acc_sel = 1 - sh.acc_sel; sh.acc_pos = 0; sh.acc_len = (int)total; }
    __syncthreads();
}

// dst <- A xor B (symmetric difference of two descending arrays of distinct entries); returns |dst|.
// Tiles of RD_TILE outputs: both windows staged in shared memory, a merge-path split per thread, RD_IPT
// outputs merged serially per thread, an entry present in both arrays dropped on both sides (with A first on
// ties the two copies are neighbours in the merged order, so each side sees the other by looking one step
// across), survivors compacted through shared memory and stored coalesced.
__device__ i64 block_merge_xor(const u64* A, i64 a, const u64* B, i64 b, u64* dst, u64* sm, RdShared& sh)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    u64* sA = sm;                    // [1 + RD_TILE]: sA[0] = the entry of A before the window
    u64* sB = sm + 1 + RD_TILE;      // [RD_TILE]
    i64 ia = 0, ib = 0, out = 0;
    while (ia < a || ib < b) {
        const int na = (int)min((i64)RD_TILE, a - ia), nb = (int)min((i64)RD_TILE, b - ib);
        for (int i = tid; i < na; i += RD_THREADS) sA[1 + i] = ld_cg_u64(A + ia + i);
        for (int i = tid; i < nb; i += RD_THREADS) sB[i] = ld_cg_u64(B + ib + i);
        if (tid == 0) sA[0] = ia > 0 ? ld_cg_u64(A + ia - 1) : 0ull;
        __syncthreads();
        const int tile_n = min(RD_TILE, na + nb);
        const int d0 = min(tid * RD_IPT, tile_n), d1 = min(d0 + RD_IPT, tile_n);
        int lo = max(0, d0 - nb), hi = min(d0, na);
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (sA[1 + mid] >= sB[d0 - 1 - mid]) lo = mid + 1;
            else hi = mid;
        }
        int i = lo, j = d0 - lo;
        u64 item[RD_IPT];
        int nlive = 0;
#pragma unroll
        for (int k = 0; k < RD_IPT; ++k) {
            if (d0 + k < d1) {
                const bool take_a = (j >= nb) || (i < na && sA[1 + i] >= sB[j]);
                u64 x;
                bool dead;
                if (take_a) { x = sA[1 + i]; dead = (j < nb) && (sB[j] == x); ++i; }
                else { x = sB[j]; dead = (sA[i] == x); ++j; } // sA[i] = the entry of A just before position i
                item[k] = dead ? 0ull : x;
                nlive += dead ? 0 : 1;
            } else
                item[k] = 0ull;
        }
        if (d1 == tile_n && d0 < d1) { sh.bc_int[0] = i; sh.bc_int[1] = j; }
        // exclusive scan of nlive over the block
        u32 incl = (u32)nlive;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const u32 t = __shfl_up_sync(RIPS_FULL_MASK, incl, o);
            if (lane >= o) incl += t;
        }
        __syncthreads(); // every thread is done reading the windows: they become the staging area
        if (lane == 31) sh.wsum[warp] = incl;
        __syncthreads();
        u32 woff = 0, total = 0;
#pragma unroll
        for (int w = 0; w < RD_WARPS; ++w) {
            const u32 c = sh.wsum[w];
            if (w < warp) woff += c;
            total += c;
        }
        u32 pos = woff + incl - (u32)nlive;
#pragma unroll
        for (int k = 0; k < RD_IPT; ++k)
            if (item[k] != 0ull) sm[pos++] = item[k];
        const int ca = sh.bc_int[0], cb = sh.bc_int[1];
        __syncthreads();
        for (u32 q = tid; q < total; q += RD_THREADS) dst[out + q] = sm[q];
        __syncthreads();
        out += total;
        ia += ca;
        ib += cb;
    }
    return out;
}

// Is row t (cidx of a simplex of M+1 vertices) the row of an apparent pair (s', t)?  Evaluated from Definition 5
// by warp 0 instead of searching the sorted layers: s' must be the youngest facet of t (the
// facet of diameter diam(t) with the smallest index = vertices removed in decreasing order, Algorithm 6) and t
// the oldest cofacet of s' of that diameter (the largest vertex v with every new edge no longer than diam(s')).
// An apparent s' is a birth simplex, so it is never cleared and (s', t) is in the pair store.  Result in
// sh.bc_int[2] (1 = apparent) and sh.sv (the vertices of s').
template <int M, typename KT>
__device__ void warp0_apparent_of_row(const ReduceParams& p, const KT* __restrict__ Kf, u64 t, RdShared& sh)
{
    const int lane = threadIdx.x & 31;
    int tv[M + 1];
    decode_simplex_fast<M + 1>(p.bt, t, p.n, tv);
    u32 pk[M + 1][M + 1];
    u32 key_t = 0xffffffffu;
#pragma unroll
    for (int a = 1; a <= M; ++a)
#pragma unroll
        for (int b = 0; b < a; ++b) {
            pk[a][b] = (u32)__ldg(Kf + tv[a] * p.pitch + tv[b]);
            key_t = min(key_t, pk[a][b]);
        }
    int drop = -1;
#pragma unroll
    for (int r = M; r >= 0; --r) { // facets in increasing index: remove the vertices in decreasing order
        u32 kf = 0xffffffffu;
#pragma unroll
        for (int a = 1; a <= M; ++a)
#pragma unroll
            for (int b = 0; b < a; ++b)
                if (a != r && b != r) kf = min(kf, pk[a][b]);
        if (drop < 0 && kf == key_t) drop = r;
    }
    int s[M];
    int vr = -1;
#pragma unroll
    for (int i = 0, m = 0; i <= M; ++i) {
        if (i == drop) vr = tv[i];
        else if (m < M) s[m++] = tv[i];
    }
    // the oldest cofacet of s' with its diameter: the largest v with every edge (v, s'_j) of key >= key_t
    int res = -1;
    if (drop >= 0) {
        for (int base = p.n - 1; base >= 0; base -= 32) {
            const int v = base - lane;
            bool ok = false;
            if (v >= 0) {
                u32 m = 0xffffffffu;
#pragma unroll
                for (int j = 0; j < M; ++j) m = min(m, (u32)__ldg(Kf + s[j] * p.pitch + v));
                ok = m >= key_t; // a vertex of s' reads the zero diagonal and fails by itself
            }
            const u32 bal = __ballot_sync(RIPS_FULL_MASK, ok);
            if (bal) { res = base - (__ffs(bal) - 1); break; }
        }
    }
    if (lane == 0) {
        sh.bc_int[2] = (drop >= 0 && res == vr) ? 1 : 0;
#pragma unroll
        for (int j = 0; j < M; ++j) sh.sv[j] = s[j];
    }
}

// ---------------------------------------------------------------------------------------------------------------
// The working column of one CTA: a set of RUNS, each a descending array of distinct entries, the column being
// their sum over Z/2 (an entry held by an even number of runs is absent).  Adding a column is appending a run --
// a reduced column of the arena by reference, a coboundary by copy -- so an addition costs what is added, not
// what the working column has grown to; the pivot is the largest run head of odd multiplicity.  Runs are kept
// geometrically decreasing in length (the last two are merged while the last is more than half the one before),
// so there are at most ~log2(entries) of them, one per lane of warp 0, and every entry is merged O(log) times.
// Runs the CTA made itself live in a private stack buffer (merges go through a private scratch buffer and back);
// both grow by doubling.  Only the finished column is copied into an arena allocation of its exact size.
// ---------------------------------------------------------------------------------------------------------------
constexpr int WS_MAX_RUNS = 31;   // lane 31 of warp 0 looks after the shared-memory accumulator
struct WorkSet {
    const u64* ptr[WS_MAX_RUNS];
    u32 pos[WS_MAX_RUNS], len[WS_MAX_RUNS];
    u64 head[WS_MAX_RUNS];          // entry at pos, 0 = the run is used up
    u64 win[WS_MAX_RUNS][8];        // entries [wbase, wbase + 8) of the run, read ahead so that consuming an entry is not a trip to HBM
    u32 wbase[WS_MAX_RUNS];         // 0xffffffff = nothing read ahead
    unsigned char own[WS_MAX_RUNS]; // the run lives in the private stack
    int nruns;
    u64 a_off, a_cap;               // private stack (arena offset, capacity in entries)
    u64 b_off, b_cap;               // private scratch
    u64 pivot;                      // result of ws_peek
};

__device__ __forceinline__ void block_copy(u64* dst, const u64* src, u64 n)
{
    for (u64 i = threadIdx.x; i < n; i += RD_THREADS) dst[i] = ld_cg_u64(src + i);
}
__device__ __forceinline__ void block_copy_from_shared(u64* dst, const u64* src, u64 n)
{
    for (u64 i = threadIdx.x; i < n; i += RD_THREADS) dst[i] = src[i];
}

// entries of the private stack in use: up to the end of the last run that lives in it
__device__ __forceinline__ u64 ws_top(const ReduceParams& p, const WorkSet& ws)
{
    for (int r = ws.nruns - 1; r >= 0; --r)
        if (ws.own[r]) return (u64)(ws.ptr[r] - (p.arena + ws.a_off)) + ws.len[r];
    return 0;
}

// private buffer `which` (0 = stack, 1 = scratch) of at least `need` entries; the stack keeps its contents
__device__ bool ws_reserve(const ReduceParams& p, WorkSet& ws, int which, u64 need, RdShared& sh)
{
    const u64 cap0 = which ? ws.b_cap : ws.a_cap;
    if (cap0 >= need) return true;
    u64 cap = cap0 ? cap0 : RD_BUF0;
    while (cap < need) cap <<= 1;
    __syncthreads();
    if (threadIdx.x == 0) sh.bc_u64[3] = arena_alloc(p, cap);
    __syncthreads();
    const u64 off = sh.bc_u64[3];
    if (off == ~0ull) return false;
    if (which == 0) {
        const u64* old_base = p.arena + ws.a_off;
        u64* new_base = p.arena + off;
        const u64 top = ws_top(p, ws);
        if (top) block_copy(new_base, old_base, top);
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int r = 0; r < ws.nruns; ++r)
                if (ws.own[r]) ws.ptr[r] = new_base + (ws.ptr[r] - old_base);
            ws.a_off = off;
            ws.a_cap = cap;
        }
    } else if (threadIdx.x == 0) {
        ws.b_off = off;
        ws.b_cap = cap;
    }
    __syncthreads();
    return true;
}

// drop the runs that are used up (order kept); thread 0 only, between barriers
__device__ __forceinline__ void ws_prune_t0(WorkSet& ws)
{
    int w = 0;
    for (int r = 0; r < ws.nruns; ++r) {
        if (ws.head[r] == 0ull) continue;
        if (w != r) { ws.ptr[w] = ws.ptr[r]; ws.pos[w] = ws.pos[r]; ws.len[w] = ws.len[r]; ws.head[w] = ws.head[r]; ws.own[w] = ws.own[r]; ws.wbase[w] = 0xffffffffu; }
        ++w;
    }
    ws.nruns = w;
}

// the last two runs merged into one (their unused parts; equal entries cancel); the result lives in the stack
__device__ bool ws_merge_last_two(const ReduceParams& p, WorkSet& ws, u64* sm, RdShared& sh)
{
    const int k = ws.nruns;
    const u64* A = ws.ptr[k - 2] + ws.pos[k - 2];
    const u64* B = ws.ptr[k - 1] + ws.pos[k - 1];
    const i64 a = (i64)ws.len[k - 2] - ws.pos[k - 2], b = (i64)ws.len[k - 1] - ws.pos[k - 1];
    if (!ws_reserve(p, ws, 1, (u64)(a + b), sh)) return false;
    const i64 out = block_merge_xor(A, a, B, b, p.arena + ws.b_off, sm, sh);
#ifdef RIPS_REDUCE_PROFILE
    if (threadIdx.x == 0) atomicAdd((unsigned long long*)(p.counters + RDC_DBG + 5), (unsigned long long)((a + b + RD_TILE - 1) / RD_TILE));
#endif
    __syncthreads();
    if (threadIdx.x == 0) ws.nruns = k - 2; // both inputs are gone: the stack ends below them
    __syncthreads();
    if (out == 0) return true;
    const u64 top = ws_top(p, ws);
    if (!ws_reserve(p, ws, 0, top + (u64)out, sh)) return false;
    u64* dst = p.arena + ws.a_off + top;
    block_copy(dst, p.arena + ws.b_off, (u64)out);
    __syncthreads();
    if (threadIdx.x == 0) {
        const int r = ws.nruns;
        ws.ptr[r] = dst; ws.pos[r] = 0; ws.len[r] = (u32)out; ws.own[r] = 1; ws.head[r] = ld_cg_u64(dst); ws.wbase[r] = 0xffffffffu;
        ws.nruns = r + 1;
    }
    __syncthreads();
    return true;
}

// restore the geometric run lengths (and room for one more run)
__device__ bool ws_balance(const ReduceParams& p, WorkSet& ws, u64* sm, RdShared& sh)
{
    for (;;) {
        __syncthreads();
        const int k = ws.nruns;
        if (k < 2) return true;
        const u64 last = (u64)ws.len[k - 1] - ws.pos[k - 1], prev = (u64)ws.len[k - 2] - ws.pos[k - 2];
        if (2 * last <= prev && k < WS_MAX_RUNS - 1) return true;
        if (!ws_merge_last_two(p, ws, sm, sh)) return false;
    }
}

// append a run by reference (an immutable sorted column of the arena)
__device__ bool ws_push_ref(const ReduceParams& p, WorkSet& ws, const u64* src, i64 len, u64* sm, RdShared& sh)
{
    __syncthreads();
    if (len > 0 && threadIdx.x == 0) {
        ws_prune_t0(ws);
        const int r = ws.nruns;
        ws.ptr[r] = src; ws.pos[r] = 0; ws.len[r] = (u32)len; ws.own[r] = 0; ws.head[r] = ld_cg_u64(src); ws.wbase[r] = 0xffffffffu;
        ws.nruns = r + 1;
    }
    __syncthreads();
    return ws_balance(p, ws, sm, sh);
}

// append a run by copy (from shared memory) into the private stack
__device__ bool ws_push_copy(const ReduceParams& p, WorkSet& ws, const u64* src, i64 len, u64* sm, RdShared& sh)
{
    if (len <= 0) return true;
    __syncthreads();
    if (threadIdx.x == 0) ws_prune_t0(ws);
    __syncthreads();
    const u64 top = ws_top(p, ws);
    if (!ws_reserve(p, ws, 0, top + (u64)len, sh)) return false;
    u64* dst = p.arena + ws.a_off + top;
    block_copy_from_shared(dst, src, (u64)len);
    __syncthreads();
    if (threadIdx.x == 0) {
        const int r = ws.nruns;
        ws.ptr[r] = dst; ws.pos[r] = 0; ws.len[r] = (u32)len; ws.own[r] = 1; ws.head[r] = src[0]; ws.wbase[r] = 0xffffffffu;
        ws.nruns = r + 1;
    }
    __syncthreads();
    return ws_balance(p, ws, sm, sh);
}

// the accumulator becomes a run of the private stack
__device__ bool acc_flush(const ReduceParams& p, WorkSet& ws, u64* sm, RdShared& sh)
{
    __syncthreads();
    const int n = sh.acc_len - sh.acc_pos;
    if (n <= 0) return true;
#ifdef RIPS_REDUCE_PROFILE
    if (threadIdx.x == 0) atomicAdd((unsigned long long*)(p.counters + RDC_DBG + 5), 1ull << 40);
#endif
    const u64* src = sh.acc[sh.acc_sel] + sh.acc_pos;
    if (!ws_push_copy(p, ws, src, n, sm, sh)) return false;
    if (threadIdx.x == 0) { sh.acc_pos = 0; sh.acc_len = 0; }
    __syncthreads();
    return true;
}

// working column += X (sorted, distinct, in shared memory at sh.x)
__device__ bool ws_add_shared(const ReduceParams& p, WorkSet& ws, int xl, u64* sm, RdShared& sh)
{
    if (xl <= 0) return true;
    if (xl <= X_SMEM_MAX) {
        acc_merge(sh, sh.x, xl);
        if (sh.acc_len - sh.acc_pos > ACC_CAP) return acc_flush(p, ws, sm, sh);
        return true;
    }
    return ws_push_copy(p, ws, sh.x, xl, sm, sh); // a coboundary larger than the accumulator takes: a run of its own
}

// ws.pivot <- the largest entry of odd multiplicity (it stays where it is), 0 if the column is zero; entries of
// even multiplicity met on the way are consumed.  Warp 0 works, one lane per run, lane 31 for the accumulator.
__device__ void ws_peek(WorkSet& ws, RdShared& sh)
{
    __syncthreads();
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        const bool is_acc = lane == 31;
        const bool act = is_acc || lane < ws.nruns;
        u32 pos = is_acc ? (u32)sh.acc_pos : (act ? ws.pos[lane] : 0u);
        const u32 len = is_acc ? (u32)sh.acc_len : (act ? ws.len[lane] : 0u);
        const u64* ptr = is_acc ? sh.acc[sh.acc_sel] : (act ? ws.ptr[lane] : nullptr);
        u64 h = is_acc ? (pos < len ? ptr[pos] : 0ull) : (act ? ws.head[lane] : 0ull);
        u64 m;
        for (;;) {
            // the largest head: two 32-bit warp maxima (redux.sync) instead of a 64-bit butterfly of shuffles -- this loop
            // runs once per consumed entry and is the longest part of an addition of a long chain
            const u32 hh = (u32)(h >> 32);
            const u32 mh = __reduce_max_sync(RIPS_FULL_MASK, hh);
            const u32 ml = __reduce_max_sync(RIPS_FULL_MASK, hh == mh ? (u32)h : 0u);
            m = ((u64)mh << 32) | (u64)ml;
            if (m == 0ull) break;
            const bool mine = (h == m);
            const u32 bal = __ballot_sync(RIPS_FULL_MASK, mine);
            if (__popc(bal) & 1) break;
            if (mine) {
                ++pos;
                if (pos >= len) h = 0ull;
                else if (is_acc) h = ptr[pos];
                else {
                    u32 wb = ws.wbase[lane];
                    if (wb == 0xffffffffu || pos - wb >= 8u) {
                        wb = pos;
#pragma unroll
                        for (int k = 0; k < 8; ++k) ws.win[lane][k] = (pos + k < len) ? ld_cg_u64(ptr + pos + k) : 0ull;
                        ws.wbase[lane] = wb;
                    }
                    h = ws.win[lane][pos - wb];
                }
            }
        }
        if (is_acc) sh.acc_pos = (int)pos;
        else if (act) { ws.head[lane] = h; ws.pos[lane] = pos; }
        if (lane == 0) ws.pivot = m;
    }
    __syncthreads();
}

// all runs merged into one; returns its length (0: zero column), the run is ws run 0
__device__ i64 ws_collapse(const ReduceParams& p, WorkSet& ws, u64* sm, RdShared& sh)
{
    if (!acc_flush(p, ws, sm, sh)) return -1;
    __syncthreads();
    if (threadIdx.x == 0) ws_prune_t0(ws);
    __syncthreads();
    while (ws.nruns >= 2) {
        if (!ws_merge_last_two(p, ws, sm, sh)) return -1;
        __syncthreads();
    }
    if (ws.nruns == 0) return 0;
    return (i64)ws.len[0] - ws.pos[0];
}

template <int M, typename KT>
__global__ void __launch_bounds__(RD_THREADS) reduce_kernel(const ReduceParams p)
{
    extern __shared__ __align__(16) unsigned char smem_rd[];
    __shared__ RdShared sh;
    __shared__ WorkSet ws;
    u64* sm = reinterpret_cast<u64*>(smem_rd);   // sort buffer / merge staging: max(sort_cap, 2 * RD_TILE + 1) entries
    const KT* __restrict__ Kf = reinterpret_cast<const KT*>(p.Kf);
    const int tid = threadIdx.x;
    const u64 tmask = (1ull << p.tbits) - 1ull;
    if (tid == 0) {
        u64* accbase = sm + max(p.sort_cap, 2 * RD_TILE + 2);
        sh.acc[0] = accbase;
        sh.acc[1] = accbase + ACC_BUF;
        sh.acc_sel = sh.acc_pos = sh.acc_len = 0;
        ws.nruns = 0; ws.a_off = ws.b_off = 0; ws.a_cap = ws.b_cap = 0; ws.pivot = 0;
    }
    u64 n_adds = 0, n_steals = 0;
#ifdef RIPS_REDUCE_PROFILE
    long long tp[6] = {0, 0, 0, 0, 0, 0}, t_a, t_b;
#define TP(i) do { t_b = clock64(); tp[i] += t_b - t_a; t_a = t_b; } while (0)
#else
#define TP(i) do { } while (0)
#endif

    for (;;) {
        // ---- next flagged column, in coboundary order (32 columns per ticket)
        __syncthreads();
        if (tid == 0) sh.bc_i64[0] = (i64)atomicAdd((unsigned long long*)(p.counters + RDC_TICKET), 1ull) * 32;
        __syncthreads();
        const i64 first = sh.bc_i64[0];
        if (first >= p.ncols) break;
        for (int q = 0; q < 32; ++q) {
            const i64 j0 = first + q;
            if (j0 >= p.ncols) break;
            if (!p.todo[j0]) continue;
            if (*((volatile u32*)p.error)) goto fail;
            i64 cur = j0;
            // ---- W <- the column as prereduce_kernel left it (published, unsorted), or D_j
            __syncthreads();
            if (tid == 0) { ws.nruns = 0; sh.acc_pos = sh.acc_len = 0; }
            __syncthreads();
            {
                const u64 e = p.piv[cur];
                int cnt;
                if (e != ~0ull) {
                    const u64 ref = p.colref[cur];
                    cnt = block_sort_column(p, p.arena + RD_REF_OFF(ref), (int)RD_REF_LEN(ref), sm, sh);
                } else {
                    if (tid < M) {
                        const u64 rec = __ldg(p.cols + cur);
                        sh.sv[tid] = (int)((u32)(rec >> (tid * p.vbits)) & ((1u << p.vbits) - 1u));
                    }
                    __syncthreads();
                    cnt = block_coboundary_sorted<M, KT>(p, Kf, sh, sm);
                }
                if (cnt < 0) goto fail;
                if (!ws_add_shared(p, ws, cnt, sm, sh)) goto fail;
            }
            // ---- the reduction of column `cur` (and of the columns it displaces)
            u32 rounds = 0;
            for (;;) {
                if (++rounds > (1u << 24)) { // cannot happen (every round removes the pivot or ends the column): never spin
                    if (tid == 0 && !(atomicOr((unsigned int*)p.error, RD_ERR_STUCK) & RD_ERR_STUCK)) {
                        p.counters[RDC_DBG + 0] = (u64)cur; p.counters[RDC_DBG + 1] = (u64)ws.nruns;
                        p.counters[RDC_DBG + 2] = ws.pivot; p.counters[RDC_DBG + 3] = (u64)j0;
                    }
                    goto fail;
                }
#ifdef RIPS_REDUCE_PROFILE
                t_a = clock64();
#endif
                ws_peek(ws, sh);
                TP(0);
                const u64 pe = ws.pivot; // the pivot entry (+1)
                if (pe == 0ull) { // zero column: an essential class
                    if (tid == 0) p.piv[cur] = 0;
                    break;
                }
                const u64 t = (pe - 1ull) & tmask;
                // (1) the row of an apparent pair: R <- R + D_{s'}
                if (tid < 32) warp0_apparent_of_row<M, KT>(p, Kf, t, sh);
                __syncthreads();
                TP(1);
                if (sh.bc_int[2]) {
                    const int cnt = block_coboundary_sorted<M, KT>(p, Kf, sh, sm);
                    TP(2);
                    if (cnt < 0) goto fail;
                    if (!ws_add_shared(p, ws, cnt, sm, sh)) goto fail;
                    TP(3);
                    ++n_adds;
                    continue;
                }
                // (2) the second layer: claim the row, add its earlier owner, or displace its later owner
                if (tid == 0) {
                    const u32 slot = ht_find_or_insert(p, t);
                    sh.bc_int[3] = (int)slot;
                    sh.bc_u64[0] = (u64)*((volatile u32*)(p.ht_vals + slot));
                }
                __syncthreads();
                const u32 slot = (u32)sh.bc_int[3];
                const u32 owner = (u32)sh.bc_u64[0];
                bool steal = false;
                if (owner == 0xffffffffu || (i64)owner > cur) {
                    // publish R_cur (everything merged into one array of an arena allocation of its size), then take the row
                    i64 rlen;
                    const u64* rsrc;
                    bool from_acc = false;
                    if (ws.nruns == 0) { rlen = sh.acc_len - sh.acc_pos; rsrc = sh.acc[sh.acc_sel] + sh.acc_pos; from_acc = true; }
                    else {
                        rlen = ws_collapse(p, ws, sm, sh);
                        rsrc = rlen > 0 ? ws.ptr[0] + ws.pos[0] : nullptr;
                    }
                    if (rlen <= 0) { if (tid == 0) atomicOr((unsigned int*)p.error, RD_ERR_PROTOCOL); goto fail; }
                    if (tid == 0) sh.bc_u64[1] = arena_alloc(p, (u64)rlen);
                    __syncthreads();
                    const u64 roff = sh.bc_u64[1];
                    if (roff == ~0ull) goto fail;
                    if (from_acc) block_copy_from_shared(p.arena + roff, rsrc, (u64)rlen);
                    else block_copy(p.arena + roff, rsrc, (u64)rlen);
                    __threadfence();
                    __syncthreads();
                    if (tid == 0) {
                        p.colref[cur] = RD_REF(roff, (u64)rlen, 1);
                        p.piv[cur] = pe;
                        __threadfence();
                        stress_jitter((u32)cur);
                        sh.bc_u64[1] = (u64)atomicCAS(p.ht_vals + slot, owner, (u32)cur);
                        // the working column is now that published copy, by reference
                        ws.ptr[0] = p.arena + roff; ws.pos[0] = 0; ws.len[0] = (u32)rlen; ws.own[0] = 0; ws.head[0] = pe; ws.wbase[0] = 0xffffffffu; ws.nruns = 1;
                        sh.acc_pos = sh.acc_len = 0;
                    }
                    __syncthreads();
                    if ((u32)sh.bc_u64[1] != owner) continue; // someone else moved first: look again
                    if (owner == 0xffffffffu) break;           // claimed: column `cur` is reduced
                    steal = true;                              // the row's later owner is displaced: go on with it
                    ++n_steals;
                }
                // the column to add: R_owner (an earlier column), or R_displaced, which R_cur is added to
                if (tid == 0) sh.bc_u64[2] = ld_volatile_u64(p.colref + owner);
                __syncthreads();
                const u64 ref = sh.bc_u64[2];
                const u64* R = p.arena + RD_REF_OFF(ref);
                const i64 rl = (i64)RD_REF_LEN(ref);
                if (ld_cg_u64(R) != pe) { // a version of that column from after it lost this row: look again
                    if (steal) { if (tid == 0) atomicOr((unsigned int*)p.error, RD_ERR_PROTOCOL); goto fail; }
                    continue;
                }
                if (!RD_REF_SORTED(ref)) {
                    const int xl = block_sort_column(p, R, (int)rl, sm, sh);
                    if (!ws_add_shared(p, ws, xl, sm, sh)) goto fail;
                } else if (rl <= X_SMEM_MAX) {
                    __syncthreads(); // sm may still be read as the previous addition
                    for (int i = tid; i < (int)rl; i += RD_THREADS) sm[i] = ld_cg_u64(R + i);
                    if (tid == 0) sh.x = sm;
                    __syncthreads();
                    if (!ws_add_shared(p, ws, (int)rl, sm, sh)) goto fail;
                } else {
                    if (!ws_push_ref(p, ws, R, rl, sm, sh)) goto fail;
                }
                if (steal) cur = (i64)owner;
                ++n_adds;
                TP(4);
            }
        }
    }
fail:
#ifdef RIPS_REDUCE_PROFILE
    if (tid == 0) for (int i = 0; i < 5; ++i) atomicAdd((unsigned long long*)(p.counters + RDC_DBG + i), (unsigned long long)tp[i]);
#endif
    if (tid == 0) {
        if (n_adds) atomicAdd((unsigned long long*)(p.counters + RDC_ADDS), (unsigned long long)n_adds);
        if (n_steals) atomicAdd((unsigned long long*)(p.counters + RDC_STEALS), (unsigned long long)n_steals);
    }
}

// ============================================================================== results
// rec[j] = (cidx(t) << jbits) | j for the columns with a pivot, all ones for the zero columns (sorted last)
__global__ void pivot_records_kernel(const ReduceParams p, int jbits, u64* rec)
{
    const i64 j = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= p.ncols) return;
    const u64 e = p.piv[j];
    const u64 tmask = (1ull << p.tbits) - 1ull;
    if (e == 0) { rec[j] = ~0ull; return; }
    rec[j] = (((e - 1ull) & tmask) << jbits) | (u64)j;
    atomicAdd((unsigned long long*)(p.counters + RDC_PIVOTS), 1ull);
}

template <int M>
__global__ void pivot_arrays_kernel(const ReduceParams p, int jbits, const u64* __restrict__ rec, i64 n_piv, u64* t_out, u64* s_out)
{
    const i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_piv) return;
    const u64 r = __ldg(rec + i);
    const i64 j = (i64)(r & ((1ull << jbits) - 1ull));
    int s[M];
    unpack_vertices<M>(__ldg(p.cols + j), p.vbits, s);
    u64 c = 0;
#pragma unroll
    for (int k = 0; k < M; ++k) c += p.bt(s[k], k + 1); // Eq. 2
    t_out[i] = r >> jbits;
    s_out[i] = c;
}

// bars in column order: (birth, death) of every column whose pivot has another diameter, (birth, +inf) of every
// zero column.  One CTA, ordered compaction.
__global__ void __launch_bounds__(1024) bars_kernel(const ReduceParams p, int lowbits, const float* __restrict__ values,
                                                    float* bars, u64* n_bars, u64* n_essential)
{
    __shared__ u32 s_w[32];
    __shared__ u64 s_base;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_base = 0;
    u64 ess = 0;
    __syncthreads();
    for (i64 base = 0; base < p.ncols; base += 1024) {
        const i64 j = base + tid;
        bool has = false;
        float b = 0.f, d = 0.f;
        if (j < p.ncols) {
            const u64 e = p.piv[j];
            const u32 key_s = (u32)(__ldg(p.cols + j) >> lowbits);
            b = __ldg(values + key_s);
            if (e == 0) { has = true; d = __int_as_float(0x7f800000); ++ess; }
            else {
                const u32 key_t = (u32)((e - 1ull) >> p.tbits);
                if (key_t != key_s) { has = true; d = __ldg(values + key_t); }
            }
        }
        const u32 bal = __ballot_sync(RIPS_FULL_MASK, has);
        if (lane == 0) s_w[warp] = __popc(bal);
        __syncthreads();
        u32 off = 0, tot = 0;
        for (int w = 0; w < 32; ++w) {
            const u32 c = s_w[w];
            if (w < warp) off += c;
            tot += c;
        }
        const u64 at = s_base + off + __popc(bal & ((1u << lane) - 1u));
        if (has) { bars[2 * at] = b; bars[2 * at + 1] = d; }
        __syncthreads();
        if (tid == 0) s_base += tot;
        __syncthreads();
    }
    ess = warp_sum_u64(ess);
    if (lane == 0 && ess) atomicAdd((unsigned long long*)n_essential, (unsigned long long)ess);
    if (tid == 0) *n_bars = s_base;
}

template <int M, typename KT>
cudaError_t launch_reduce_t(const ReduceParams& p, int sms, cudaStream_t st)
{
    {
        const size_t smem = (size_t)PR_WARPS * PR_CAP * 8;
        auto kern = prereduce_kernel<M, KT>;
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        i64 g = (p.ncols + PR_WARPS - 1) / PR_WARPS;
        if (g > (i64)sms * 24) g = (i64)sms * 24;
        kern<<<(unsigned)g, PR_THREADS, smem, st>>>(p);
    }
    const unsigned gb = (unsigned)((p.ncols + 255) / 256);
    claim_kernel<<<gb, 256, 0, st>>>(p);
    worklist_kernel<<<gb, 256, 0, st>>>(p);
    {
        const size_t smem = reduce_smem_bytes(p.sort_cap);
        auto kern = reduce_kernel<M, KT>;
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        kern<<<(unsigned)p.workers, RD_THREADS, smem, st>>>(p);
    }
    return cudaGetLastError();
}

} // namespace

size_t reduce_smem_bytes(int sort_cap)
{   // sort buffer / merge staging, then the accumulator's two buffers
    const size_t a = (size_t)sort_cap * 8, b = (size_t)(2 * RD_TILE + 2) * 8;
    return (a > b ? a : b) + (size_t)2 * ACC_BUF * 8;
}

int reduce_sort_cap(int n)
{
    int c = 2048; // a column published by prereduce_kernel has at most PR_CAP entries
    while (c < n) c <<= 1;
    return c;
}

int reduce_workers(int sms, int sort_cap)
{
    const size_t smem = reduce_smem_bytes(sort_cap);
    int per_sm = (int)((200u * 1024u) / (smem + 1024));
    if (per_sm < 1) per_sm = 1;
    if (per_sm > 4) per_sm = 4;
    return sms * per_sm;
}

cudaError_t launch_reduce(int M, int kf_u16, const ReduceParams& p, int sms, cudaStream_t st)
{
    if (p.ncols == 0) return cudaSuccess;
#define RD_CASE(MM)                                                                          \
    case MM: return kf_u16 ? launch_reduce_t<MM, unsigned short>(p, sms, st) : launch_reduce_t<MM, u32>(p, sms, st);
    switch (M) {
        RD_CASE(2) RD_CASE(3) RD_CASE(4) RD_CASE(5) RD_CASE(6)
    default: return cudaErrorInvalidValue;
    }
#undef RD_CASE
}

cudaError_t launch_pivot_records(const ReduceParams& p, int jbits, u64* rec, cudaStream_t st)
{
    if (p.ncols == 0) return cudaSuccess;
    pivot_records_kernel<<<(unsigned)((p.ncols + 255) / 256), 256, 0, st>>>(p, jbits, rec);
    return cudaGetLastError();
}

cudaError_t launch_pivot_arrays(int M, const ReduceParams& p, int jbits, const u64* rec, i64 n_piv, u64* t_out, u64* s_out,
                                cudaStream_t st)
{
    if (n_piv == 0) return cudaSuccess;
    const unsigned g = (unsigned)((n_piv + 255) / 256);
    switch (M) {
    case 2: pivot_arrays_kernel<2><<<g, 256, 0, st>>>(p, jbits, rec, n_piv, t_out, s_out); break;
    case 3: pivot_arrays_kernel<3><<<g, 256, 0, st>>>(p, jbits, rec, n_piv, t_out, s_out); break;
    case 4: pivot_arrays_kernel<4><<<g, 256, 0, st>>>(p, jbits, rec, n_piv, t_out, s_out); break;
    case 5: pivot_arrays_kernel<5><<<g, 256, 0, st>>>(p, jbits, rec, n_piv, t_out, s_out); break;
    case 6: pivot_arrays_kernel<6><<<g, 256, 0, st>>>(p, jbits, rec, n_piv, t_out, s_out); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

cudaError_t launch_bars(const ReduceParams& p, int lowbits, const float* values, float* bars, u64* n_bars, u64* n_essential,
                        cudaStream_t st)
{
    bars_kernel<<<1, 1024, 0, st>>>(p, lowbits, values, bars, n_bars, n_essential);
    return cudaGetLastError();
}
