// stage1.cu -- the fused hot kernel: steps a3-a5 (enumerate + diameter + threshold + clearing +
// compaction, Algorithms 7-8) and a7 (the apparent-pair test, Algorithm 3 /
// Lemma 7) in one pass over the candidate index space.
//
// Redesign against the paper (which launches one thread per candidate with a binary-search decode,
// PAPER.md:359, :605, sorts, and only then runs one thread per sorted column):
//   * a warp owns a chunk of consecutive combinatorial indices and walks it row by row: a row fixes
//     the vertices v[M-1] > ... > v[1] (warp-uniform) and the lanes take consecutive lowest
//     vertices v[0].  What depends only on the row -- the keys among the upper vertices, and
//     U[v] = min_j key(v_j, v) for the 32 highest v, the part of every cofacet test the row shares --
//     is computed once per row; each lane adds one read of its own row of Kf.
//   * the apparent test of a column is independent of the column order (Corollary 8, PAPER.md:
//     297-299; Prop. 10), so it runs here, where the column's vertices and key are
//     in registers, in increasing cidx.  In that order the regular pairs (apparent.cuh) need a single
//     stable partition by v to be sorted by cidx(t), instead of a full radix sort of 31+ bits.
//   * lanes whose scan leaves the 32-vertex window, or stops below the top vertex of s (the facet
//     test is then needed), go to a small per-warp queue that the warp drains cooperatively, 32
//     cofacet vertices per step: the long tail of the scan never serialises a warp.
//   * without a threshold (>= 98 % survive) every candidate keeps its slot and dropped ones get a
//     sentinel that the sort sinks (the paper's device): no compaction, fully
//     coalesced stores.  With a threshold survivors are compacted in increasing index with a
//     warp-level decoupled look-back.
//   * the digit histograms of the two sorts that follow are accumulated on the way out.
#include <algorithm>

#include "apparent.cuh"
#include "kernels.cuh"

namespace {

constexpr int S1_THREADS = 1024;
constexpr int S1_WARPS = S1_THREADS / 32;
constexpr int S1_QCAP = 64;     // slot kernel: entries of a warp's queue of open cofacet scans (31 waiting + 32 new at most)
constexpr int S1_QVISITS = 12;  // cofacet vertices every drained candidate tests on its own before the warp takes its scan over
constexpr int S1_CHUNK = 1024;         // most candidates per warp chunk (unit of work and of the look-back chain)
constexpr int S1_MAX_FUSED = 3;        // digits of the filtration sort histogrammed on the way out
constexpr int S1_MAX_FUSED_P = 2;      // digits of the pair partition
constexpr size_t S1_KF_SMEM_LIMIT = 100 * 1024;  // two blocks per SM

__device__ __forceinline__ bool in_sorted(const u64* __restrict__ a, i64 n, int shift, u64 x)
{
    i64 lo = 0, hi = n;
    while (lo < hi) {
        i64 mid = lo + ((hi - lo) >> 1);
        if ((__ldg(a + mid) >> shift) < x) lo = mid + 1;
        else hi = mid;
    }
    return lo < n && (__ldg(a + lo) >> shift) == x;
}

// a lane's pair (v1, x), x < v1, 32 positions further in the order e = C(v1, 2) + x
__device__ __forceinline__ void lane_advance(int& v1, int& x)
{
    x += 32;
    while (x >= v1) { x -= v1; ++v1; }
}

// shared-memory digit histograms of one block
struct BlockHists {
    u32 (*cols)[256];   // [S1_MAX_FUSED][256]
    u32 (*pairs)[256];  // [S1_MAX_FUSED_P][256]
    int ncols, npairs;
    int csh[S1_MAX_FUSED];
    u32 cmk[S1_MAX_FUSED];
    int psh[S1_MAX_FUSED_P];
    u32 pmk[S1_MAX_FUSED_P];
};

// The warp's scan of the cofacet vertices base, base-1, ..., 0 of one simplex (rows Kf + xs and Kf + v1s of its two
// lowest vertices xq < v1q; `extra(v)` is the part of the test its other vertices contribute), guided by the block
// maxima Sf (init.cu, build_block_max_kernel): lane l reads the maxima of block bt - l of both rows, and only blocks
// whose maximum reaches ks in BOTH rows are read vertex by vertex, four blocks per round (their loads independent),
// from the top.  Returns the largest vertex <= base | 31 that passes, or -1.  Vertices above `base` in the first block
// were tested by the caller and fail again.  With keys of a random matrix a column without such a cofacet costs
// n / 512 coalesced loads instead of n / 16: the scan of all n vertices is what binds the fused kernel when n is in
// the thousands (Section 6.6's workload).  Every lane of the warp must call it with the same arguments.
template <typename KT, typename EX>
__device__ __forceinline__ int summary_scan(const KT* __restrict__ Kf, const KT* __restrict__ Sf, const int spitch, const int n,
                                            const int xs, const int v1s, const int xq, const int v1q, const u32 ks, const int base,
                                            const int lane, EX extra)
{
    int res = -1;
    const KT* __restrict__ sx = Sf + (size_t)xq * spitch;
    const KT* __restrict__ s1 = Sf + (size_t)v1q * spitch;
    const KT* __restrict__ rx = Kf + xs + (31 - lane); // vertex 32 blk + 31 - lane of the two rows: r[32 blk]
    const KT* __restrict__ r1 = Kf + v1s + (31 - lane);
    const int nl = n - (31 - lane);                      // 32 blk < nl: the vertex exists
    for (int bt = base >> 5; bt >= 0 && res < 0; bt -= 32) {
        const int b = bt - lane;
        u32 s = 0u;
        if (b >= 0) s = min((u32)__ldg(sx + b), (u32)__ldg(s1 + b));
        u32 cand = __ballot_sync(RIPS_FULL_MASK, s >= ks);
        while (cand && res < 0) {
            int b32[4]; // 32 x block, or past the end of the rows for an absent one
            u32 mm[4], bb[4];
#pragma unroll
            for (int g = 0; g < 4; ++g) {
                b32[g] = 0x7fffffe0;
                if (cand) {
                    b32[g] = (bt - (__ffs(cand) - 1)) << 5;
                    cand &= cand - 1;
                }
            }
#pragma unroll
            for (int g = 0; g < 4; ++g) {
                mm[g] = 0u;
                if (b32[g] < nl) mm[g] = min(min((u32)rx[b32[g]], (u32)r1[b32[g]]), extra(b32[g] + 31 - lane));
            }
#pragma unroll
            for (int g = 0; g < 4; ++g) bb[g] = __ballot_sync(RIPS_FULL_MASK, mm[g] >= ks);
            if (bb[0] | bb[1] | bb[2] | bb[3]) { // the first block of the round that holds one, its highest vertex
                const int g0 = bb[0] ? 0 : bb[1] ? 1 : bb[2] ? 2 : 3;
                const u32 bg = bb[0] ? bb[0] : bb[1] ? bb[1] : bb[2] ? bb[2] : bb[3];
                const int bg32 = g0 == 0 ? b32[0] : g0 == 1 ? b32[1] : g0 == 2 ? b32[2] : b32[3];
                res = bg32 + 31 - (__ffs(bg) - 1);
            }
        }
    }
    return res;
}

// KS: the key matrix is staged in shared memory.  A template parameter, not a run-time flag, so that the
// compiler addresses Kf with 32-bit shared-memory addresses (LDS) instead of generic 64-bit ones: the
// kernel is bound by instruction issue, and address arithmetic is a large part of its instructions.
template <int M, typename KT, bool KS>
__global__ void __launch_bounds__(S1_THREADS) enumerate_apparent_kernel(const Stage1Params p)
{
    extern __shared__ __align__(16) unsigned char smem1[];
    __shared__ u32 s_hist_cols[S1_MAX_FUSED][256];
    __shared__ u32 s_hist_pairs[S1_MAX_FUSED_P][256];
    __shared__ u32 s_uwin[S1_WARPS][32];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = p.n, pitch = p.pitch, vbits = p.vbits, lowbits = p.lowbits;
    const u32 lt_mask = (1u << lane) - 1u;
    const u32 thr1 = p.thr_key + 1u; // keys in Kf are shifted by one
    const bool compact = p.compact != 0, count_only = p.count_only != 0;
    const u64 csentinel = (u64)p.sentinel_key << lowbits;
    const u64 psentinel = (u64)(u32)n << p.tbits;

    // ---- shared memory carve-up: [Kf] [staging (compact mode)]
    size_t off_b = 0;
    const KT* __restrict__ Kf;
    if (KS) {
        const int cnt16 = (int)(((size_t)n * pitch * sizeof(KT) + 15) / 16); // the buffer is padded to 16 bytes
        uint4* dst = reinterpret_cast<uint4*>(smem1);
        const uint4* src = reinterpret_cast<const uint4*>(p.Kf);
        for (int i = tid; i < cnt16; i += S1_THREADS) dst[i] = __ldg(src + i);
        Kf = reinterpret_cast<const KT*>(smem1);
        off_b = (size_t)cnt16 * 16;
    } else {
        Kf = reinterpret_cast<const KT*>(p.Kf);
    }
    u64* stage_cols = nullptr;
    u64* stage_pairs = nullptr;
    if (compact && !count_only) {
        stage_cols = reinterpret_cast<u64*>(smem1 + off_b) + (size_t)warp * (2 * p.stage_cap);
        stage_pairs = stage_cols + p.stage_cap;
    }
    BlockHists H;
    H.cols = s_hist_cols;
    H.pairs = s_hist_pairs;
    H.ncols = (!count_only && p.fh_cols.hist) ? p.fh_cols.npasses : 0;
    H.npairs = (!count_only && p.fh_pairs.hist) ? p.fh_pairs.npasses : 0;
#pragma unroll
    for (int r = 0; r < S1_MAX_FUSED; ++r) {
        H.csh[r] = r < H.ncols ? p.fh_cols.shift[r] : 0;
        H.cmk[r] = r < H.ncols ? (1u << p.fh_cols.bits[r]) - 1u : 0u;
    }
#pragma unroll
    for (int r = 0; r < S1_MAX_FUSED_P; ++r) {
        H.psh[r] = r < H.npairs ? p.fh_pairs.shift[r] : 0;
        H.pmk[r] = r < H.npairs ? (1u << p.fh_pairs.bits[r]) - 1u : 0u;
    }
    for (int i = tid; i < S1_MAX_FUSED * 256; i += S1_THREADS) (&s_hist_cols[0][0])[i] = 0;
    for (int i = tid; i < S1_MAX_FUSED_P * 256; i += S1_THREADS) (&s_hist_pairs[0][0])[i] = 0;
    __syncthreads();

    u32 n_clr = 0, n_reg = 0;
    u64 n_over = 0;
    u64 n_kept = 0;
    const int kwin = n < 32 ? n : 32;
    const int kfast = p.fast_visits < kwin ? p.fast_visits : kwin; // vertices n-1 .. n-kfast: per-lane scan of the row's window
    u32* const uw = s_uwin[warp];

    // Compact mode: the unit of the look-back chain is a ROUND of the block (one chunk per warp), so that the
    // chain has S1_WARPS times fewer links than chunks (with most candidates dropped the chunks are cheap, and a
    // chain of one link per chunk was what bounded the kernel).  Slot mode needs no chain: warps take chunks alone.
    const bool block_rounds = compact && !count_only;
    __shared__ u32 s_round;
    __shared__ u32 s_wc[S1_WARPS];
    __shared__ u64 s_excl;
    for (;;) {
        u32 chunk = 0, round = 0;
        bool active = true;
        if (block_rounds) {
            __syncthreads(); // the previous round's shared words are no longer read
            if (tid == 0) s_round = atomicAdd(p.ticket, 1u);
            __syncthreads();
            round = s_round;
            if ((i64)round * S1_WARPS >= p.tiles) break;
            chunk = round * S1_WARPS + warp;
            active = (i64)chunk < p.tiles;
        } else {
            if (lane == 0) chunk = atomicAdd(p.ticket, 1u);
            chunk = __shfl_sync(RIPS_FULL_MASK, chunk, 0);
            if ((i64)chunk >= p.tiles) break;
        }

        u64 idx = active ? (u64)chunk * (u64)p.chunk : 0;
        int rem = !active ? 0 : (p.total - idx) < (u64)p.chunk ? (int)(p.total - idx) : p.chunk;
        int v[M];
        decode_simplex_fast<M>(p.bt, idx, n, v); // warp-uniform
        u32 wcount = 0;
        // offset of the chunk's first candidate inside its slab: a slab fixes the vertices v[M-1] > ... > v[2]
        // (all of them for M = 2: one slab) and holds the C(v[2], 2) pairs v[1] > v[0] in index order
        i64 e0 = (i64)v[1] * (v[1] - 1) / 2 + v[0];

        while (rem > 0) {
            // ---- per slab (warp-uniform): keys among v[2..M-1], upper part of the record, and the window
            // uw[l] = min_j>=2 key1(v_j, n-1-l), the part of the cofacet test of vertex n-1-l the whole slab shares
            u32 up2 = 0xffffffffu;
#pragma unroll
            for (int a = 3; a < M; ++a)
#pragma unroll
                for (int b = 2; b < a; ++b) up2 = min(up2, (u32)Kf[v[a] * pitch + v[b]]);
            u64 slab_low = 0;
#pragma unroll
            for (int j = M - 1; j >= 2; --j) slab_low = (slab_low << vbits) | (u64)(u32)v[j];
            slab_low <<= 2 * vbits;
            const i64 slab_len = (M > 2) ? (i64)v[M > 2 ? 2 : 1] * (v[M > 2 ? 2 : 1] - 1) / 2 : (i64)n * (n - 1) / 2;
            const int seg = (slab_len - e0) < (i64)rem ? (int)(slab_len - e0) : rem;
            if (!count_only) {
                __syncwarp();
                u32 u = 0;
                if (lane < kwin) {
                    u = 0xffffffffu;
#pragma unroll
                    for (int j = 2; j < M; ++j) u = min(u, (u32)Kf[v[j] * pitch + (n - 1 - lane)]);
                }
                uw[lane] = u;
                __syncwarp();
            }
            // one warp step: this lane's candidate (v[M-1..2], v1, x) with index ci
            auto step = [&](const int v1, const int x, const bool valid, const u64 ci) {
                bool keep = false;
                u32 key1 = up2;
                const KT* row1 = Kf + v1 * pitch;
                if (valid) {
#pragma unroll
                    for (int j = 2; j < M; ++j) key1 = min(key1, (u32)Kf[v[j] * pitch + v1]);
                    key1 = min(key1, (u32)row1[x]);
#pragma unroll
                    for (int j = 2; j < M; ++j) key1 = min(key1, (u32)Kf[v[j] * pitch + x]);
                    if (key1 >= thr1) {
                        bool clr;
                        if (p.clear.bitmap) clr = (__ldg(p.clear.bitmap + (ci >> 5)) >> (ci & 31)) & 1u;
                        else
                            clr = in_sorted(p.clear.layer1, p.clear.n1, p.clear.shift1, ci) ||
                                  in_sorted(p.clear.layer2, p.clear.n2, 0, ci);
                        keep = !clr;
                        n_clr += clr;
                    } else
                        ++n_over;
                }
                const u32 bal = __ballot_sync(RIPS_FULL_MASK, keep);
                const u32 slot = wcount + __popc(bal & lt_mask);
                wcount += __popc(bal);
                if (count_only || (compact && bal == 0)) return; // compact mode writes nothing for an all-dropped warp step

                // ---- a7, fast path: cofacet vertices n-1, n-2, ... against the row's window
                const u64 rec = keep ? (((u64)(key1 - 1u) << lowbits) | slab_low | ((u64)(u32)v1 << vbits) | (u64)(u32)x) : csentinel;
                int fv = -1;
                const KT* rowx = Kf + x * pitch;
                if (keep) { // each lane on its own, up to kfast vertices (the common case ends after one or two)
                    for (int k = 0; k < kfast; ++k) {
                        if (min(min(uw[k], (u32)row1[n - 1 - k]), (u32)rowx[n - 1 - k]) >= key1) { fv = n - 1 - k; break; }
                    }
                }
                // the lanes still scanning are finished by the whole warp, one after the other: 32 cofacet
                // vertices per step (lane l takes vertex base - l, so all reads of Kf are consecutive)
                u32 open = __ballot_sync(RIPS_FULL_MASK, keep && fv < 0);
                while (open) {
                    const int src = __ffs(open) - 1;
                    open &= open - 1;
                    const int xs = __shfl_sync(RIPS_FULL_MASK, x, src);
                    const int v1s = __shfl_sync(RIPS_FULL_MASK, v1, src);
                    const u32 ks = __shfl_sync(RIPS_FULL_MASK, key1, src);
                    int res = -1;
                    for (int base = n - 1 - kfast; base >= 0; base -= 32) {
                        const int vv = base - lane;
                        bool ok = false;
                        if (vv >= 0) {
                            u32 m = min((u32)Kf[xs * pitch + vv], (u32)Kf[v1s * pitch + vv]);
#pragma unroll
                            for (int j = 2; j < M; ++j) m = min(m, (u32)Kf[v[j] * pitch + vv]);
                            ok = m >= ks;
                        }
                        const u32 b = __ballot_sync(RIPS_FULL_MASK, ok);
                        if (b) { res = base - (__ffs(b) - 1); break; }
                        if (p.Sf) { // the rest guided by the block maxima of the two rows
                            res = summary_scan<KT>(Kf, reinterpret_cast<const KT*>(p.Sf), p.spitch, n, xs * pitch, v1s * pitch, xs, v1s, ks,
                                                   base - 32, lane, [&](const int w) {
                                                       u32 m2 = 0xffffffffu;
#pragma unroll
                                                       for (int j = 2; j < M; ++j) m2 = min(m2, (u32)Kf[v[j] * pitch + w]);
                                                       return m2;
                                                   });
                            break;
                        }
                    }
                    if (lane == src) fv = res;
                }
                const bool found = keep && fv >= 0;
                const int vtop = (M > 2) ? v[M - 1] : v1;
                const bool regular = found && fv > vtop;
                u64 prec = psentinel;
                if (regular) {
                    prec = ((u64)(u32)fv << p.tbits) | (ci + p.bt(fv, M + 1));
                    ++n_reg;
                }
                // ---- cofacet vertex below the top of s: facet test.  The top vertex is the row's, so
                // these lanes come in whole rows (every column of a row whose top vertex is n-1, ...)
                bool is_irr = false, is_non = keep && !found;
                u64 irr_rec = 0;
                if (found && !regular) {
                    int sv[M];
                    sv[0] = x;
                    sv[1] = v1;
#pragma unroll
                    for (int j = 2; j < M; ++j) sv[j] = v[j];
                    int fseg = 0;
#pragma unroll
                    for (int j = 0; j < M; ++j) fseg += (sv[j] < fv) ? 1 : 0;
                    if (s_is_youngest_facet<M, KT>(Kf, pitch, sv, key1, fv, fseg)) {
                        irr_rec = (cofacet_index<M>(p.bt, sv, fv, fseg) << RIPS_PAIR_POS_BITS) | (u64)fseg;
                        is_irr = true;
                    } else
                        is_non = true;
                }
                const u32 b_irr = __ballot_sync(RIPS_FULL_MASK, is_irr);
                if (b_irr) {
                    u64 base = 0;
                    if (lane == __ffs(b_irr) - 1)
                        base = atomicAdd((unsigned long long*)(p.counters + S1C_IRREGULAR), (unsigned long long)__popc(b_irr));
                    base = __shfl_sync(RIPS_FULL_MASK, base, __ffs(b_irr) - 1) + __popc(b_irr & lt_mask);
                    if (is_irr && base < p.irr_cap) p.irr_out[base] = irr_rec;
                }
                const u32 b_non = __ballot_sync(RIPS_FULL_MASK, is_non);
                if (b_non) {
                    u64 base = 0;
                    if (lane == __ffs(b_non) - 1)
                        base = atomicAdd((unsigned long long*)(p.counters + S1C_NONAPP), (unsigned long long)__popc(b_non));
                    base = __shfl_sync(RIPS_FULL_MASK, base, __ffs(b_non) - 1) + __popc(b_non & lt_mask);
                    if (is_non && base < p.non_cap) p.non_out[base] = rec;
                }
                // ---- stores
                if (compact) {
                    if (keep) {
                        if (slot < (u32)p.stage_cap) {
                            stage_cols[slot] = rec;
                            stage_pairs[slot] = prec;
                        } else // more survivors than provisioned for this chunk: the host repeats the launch with smaller chunks
                            atomicOr((unsigned long long*)(p.counters + S1C_STAGE_OVERFLOW), 1ull);
                    }
                } else if (valid) {
                    __stcs(p.cols_out + ci, rec);
                    __stcs(p.pairs_out + ci, prec);
                }
                // ---- fused histograms over every slot written
                const bool wrote_col = compact ? keep : valid;
                if (wrote_col) {
#pragma unroll
                    for (int r = 0; r < S1_MAX_FUSED; ++r)
                        if (r < H.ncols) atomicAdd(&H.cols[r][(u32)(rec >> H.csh[r]) & H.cmk[r]], 1u);
                }
                const bool wrote_pair = wrote_col;
#pragma unroll
                for (int r = 0; r < S1_MAX_FUSED_P; ++r) {
                    if (r < H.npairs) { // few distinct digits in a warp: aggregate
                        const u32 dg = wrote_pair ? ((u32)(prec >> H.psh[r]) & H.pmk[r]) : 0xffffffffu;
                        const u32 peers = __match_any_sync(RIPS_FULL_MASK, dg);
                        if (wrote_pair && lane == __ffs(peers) - 1) atomicAdd(&H.pairs[r][dg], (u32)__popc(peers));
                    }
                }
            };

            if (!compact) {
                // ---- slot mode: the lanes walk the segment's pairs (v1, x) in index order, 32 at a time
                int lv1, lx;
                {
                    const i64 e = e0 + lane;
                    lv1 = (int)((1.0f + sqrtf(1.0f + 8.0f * (float)e)) * 0.5f);
                    if (lv1 < 1) lv1 = 1;
                    while ((i64)lv1 * (lv1 - 1) / 2 > e) --lv1;
                    while ((i64)(lv1 + 1) * lv1 / 2 <= e) ++lv1;
                    lx = (int)(e - (i64)lv1 * (lv1 - 1) / 2);
                }
                for (int off = lane; off - lane < seg; off += 32, lane_advance(lv1, lx))
                    step(lv1, lx, off < seg, idx + (u64)off);
            } else {
                // ---- compact mode (a threshold drops most candidates): row by row, v1 warp-uniform, so that a row
                // whose upper edges already exceed the threshold is skipped as a whole -- the pruning of the index
                // space that makes a thresholded (sparse) complex cheap: under a threshold that keeps a share q of
                // the edges only about q of the rows are walked at all
                int r1;
                {
                    r1 = (int)((1.0f + sqrtf(1.0f + 8.0f * (float)e0)) * 0.5f);
                    if (r1 < 1) r1 = 1;
                    while ((i64)r1 * (r1 - 1) / 2 > e0) --r1;
                    while ((i64)(r1 + 1) * r1 / 2 <= e0) ++r1;
                }
                int x0 = (int)(e0 - (i64)r1 * (r1 - 1) / 2);
                int left = seg;
                u64 ci0 = idx;
                while (left > 0) {
                    const int row_n = min(r1 - x0, left);
                    u32 rowkey = up2;
#pragma unroll
                    for (int j = 2; j < M; ++j) rowkey = min(rowkey, (u32)Kf[v[j] * pitch + r1]);
                    if (rowkey < thr1) {
                        if (lane == 0) n_over += (u64)row_n; // every candidate of the row is above the threshold
                    } else {
                        for (int off = lane; off - lane < row_n; off += 32)
                            step(r1, x0 + off, off < row_n, ci0 + (u64)off);
                    }
                    ci0 += (u64)row_n;
                    left -= row_n;
                    x0 = 0;
                    ++r1;
                }
            }
            idx += (u64)seg;
            rem -= seg;
            e0 += seg;
            if (e0 >= slab_len) { // next slab (colex successor of (v[M-1..2]))
                e0 = 0;
                if (M > 2) {
#pragma unroll
                    for (int j = 2; j < M; ++j) {
                        v[j] += 1;
                        if (j + 1 < M && v[j] == v[j + 1 < M ? j + 1 : j]) v[j] = j;
                        else break;
                    }
                }
            }
        }

        n_kept += wcount;
        if (count_only) continue;
        if (compact) {
            // ---- ordered compaction: look-back over the block's rounds, then every warp writes its staged records
            if (lane == 0) s_wc[warp] = wcount;
            __syncthreads();
            if (warp == 0) {
                u32 c = lane < S1_WARPS ? s_wc[lane] : 0u;
                const u64 total_round = (u64)__reduce_add_sync(RIPS_FULL_MASK, c);
                const u64 e = lookback_exclusive(p.status, (i64)round, total_round);
                if (lane == 0) s_excl = e;
            }
            __syncthreads();
            u64 excl = s_excl;
            for (int w = 0; w < warp; ++w) excl += s_wc[w];
            for (u32 i = lane; i < wcount && i < (u32)p.stage_cap; i += 32) {
                __stcs(p.cols_out + excl + i, stage_cols[i]);
                __stcs(p.pairs_out + excl + i, stage_pairs[i]);
            }
            __syncwarp();
        }
    }

    // ---- counters and the fused histograms: once per block
    n_over = warp_sum_u64(n_over);
    n_clr = warp_sum_u32(n_clr);
    n_reg = warp_sum_u32(n_reg);
    if (lane == 0) {
        if (n_kept) atomicAdd((unsigned long long*)&p.counters[S1C_KEPT], (unsigned long long)n_kept);
        if (n_over) atomicAdd((unsigned long long*)&p.counters[S1C_OVER], (unsigned long long)n_over);
        if (n_clr) atomicAdd((unsigned long long*)&p.counters[S1C_CLEARED], (unsigned long long)n_clr);
        if (n_reg) atomicAdd((unsigned long long*)&p.counters[S1C_REGULAR], (unsigned long long)n_reg);
    }
    __syncthreads();
    for (int i = tid; i < H.ncols * 256; i += S1_THREADS) {
        u32 c = (&s_hist_cols[0][0])[i];
        if (c) atomicAdd((unsigned long long*)&p.fh_cols.hist[i], (unsigned long long)c);
    }
    for (int i = tid; i < H.npairs * 256; i += S1_THREADS) {
        u32 c = (&s_hist_pairs[0][0])[i];
        if (c) atomicAdd((unsigned long long*)&p.fh_pairs.hist[i], (unsigned long long)c);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// The same steps for SLOT mode only (every candidate keeps its slot: no threshold, or one that keeps most), written
// for the instruction budget: the kernel is bound by instruction issue, so what is warp- or slab-uniform is taken out
// of the per-candidate path.
//   * per slab, U2[w] = min_{j>=2} key1(v_j, w) for every vertex w, in a per-warp row of shared memory: key(s) is then
//     min(up2, U2[v1], U2[x], Kf[v1][x]) -- three gathers instead of 2(M-2)+1 -- and the same row is the shared part of
//     every cofacet test of the slab;
//   * row offsets v1*pitch and x*pitch are carried along by lane_advance (additions only);
//   * the cofacet scan tests the first four vertices n-1..n-4 of every lane at once, branch-free (the mean number of
//     visits is about two: one lane-serial loop made the whole warp wait for its slowest lane).  The lanes still open
//     after that (one in ten) do not hold the step up: they put (cidx, key, v1, x) into a queue of their warp in shared
//     memory, and the warp finishes 32 of them at a time (drain: twelve more vertices for every lane at once, the rest by
//     the warp-cooperative scan, then the pair slot, the pair histogram and the small lists).  With block maxima (SUM:
//     thousands of points, where the scans are the kernel) they are finished inside the step as in the general kernel;
//   * digits of the fused histograms are taken from the 32-bit key / cofacet vertex, not from the 64-bit records;
//   * C(v, M+1), the offset of a regular pair's row, comes from a copy of that binomial column in shared memory;
//   * nothing is counted per warp step: the number of columns is total - over - cleared.
// Same records, same lists, same counters as enumerate_apparent_kernel (the tests compare both with the oracle).
// ---------------------------------------------------------------------------------------------------------------
template <int M, typename KT, bool KS, bool SUM>
__global__ void __launch_bounds__(S1_THREADS, SUM ? 2 : 0) enumerate_slot_kernel(const Stage1Params p)
{
    extern __shared__ __align__(16) unsigned char smem1[];
    __shared__ u32 s_hist_cols[S1_MAX_FUSED][256];
    __shared__ u32 s_hist_pairs[S1_MAX_FUSED_P][256];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = p.n, pitch = p.pitch;

    // ---- shared memory: [Kf (KS)] [C(., M+1) : n u64] [U2 : S1_WARPS rows of n KT (M > 2)]
    size_t off_b = 0;
    const KT* __restrict__ Kf;
    if (KS) {
        const int cnt16 = (int)(((size_t)n * pitch * sizeof(KT) + 15) / 16);
        uint4* dst = reinterpret_cast<uint4*>(smem1);
        const uint4* src = reinterpret_cast<const uint4*>(p.Kf);
        for (int i = tid; i < cnt16; i += S1_THREADS) dst[i] = __ldg(src + i);
        Kf = reinterpret_cast<const KT*>(smem1);
        off_b = (size_t)cnt16 * 16;
    } else {
        Kf = reinterpret_cast<const KT*>(p.Kf);
    }
    u64* const sprec = reinterpret_cast<u64*>(smem1 + off_b); // record of a regular pair with cofacet vertex v, minus cidx(s)
    if (!SUM) { // (SUM: thousands of points, where this table would cost the second resident block; C(v, M+1) is read from HBM's copy)
        for (int i = tid; i < n; i += S1_THREADS) sprec[i] = ((u64)(u32)i << p.tbits) + p.bt(i, M + 1);
        off_b += (size_t)n * 8;
    }
    KT* const u2 = reinterpret_cast<KT*>(smem1 + off_b) + (size_t)warp * ((n + 7) & ~7);
    // (!SUM) the warp's queue of candidates whose cofacet scan is still open after four vertices: S1_QCAP entries of
    // (cidx, key, v1, v0), behind the U2 rows
    const size_t q_off = (off_b + ((M > 2) ? (size_t)S1_WARPS * ((n + 7) & ~7) * sizeof(KT) : 0) + 15) & ~(size_t)15;
    uint4* const q = reinterpret_cast<uint4*>(smem1 + q_off) + (size_t)warp * S1_QCAP;
    int qcnt = 0;
    const u32 lt_mask_q = (1u << lane) - 1u;
    for (int i = tid; i < S1_MAX_FUSED * 256; i += S1_THREADS) (&s_hist_cols[0][0])[i] = 0;
    for (int i = tid; i < S1_MAX_FUSED_P * 256; i += S1_THREADS) (&s_hist_pairs[0][0])[i] = 0;
    __syncthreads();

    // digits of the two sorts: byte r of the 32-bit key / cofacet vertex (sort_make_plan: 8-bit digits from the
    // bottom of the field)
    const int ncd = p.fh_cols.hist ? p.fh_cols.npasses : 0, npd = p.fh_pairs.hist ? p.fh_pairs.npasses : 0;
    const u32 thr1 = p.thr_key + 1u;
    const u32 sentinel_key = p.sentinel_key;
    const int vbits = p.vbits, lowbits = p.lowbits;
    const u32 vmul = 1u << vbits;
    const u64 psentinel = (u64)(u32)n << p.tbits;
    u32 n_clr = 0, n_reg = 0;
    u64 n_over = 0;

    for (;;) {
        u32 chunk = 0;
        if (lane == 0) chunk = atomicAdd(p.ticket, 1u);
        chunk = __shfl_sync(RIPS_FULL_MASK, chunk, 0);
        if ((i64)chunk >= p.tiles) break;
        u64 idx = (u64)chunk * (u64)p.chunk;
        int rem = (p.total - idx) < (u64)p.chunk ? (int)(p.total - idx) : p.chunk;
        int v[M];
        decode_simplex_fast<M>(p.bt, idx, n, v); // warp-uniform
        i64 e0 = (i64)v[1] * (v[1] - 1) / 2 + v[0];

        while (rem > 0) {
            // ---- per slab (warp-uniform)
            u32 up2 = 0xffffffffu;
#pragma unroll
            for (int a = 3; a < M; ++a)
#pragma unroll
                for (int b = 2; b < a; ++b) up2 = min(up2, (u32)Kf[v[a] * pitch + v[b]]);
            u64 slab_low = 0;
#pragma unroll
            for (int j = M - 1; j >= 2; --j) slab_low = (slab_low << vbits) | (u64)(u32)v[j];
            slab_low <<= 2 * vbits;
            const i64 slab_len = (M > 2) ? (i64)v[M > 2 ? 2 : 1] * (v[M > 2 ? 2 : 1] - 1) / 2 : (i64)n * (n - 1) / 2;
            const int seg = (slab_len - e0) < (i64)rem ? (int)(slab_len - e0) : rem;
            u32 ur0 = 0xffffffffu, ur1 = 0xffffffffu, ur2 = 0xffffffffu, ur3 = 0xffffffffu;
            if (M > 2) {
                __syncwarp();
                for (int w = lane; w < n; w += 32) {
                    u32 u = 0xffffffffu;
#pragma unroll
                    for (int j = 2; j < M; ++j) u = min(u, (u32)Kf[v[j] * pitch + w]);
                    u2[w] = (KT)u; // a diagonal zero stays zero: vertices of the slab fail every test by themselves
                }
                __syncwarp();
                ur0 = n >= 1 ? (u32)u2[n - 1] : 0u;
                ur1 = n >= 2 ? (u32)u2[n - 2] : 0u;
                ur2 = n >= 3 ? (u32)u2[n - 3] : 0u;
                ur3 = n >= 4 ? (u32)u2[n - 4] : 0u;
            } else {
                if (n < 4) ur3 = 0u;
                if (n < 3) ur2 = 0u;
                if (n < 2) ur1 = 0u;
            }
            const int vtop_slab = (M > 2) ? v[M - 1] : 0;

            // ---- what follows the cofacet scan of a candidate: the pair slot, the pair histogram, and for a cofacet vertex
            // below the top of s (whole rows of lanes: the columns holding the top vertices) or no cofacet of equal diameter
            // the facet test and the two small lists.  Called by the whole warp: in the walk for the lanes whose scan
            // ended within four vertices (and the dropped candidates), in drain() for the others.
            auto finish = [&](const bool act, const bool keep_, const u64 ci_, const u32 key1_, const int lv1_, const int lx_, const int fv_) {
                const bool found = fv_ >= 0;
                const int vtop = (M > 2) ? vtop_slab : lv1_;
                const bool regular = act && found && fv_ > vtop;
                const u32 fvv = regular ? (u32)fv_ : (u32)n;
                u64 prec = psentinel;
                if (regular) {
                    prec = SUM ? ci_ + ((u64)(u32)fv_ << p.tbits) + p.bt(fv_, M + 1) : ci_ + sprec[fv_];
                    ++n_reg;
                }
                if (__any_sync(RIPS_FULL_MASK, act && keep_ && !regular)) {
                    bool is_irr = false, is_non = act && keep_ && !found;
                    u64 irr_rec = 0;
                    if (act && keep_ && found && !regular) {
                        int sv[M];
                        sv[0] = lx_;
                        sv[1] = lv1_;
#pragma unroll
                        for (int j = 2; j < M; ++j) sv[j] = v[j];
                        int fseg = 0;
#pragma unroll
                        for (int j = 0; j < M; ++j) fseg += (sv[j] < fv_) ? 1 : 0;
                        if (s_is_youngest_facet<M, KT>(Kf, pitch, sv, key1_, fv_, fseg)) {
                            irr_rec = (cofacet_index<M>(p.bt, sv, fv_, fseg) << RIPS_PAIR_POS_BITS) | (u64)fseg;
                            is_irr = true;
                        } else
                            is_non = true;
                    }
                    const u32 lt_mask = (1u << lane) - 1u;
                    const u32 b_irr = __ballot_sync(RIPS_FULL_MASK, is_irr);
                    if (b_irr) {
                        u64 base = 0;
                        if (lane == __ffs(b_irr) - 1)
                            base = atomicAdd((unsigned long long*)(p.counters + S1C_IRREGULAR), (unsigned long long)__popc(b_irr));
                        base = __shfl_sync(RIPS_FULL_MASK, base, __ffs(b_irr) - 1) + __popc(b_irr & lt_mask);
                        if (is_irr && base < p.irr_cap) p.irr_out[base] = irr_rec;
                    }
                    const u32 b_non = __ballot_sync(RIPS_FULL_MASK, is_non);
                    if (b_non) {
                        u64 base = 0;
                        if (lane == __ffs(b_non) - 1)
                            base = atomicAdd((unsigned long long*)(p.counters + S1C_NONAPP), (unsigned long long)__popc(b_non));
                        base = __shfl_sync(RIPS_FULL_MASK, base, __ffs(b_non) - 1) + __popc(b_non & lt_mask);
                        if (is_non && base < p.non_cap)
                            p.non_out[base] = ((u64)(key1_ - 1u) << lowbits) | slab_low | (u64)((u32)lv1_ * vmul + (u32)lx_);
                    }
                }
                if (act) __stcs(p.pairs_out + ci_, prec);
#pragma unroll
                for (int r = 0; r < S1_MAX_FUSED_P; ++r) {
                    if (r < npd) { // few distinct digits in a warp: aggregate
                        const u32 dg = act ? ((fvv >> (8 * r)) & 0xffu) : 0xffffffffu;
                        const u32 peers = __match_any_sync(RIPS_FULL_MASK, dg);
                        if (act && lane == __ffs(peers) - 1) atomicAdd(&s_hist_pairs[r][dg], (u32)__popc(peers));
                    }
                }
            };
            // ---- (!SUM) the last m entries of the warp's queue, one per lane: S1_QVISITS more cofacet vertices for every lane
            // at once, branch-free (three in four end there), the rest by the whole warp, 32 vertices per step, then finish()
            auto drain = [&](const int m) {
                __syncwarp();
                const bool act = lane < m;
                const uint4 e = q[qcnt - m + (act ? lane : 0)];
                qcnt -= m;
                __syncwarp();
                const u64 ci_ = ((u64)e.y << 32) | (u64)e.x;
                const u32 key1_ = e.z;
                const int lv1_ = (int)(e.w >> 16), lx_ = (int)(e.w & 0xffffu);
                const int r1o_ = lv1_ * pitch, xo_ = lx_ * pitch;
                const int kend = n < 4 + S1_QVISITS ? n : 4 + S1_QVISITS;
                int fv_ = -1;
#pragma unroll
                for (int k = 4 + S1_QVISITS - 1; k >= 4; --k) {
                    if (k < kend) {
                        const u32 uu = (M > 2) ? (u32)u2[n - 1 - k] : 0xffffffffu;
                        if (min(min(uu, (u32)Kf[r1o_ + n - 1 - k]), (u32)Kf[xo_ + n - 1 - k]) >= key1_) fv_ = n - 1 - k;
                    }
                }
                u32 open = __ballot_sync(RIPS_FULL_MASK, act && fv_ < 0);
                while (open) {
                    const int src = __ffs(open) - 1;
                    open &= open - 1;
                    const int xs = __shfl_sync(RIPS_FULL_MASK, xo_, src);
                    const int v1s = __shfl_sync(RIPS_FULL_MASK, r1o_, src);
                    const u32 ks = __shfl_sync(RIPS_FULL_MASK, key1_, src);
                    int res = -1;
                    for (int base = n - 1 - kend; base >= 0 && res < 0; base -= 32) {
                        const int vv = base - lane;
                        u32 m0 = 0u;
                        if (vv >= 0) {
                            m0 = min((u32)Kf[xs + vv], (u32)Kf[v1s + vv]);
                            if (M > 2) m0 = min(m0, (u32)u2[vv]);
                        }
                        const u32 bb = __ballot_sync(RIPS_FULL_MASK, m0 >= ks); // (ks >= 1: an absent vertex never passes)
                        if (bb) res = base - (__ffs(bb) - 1);
                    }
                    if (lane == src) fv_ = res;
                }
                finish(act, true, ci_, key1_, lv1_, lx_, fv_);
            };

            // ---- the lanes walk the segment's pairs (v1, x) in index order, 32 at a time
            int lv1, lx;
            {
                const i64 e = e0 + lane;
                lv1 = (int)((1.0f + sqrtf(1.0f + 8.0f * (float)e)) * 0.5f);
                if (lv1 < 1) lv1 = 1;
                while ((i64)lv1 * (lv1 - 1) / 2 > e) --lv1;
                while ((i64)(lv1 + 1) * lv1 / 2 <= e) ++lv1;
                lx = (int)(e - (i64)lv1 * (lv1 - 1) / 2);
            }
            int r1o = lv1 * pitch, xo = lx * pitch; // row offsets, carried along
            const int pitch32 = 32 * pitch;
            for (int off = lane; off - lane < seg; off += 32) {
                const bool valid = off < seg;
                const u64 ci = idx + (u64)off;
                // ---- a3/a4: key of the simplex, threshold, clearing
                bool keep = false;
                u32 key1 = up2;
                if (valid) {
                    if (M > 2) key1 = min(min(key1, (u32)u2[lv1]), (u32)u2[lx]);
                    key1 = min(key1, (u32)Kf[r1o + lx]);
                    if (key1 >= thr1) {
                        bool clr;
                        if (p.clear.bitmap) clr = (__ldg(p.clear.bitmap + (ci >> 5)) >> ((u32)ci & 31u)) & 1u;
                        else
                            clr = in_sorted(p.clear.layer1, p.clear.n1, p.clear.shift1, ci) ||
                                  in_sorted(p.clear.layer2, p.clear.n2, 0, ci);
                        keep = !clr;
                        n_clr += clr;
                    } else
                        ++n_over;
                }
                // ---- a7: cofacet vertices n-1 .. n-4 for every lane at once
                int fv = -1;
                {
                    const KT* a = Kf + r1o + (n - 1);
                    const KT* b = Kf + xo + (n - 1);
                    const bool h0 = min(min(ur0, (u32)a[0]), (u32)b[0]) >= key1;
                    const bool h1 = n >= 2 && min(min(ur1, (u32)a[n >= 2 ? -1 : 0]), (u32)b[n >= 2 ? -1 : 0]) >= key1;
                    const bool h2 = n >= 3 && min(min(ur2, (u32)a[n >= 3 ? -2 : 0]), (u32)b[n >= 3 ? -2 : 0]) >= key1;
                    const bool h3 = n >= 4 && min(min(ur3, (u32)a[n >= 4 ? -3 : 0]), (u32)b[n >= 4 ? -3 : 0]) >= key1;
                    fv = h0 ? n - 1 : h1 ? n - 2 : h2 ? n - 3 : h3 ? n - 4 : -1;
                    if (!keep) fv = -1;
                }
                bool defer = false;
                if (!SUM && n > 4) {
                    // the lanes still open (one in ten) wait in the warp's queue and are finished 32 at a time (drain)
                    defer = keep && fv < 0;
                    const u32 db = __ballot_sync(RIPS_FULL_MASK, defer);
                    if (db) {
                        if (defer) q[qcnt + __popc(db & lt_mask_q)] = make_uint4((u32)ci, (u32)(ci >> 32), key1, ((u32)lv1 << 16) | (u32)lx);
                        qcnt += __popc(db);
                    }
                } else {
                    u32 open = __ballot_sync(RIPS_FULL_MASK, keep && fv < 0);
                    if (open && n > 4) { // four more for the lanes still open
                        const int kend = n < 8 ? n : 8;
                        if (keep && fv < 0) {
                            for (int k = 4; k < kend; ++k) {
                                const u32 uu = (M > 2) ? (u32)u2[n - 1 - k] : 0xffffffffu;
                                if (min(min(uu, (u32)Kf[r1o + n - 1 - k]), (u32)Kf[xo + n - 1 - k]) >= key1) { fv = n - 1 - k; break; }
                            }
                        }
                        open = __ballot_sync(RIPS_FULL_MASK, keep && fv < 0);
                        // the rest by the whole warp, one open lane after the other, 32 cofacet vertices per step
                        while (open) {
                            const int src = __ffs(open) - 1;
                            open &= open - 1;
                            const int xs = __shfl_sync(RIPS_FULL_MASK, xo, src);
                            const int v1s = __shfl_sync(RIPS_FULL_MASK, r1o, src);
                            const u32 ks = __shfl_sync(RIPS_FULL_MASK, key1, src);
                            // (four groups of 32 vertices per round: the loads of a round are independent, so a column
                            // without any cofacet of equal diameter -- a scan of all n vertices -- waits for HBM n/128
                            // times, not n/32 times; that scan is what binds the kernel when n is in the thousands)
                            int res = -1;
                            int base = n - 1 - kend;
                            if (base >= 0) { // the next 32 vertices first: most open lanes end here
                                const int vv = base - lane;
                                u32 m0 = 0u;
                                if (vv >= 0) {
                                    m0 = min((u32)Kf[xs + vv], (u32)Kf[v1s + vv]);
                                    if (M > 2) m0 = min(m0, (u32)u2[vv]);
                                }
                                const u32 bb = __ballot_sync(RIPS_FULL_MASK, m0 >= ks); // (ks >= 1: an absent vertex never passes)
                                if (bb) res = base - (__ffs(bb) - 1);
                                base -= 32;
                            }
                            if (SUM) { // (the block maxima of the two rows say which blocks of 32 vertices are worth reading)
                                const int xq = __shfl_sync(RIPS_FULL_MASK, lx, src);
                                const int v1q = __shfl_sync(RIPS_FULL_MASK, lv1, src);
                                if (res < 0)
                                    res = summary_scan<KT>(Kf, reinterpret_cast<const KT*>(p.Sf), p.spitch, n, xs, v1s, xq, v1q, ks, base, lane,
                                                           [&](const int w) { return (M > 2) ? (u32)u2[w] : 0xffffffffu; });
                                base = -1;
                            }
                            for (; base >= 0 && res < 0; base -= 128) {
                                u32 mm[4];
#pragma unroll
                                for (int g = 0; g < 4; ++g) {
                                    const int vv = base - 32 * g - lane;
                                    mm[g] = 0u;
                                    if (vv >= 0) {
                                        mm[g] = min((u32)Kf[xs + vv], (u32)Kf[v1s + vv]);
                                        if (M > 2) mm[g] = min(mm[g], (u32)u2[vv]);
                                    }
                                }
#pragma unroll
                                for (int g = 0; g < 4; ++g) {
                                    const u32 bb = __ballot_sync(RIPS_FULL_MASK, mm[g] >= ks);
                                    if (bb && res < 0) res = base - 32 * g - (__ffs(bb) - 1);
                                }
                            }
                            if (lane == src) fv = res;
                        }
                    }
                }
                finish(valid && !defer, keep, ci, key1, lv1, lx, fv);
                const u32 kk = keep ? key1 - 1u : sentinel_key;
                u64 rec = (u64)kk << lowbits;
                if (keep) rec |= slab_low | (u64)((u32)lv1 * vmul + (u32)lx);
                // ---- stores and the fused histograms
                if (valid) {
                    __stcs(p.cols_out + ci, rec);
#pragma unroll
                    for (int r = 0; r < S1_MAX_FUSED; ++r)
                        if (r < ncd) atomicAdd(&s_hist_cols[r][(kk >> (8 * r)) & 0xffu], 1u);
                }
                if (!SUM && qcnt >= 32) drain(32);
                // ---- next pair, 32 positions further in the order e = C(v1, 2) + x
                lx += 32;
                xo += pitch32;
                while (lx >= lv1) { lx -= lv1; xo -= r1o; ++lv1; r1o += pitch; }
            }
            while (qcnt > 0) drain(qcnt < 32 ? qcnt : 32); // (the next slab has its own U2 row)
            idx += (u64)seg;
            rem -= seg;
            e0 += seg;
            if (e0 >= slab_len) { // next slab (colex successor of (v[M-1..2]))
                e0 = 0;
                if (M > 2) {
#pragma unroll
                    for (int j = 2; j < M; ++j) {
                        v[j] += 1;
                        if (j + 1 < M && v[j] == v[j + 1 < M ? j + 1 : j]) v[j] = j;
                        else break;
                    }
                }
            }
        }
    }

    // ---- counters and the fused histograms: once per block
    n_over = warp_sum_u64(n_over);
    n_clr = warp_sum_u32(n_clr);
    n_reg = warp_sum_u32(n_reg);
    if (lane == 0) {
        if (n_over) atomicAdd((unsigned long long*)&p.counters[S1C_OVER], (unsigned long long)n_over);
        if (n_clr) atomicAdd((unsigned long long*)&p.counters[S1C_CLEARED], (unsigned long long)n_clr);
        if (n_reg) atomicAdd((unsigned long long*)&p.counters[S1C_REGULAR], (unsigned long long)n_reg);
    }
    __syncthreads();
    for (int i = tid; i < ncd * 256; i += S1_THREADS) {
        u32 c = (&s_hist_cols[0][0])[i];
        if (c) atomicAdd((unsigned long long*)&p.fh_cols.hist[i], (unsigned long long)c);
    }
    for (int i = tid; i < npd * 256; i += S1_THREADS) {
        u32 c = (&s_hist_pairs[0][0])[i];
        if (c) atomicAdd((unsigned long long*)&p.fh_pairs.hist[i], (unsigned long long)c);
    }
}

// bitmap |= bits of the pivot rows of the three layers of dimension d-1's pair store, in one launch (grid-stride over
// the three segments one after the other).  Regular layer: every slot of the partitioned pair array, the sentinels
// (cofacet vertex = n) skipped; irregular layer: as many records as the fused kernel of dimension d-1 counted (the
// count lives on the device); reduced layer: plain row indices.
__global__ void clear_bitmap_kernel(u32* bitmap, const ClearLayers L)
{
    const i64 stride = (i64)gridDim.x * blockDim.x, t0 = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    for (i64 i = t0; i < L.n_reg; i += stride) {
        const u64 r = __ldg(L.reg + i);
        if ((r >> L.reg_tbits) == L.reg_sentinel) continue;
        const u64 t = r & L.reg_mask;
        atomicOr(bitmap + (t >> 5), 1u << (t & 31));
    }
    i64 n_irr = L.n_irr;
    if (L.n_irr_dev) n_irr = min(n_irr, (i64)__ldg(L.n_irr_dev));
    for (i64 i = t0; i < n_irr; i += stride) {
        const u64 t = __ldg(L.irr + i) >> L.irr_shift;
        atomicOr(bitmap + (t >> 5), 1u << (t & 31));
    }
    for (i64 i = t0; i < L.n_red; i += stride) {
        const u64 t = __ldg(L.red + i);
        atomicOr(bitmap + (t >> 5), 1u << (t & 31));
    }
}

template <typename K>
cudaError_t launch_persistent(K kern, const Stage1Params& p, size_t smem, cudaStream_t st)
{
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
    if (e != cudaSuccess) return e;
    int per_sm = 1;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, S1_THREADS, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) per_sm = 1;
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    i64 g = (p.tiles + S1_WARPS - 1) / S1_WARPS;
    if (g > (i64)sms * per_sm) g = (i64)sms * per_sm;
    kern<<<(unsigned)g, S1_THREADS, smem, st>>>(p);
    return cudaGetLastError();
}

template <int M, typename KT>
cudaError_t launch_stage1_t(const Stage1Params& p, cudaStream_t st)
{
    const size_t kf_bytes = (((size_t)p.n * p.pitch * sizeof(KT)) + 15) & ~(size_t)15;
    const bool kf_fits = kf_bytes <= S1_KF_SMEM_LIMIT;
    if (!p.compact && !p.count_only) {
        // slot mode: the leaner kernel, if its tables fit (C(., M+1) and one row of U2 per warp)
        const size_t u2rows = M > 2 ? (size_t)S1_WARPS * ((p.n + 7) & ~7) * sizeof(KT) : 0;
        const size_t tables = (size_t)p.n * 8 + u2rows + 16 + (size_t)S1_WARPS * S1_QCAP * 16; // C(., M+1), U2 rows, the warps' queues (16-byte aligned)
#ifdef RIPS_STRESS
        const size_t u2_limit = 8 * 1024; // beyond ~130 points the triangles and tetrahedra go to the general kernel (its slot mode with block maxima)
#else
        const size_t u2_limit = 160 * 1024;
#endif
        if (p.Sf && u2rows <= u2_limit) return launch_persistent(enumerate_slot_kernel<M, KT, false, true>, p, u2rows, st);
        if (p.Sf && u2rows > u2_limit && u2_limit < 160 * 1024) return launch_persistent(enumerate_apparent_kernel<M, KT, false>, p, 0, st);
        if (kf_fits && kf_bytes + tables <= 190 * 1024) return launch_persistent(enumerate_slot_kernel<M, KT, true, false>, p, kf_bytes + tables, st);
        if (tables <= 192 * 1024) return launch_persistent(enumerate_slot_kernel<M, KT, false, false>, p, tables, st); // (32 KB of it the queues: the same n as before them)
    }
    const int k_in = (!p.compact && !p.count_only && kf_fits) ? 1 : 0;
    const size_t smem = (k_in ? kf_bytes : 0) +
                        ((p.compact && !p.count_only) ? (size_t)S1_WARPS * 2 * p.stage_cap * 8 : 0);
    if (k_in) return launch_persistent(enumerate_apparent_kernel<M, KT, true>, p, smem, st);
    return launch_persistent(enumerate_apparent_kernel<M, KT, false>, p, smem, st);
}

} // namespace

// Candidates per warp chunk: S1_CHUNK when there is plenty of work, less (a multiple of 32) when the
// index space is small, so that every SM still gets warps to run.  Compact mode stages the survivors of
// a chunk in shared memory (S1_STAGE_CAP records per warp) and wants long chunks, because every round of
// chunks is a link of the look-back chain: the chunk is sized so that the expected survivors
// (est_survival x chunk) fill half the staging; a chunk that overflows is reported and the launch repeated
// with chunk = S1_STAGE_CAP (retry != 0).
#ifdef RIPS_STRESS
int stage1_stage_cap() { return 64; }   // short chunks: many links in compact mode's look-back chain
#else
int stage1_stage_cap() { return 256; }
#endif
int stage1_chunk(u64 total, int compact, double est_survival, int retry, int sms)
{
    u64 c = (total / ((u64)(sms > 0 ? sms : 148) * 64) + 31) / 32 * 32;
    if (c < 32) c = 32;
    if (!compact) return (int)(c > (u64)S1_CHUNK ? (u64)S1_CHUNK : c);
    const u64 cap = (u64)stage1_stage_cap();
    u64 want = cap;
    if (!retry) {
        const double e = est_survival > 1e-3 ? est_survival : 1e-3;
        want = (u64)(0.5 * (double)cap / e) / 32 * 32;
        if (want < cap) want = cap;
        if (want > 4096) want = 4096;
    }
    return (int)(c < want ? c : want);
}

cudaError_t launch_stage1(int M, int kf_u16, const Stage1Params& p, cudaStream_t st)
{
    if (p.tiles == 0) return cudaSuccess;
    if (p.tiles > 0xffffffffLL) return cudaErrorInvalidValue;
#define S1_CASE(MM)                                                                          \
    case MM: return kf_u16 ? launch_stage1_t<MM, unsigned short>(p, st) : launch_stage1_t<MM, u32>(p, st);
    switch (M) {
        S1_CASE(2) S1_CASE(3) S1_CASE(4) S1_CASE(5) S1_CASE(6)
    default: return cudaErrorInvalidValue;
    }
#undef S1_CASE
}

cudaError_t launch_clear_bitmap(u32* bitmap, const ClearLayers& L, int sms, cudaStream_t st)
{
    const i64 n = std::max(L.n_reg, std::max(L.n_irr, L.n_red));
    if (n == 0) return cudaSuccess;
    i64 blocks = (n + 255) / 256;
    if (blocks > (i64)sms * 16) blocks = (i64)sms * 16;
    clear_bitmap_kernel<<<(unsigned)blocks, 256, 0, st>>>(bitmap, L);
    return cudaGetLastError();
}
