/* rips.h -- C ABI of the B200-native Vietoris-Rips hot path (arXiv 2003.07989, "Ripser++").
 *
 * Citations are lines of /root/reference/PAPER.md (the paper's text).  The library computes, per
 * dimension d >= 1, the two stages of Fig. 3(b):
 *
 *   stage 1  filtration construction with clearing, Algorithms 7-8: every
 *            candidate d-simplex by combinatorial index (Eq. 2), its diameter
 *            (Eq. 1), keep iff diameter <= threshold and the simplex is not the
 *            death simplex of a pair of dimension d-1 (clearing lemma), sorted
 *            by diameter descending, index ascending;
 *   stage 2  apparent pairs, Algorithm 3 / Lemma 7: per column s the
 *            oldest cofacet t of equal diameter, and the test that s is the youngest facet of t;
 *            the pairs (t, s) sorted by t with a binary-search lookup, the
 *            non-apparent columns kept in coboundary order.
 *
 * How the work is split between the two entry points: the apparent test of a
 * column does not depend on the order of the columns (Corollary 8), so it runs
 * inside the kernel of rips_stage1 that enumerates the candidates, where the column's vertices and
 * diameter are in registers; rips_stage1 then sorts the columns, and rips_stage2 puts the pairs and the
 * non-apparent columns that kernel produced into their sorted order.  The arrays each call exposes are
 * the paper's, whatever the split.
 *
 * Dimension 0 and the reduction of the non-apparent columns (Algorithm 2,
 * PAPER.md:182-200) complete the barcodes; they are not the hot path and are timed separately
 * (rips_timings).  Every step of stage 1 and stage 2 runs in hand-written CUDA kernels for
 * sm_100a; there is no CPU fallback: on a machine without a usable CUDA device every entry point
 * that needs the device returns RIPS_ECUDA.
 *
 * Conventions
 *   - A d-simplex (v_d > ... > v_0 >= 0) has index cidx = sum_k C(v_k, k+1) (Eq. 2).
 *   - Distance matrix: strict lower triangle, row-major, fp32; element (i > j) at i(i-1)/2 + j,
 *     which is the cidx of the edge (i j).  -0.0f is canonicalised to +0.0f.
 *   - All functions return 0 (RIPS_OK) or a negative error code; nothing throws or aborts.
 *   - Pointers named *_dev are device pointers, *_host host pointers.  Every output array is
 *     owned by the context and stays valid until the next call that recomputes it (rips_compute,
 *     rips_stage1/2 for the same d) or rips_free.  The input matrix is copied by rips_init.
 *   - All work is enqueued on the stream given to rips_init (rips_stage2 also uses internal streams,
 *     joined back into that stream before it returns); calls that return host-visible counts
 *     synchronise that stream.
 *   - Not thread-safe per context; distinct contexts are independent.
 */
#ifndef RIPS_H
#define RIPS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rips_ctx rips_ctx;

enum {
    RIPS_OK = 0,
    RIPS_EINVAL = -1,    /* bad argument: n < 1, dim_max out of [0,4], NaN/negative/non-finite distance,
                            NaN threshold, d out of range, stage called before its inputs exist */
    RIPS_EOVERFLOW = -2, /* n > 46340 (the n x n key matrix is indexed with 32-bit integers), C(n, dim_max+2) >= 2^62,
                            or a packed 64-bit record cannot hold (key bits + vertex bits) / (vertex + row bits) */
    RIPS_ENOMEM = -3,    /* the workspace is too small (rips_last_required_bytes), or an allocation failed */
    RIPS_ECUDA = -4      /* CUDA runtime error; text via rips_last_error */
};

/* Counts per dimension d (Table 5's bookkeeping; Table 1). */
typedef struct {
    int64_t n_candidates;          /* C(n, d+1) */
    int64_t n_removed_by_diameter; /* diameter > threshold */
    int64_t n_cleared;             /* diameter <= threshold and cleared */
    int64_t n_columns;             /* kept = length of the filtration array */
    int64_t n_apparent;            /* apparent pairs (Definition 5) among the columns */
    int64_t n_nonapparent;         /* columns left for the reduction */
    int64_t n_reduced_pivots;      /* pairs found by the reduction */
    int64_t n_essential;           /* columns that reduce to zero */
    int64_t n_additions;           /* column additions performed by the reduction */
    int64_t n_bars;                /* bars of non-zero length reported by rips_barcodes */
    int64_t n_slots;               /* records the two sorts of this dimension move: C(n,d+1) when every candidate
                                      keeps a slot (dropped ones hold a sentinel the sort sinks), n_columns when
                                      the survivors are compacted first (thresholded inputs) */
    int64_t n_regular;             /* apparent pairs whose cofacet vertex lies above every vertex of s (sorted by
                                      one stable partition); the other n_apparent - n_regular are sorted in full */
    int64_t n_reduce_serial;       /* non-apparent columns whose reduction needed another non-apparent column (or did not
                                      fit a warp's working column): taken by the CTA-level lock-free reduction */
    int64_t n_reduce_displaced;    /* times a column took a pivot row from a later column that had claimed it first */
    int64_t reduce_arena_bytes;    /* device bytes of reduced columns and working buffers the reduction used */
    int32_t key_bits;              /* bits of the diameter rank inside a packed record */
    int32_t index_bits;            /* bits of the vertex word inside a packed column record */
    int32_t sort_passes;           /* radix passes run by the filtration sort */
    int32_t pair_sort_passes;      /* radix passes run by the pair sort */
} rips_stats_t;

/* Device time per step of dimension d, milliseconds, CUDA events on the library's stream
 * (host-side pieces by a host clock).  Valid after the stream has been synchronised. */
typedef struct {
    float clear_bitmap_ms;   /* a4: clearing bitmap built from P_{d-1} */
    float enumerate_ms;      /* a3-a5 + a7: the fused kernel (enumerate, diameter, filter, slot/compaction, apparent test) */
    float sort_hist_ms;      /* a6: digit histograms (~0 when the fused kernel accumulated them) */
    float sort_pass_ms;      /* a6: all onesweep passes */
    float apparent_ms;       /* a8: full sorts of the two small lists (irregular pairs, non-apparent columns), on side
                                streams beside the fused kernel's successors */
    float pair_hist_ms;      /* a9: ~0 (the histogram is accumulated by the fused kernel, its scan runs inside the pass kernel) */
    float pair_sort_ms;      /* a9: stable partition of the pair slots by cofacet vertex (onesweep passes) */
    float stage1_ms;         /* whole stage 1 as enqueued (including memsets, scalar read-back) */
    float stage2_ms;         /* whole stage 2: from its first launch (beside stage 1's sort) to the join on the main stream */
    float dim0_ms;           /* d == 0 only: edge sort is part of rips_init; this is the union-find kernel */
    float reduce_device_ms;  /* NOT hot path: the reduction of the non-apparent columns, all of it on the device (host clock
                                around the kernels, their set-up and the read-back of the counters) */
    float reduce_host_ms;    /* always 0: no part of the reduction runs on the host (kept for the round-1 layout) */
    float reduce_xfer_ms;    /* NOT hot path: D2H copy of the bars */
} rips_timings_t;

/* Upper bound, in bytes, of the workspace rips_init + rips_compute + every accessor of dimensions 0..dim_max use for n
 * points with no threshold (a threshold only lowers the use), including 256 MB / 64 bytes per candidate of arena for
 * the reduced columns of rips_reduce.  What it does NOT bound: the reduced columns of inputs on which they fill in
 * ("difficult datasets"; e.g. a 400-point random matrix needs 42 GB in dimension 1) and the stages at
 * d = dim_max + 1.  RIPS_EOVERFLOW if the sizes do not fit. */
int rips_workspace_bytes(int64_t n, int dim_max, int64_t* bytes);

/* After a call on this thread returned RIPS_ENOMEM: the workspace size with which that request would have fitted (the
 * size in use, fragmentation included, plus the request), 0 if unknown. */
int64_t rips_last_required_bytes(void);

/* Create a context.  dist_lower: n(n-1)/2 fp32, HOST or DEVICE pointer (detected), layout above.
 * dim_max in [0,4]: H_0..H_dim_max.  threshold: keep simplices of diameter <= threshold
 * (inclusive); +INFINITY = full complex; the library never substitutes the
 * enclosing radius on its own.
 * workspace_dev / workspace_bytes: DEVICE memory (256-byte aligned) every device array of the context is carved
 * from; it stays the caller's, must outlive the context, and nothing in the library allocates or frees device
 * memory between rips_init and rips_free.  A request that does not fit returns RIPS_ENOMEM (the size that would
 * have fitted: rips_last_required_bytes); the context stays usable.  workspace_dev = NULL: rips_init allocates the
 * workspace itself (cudaMalloc, sized for this input and threshold; freed by rips_free) and adds to it only if a
 * computation needs more than was foreseen.
 * stream: a cudaStream_t cast to void*, NULL = the default stream.  Validates the matrix (RIPS_EINVAL on NaN,
 * negative or infinite entries), copies it, ranks the distinct edge values on the device and builds the binomial
 * table.  */
int rips_init(rips_ctx** out, const float* dist_lower, int64_t n, int dim_max, float threshold, void* workspace_dev,
              int64_t workspace_bytes, void* stream);

/* Which stage 1 the context runs; to be called before the first rips_stage1 / rips_compute.
 *   RIPS_MODE_DENSE   every one of the C(n, d+1) combinatorial indices is enumerated (Algorithms 7-8 as printed);
 *   RIPS_MODE_SPARSE  the sparse option of the paper (PAPER.md:395-437 Algorithm 5, :591, :932-934): neighbour lists of
 *                     the edges within the threshold, the simplices of dimension d made from those of dimension d-1,
 *                     cofacets from common neighbours; memory and time follow the size of the complex, not C(n, d+1);
 *   RIPS_MODE_AUTO    (default) sparse iff the threshold admits less than 5 % of the edges (and n >= 64).
 * Every array either mode exposes is the same (the tests compare both with the oracle). */
enum { RIPS_MODE_AUTO = 0, RIPS_MODE_DENSE = 1, RIPS_MODE_SPARSE = 2 };
int rips_set_mode(rips_ctx* ctx, int mode);

/* Dimension 0 .. dim_max, all stages: dim 0, then per d: stage 1, stage 2, reduction. */
int rips_compute(rips_ctx* ctx);

/* The two hot-path stages, separately callable for d in [1, dim_max+1] (benches, and the scale row
 * of DESIGN.md: stage 1 at d = dim_max+1 enumerates the C(n, dim_max+2) simplices the configs
 * name).  rips_stage1(d) needs the pivots of dimension d-1 (rips_compute, or rips_dim0 for d = 1);
 * rips_stage2(d) needs rips_stage1(d).  Both may be called repeatedly: the pivots an earlier
 * rips_reduce(d) found depend only on the input and stay valid, so after one rips_compute the loop
 * "for d: rips_stage1(d); rips_stage2(d)" re-runs the whole hot path (bench.py's step). */
int rips_dim0(rips_ctx* ctx);
int rips_stage1(rips_ctx* ctx, int d);
int rips_stage2(rips_ctx* ctx, int d);
/* Reduction of the non-apparent columns of dimension d (after rips_stage2(d)); completes the pivots
 * of dimension d.  Not the hot path, timed separately. */
int rips_reduce(rips_ctx* ctx, int d);
/* Alternative to rips_reduce(d) for a reduction done elsewhere (the paper's own split runs it on the
 * host): installs `count` pivots (t_host[i], s_host[i]), HOST arrays ascending by t, as the
 * pivots of dimension d that are not apparent pairs (the third layer of the pair store).  They join the
 * apparent pairs in rips_pivots / rips_pivot_lookup and in the clearing set of dimension d+1.  No bars
 * are produced for dimension d.  Needs rips_stage2(d).  RIPS_EINVAL if t is not strictly ascending. */
int rips_import_pivots(rips_ctx* ctx, int d, const uint64_t* t_host, const uint64_t* s_host, int64_t count);

/* Bars of dimension d: 2*count floats (birth, death) on the HOST; death = +INFINITY for essential
 * classes; zero-length bars omitted.  Order: d = 0: by ascending index of the merging edge, then
 * the essential classes; d >= 1: column (coboundary) order of the birth simplex. */
int rips_barcodes(rips_ctx* ctx, int d, const float** birth_death_host, int64_t* count);

/* Filtration array C of dimension d >= 1 in coboundary order. */
int rips_filtration(rips_ctx* ctx, int d, const float** diam_dev, const uint64_t** cidx_dev, int64_t* len);
/* Apparent pairs of dimension d, ascending by cidx(t). */
int rips_apparent_pairs(rips_ctx* ctx, int d, const uint64_t** t_dev, const uint64_t** s_dev, int64_t* n_app);
/* Non-apparent columns in coboundary order. */
int rips_nonapparent(rips_ctx* ctx, int d, const float** diam_dev, const uint64_t** cidx_dev, int64_t* n_non);
/* All pivots of dimension d (apparent pairs united with the reduced ones), ascending by cidx(t).
 * d = 0: t = merging edge, s = the vertex that gave birth to the dying component. */
int rips_pivots(rips_ctx* ctx, int d, const uint64_t** t_dev, const uint64_t** s_dev, int64_t* n_piv);
/* Two-layer pair store lookup: s_out_dev[i] = cidx(s) of the pivot whose row is
 * t_query_dev[i], or -1.  Device binary search over the sorted arrays. */
int rips_pivot_lookup(rips_ctx* ctx, int d, const uint64_t* t_query_dev, int64_t m, int64_t* s_out_dev);

int rips_stats(rips_ctx* ctx, int d, rips_stats_t* out);
int rips_timings(rips_ctx* ctx, int d, rips_timings_t* out);

/* Size of the context's workspace in bytes (constant between rips_init and rips_free with a caller's workspace). */
int rips_device_bytes(rips_ctx* ctx, int64_t* bytes);
/* Bytes of the workspace handed out right now, and the largest value that has had (peak may be NULL). */
int rips_workspace_in_use(rips_ctx* ctx, int64_t* bytes, int64_t* peak);
/* Number of kernels this context has launched so far. */
int rips_kernel_launches(rips_ctx* ctx, int64_t* launches);

/* Standalone primitive, exposed for tests and benches: stable LSD onesweep radix sort of n 64-bit
 * records on bits [lo_bit, hi_bit) (ascending), device pointers, tmp_dev = n more records.  The
 * sorted data ends in keys_dev.  stream as in rips_init. */
int rips_sort_u64(uint64_t* keys_dev, uint64_t* tmp_dev, int64_t n, int lo_bit, int hi_bit, void* stream);

/* The same sort for callers that must not allocate (code under CUDA graph capture, tight serving loops, harnesses that
 * forbid cudaMalloc): rips_sort_u64 allocates and frees its scratch (histograms, tickets, look-back status words) with
 * cudaMalloc / cudaFree on every call; this entry point keeps that scratch in a static device array of 16 MiB inside the
 * library (every GPU that loads the library holds it until the process exits) and calls no cudaMalloc, cudaFree or
 * allocating library routine.  Same arguments, same result in keys_dev (tmp_dev = n more records, the caller's).
 *   - n <= 4,194,304 records (2^22: what the array is sized for); more: RIPS_EINVAL, rips_last_error says so.
 *   - Asynchronous: the work is enqueued on `stream` and the call returns; the result is valid once the stream has
 *     been synchronised.
 *   - The array is SHARED by every call on the device, whatever the stream or thread, and keeps the last call's
 *     contents (the call clears what must start at zero): calls that overlap on the GPU race.  Serialise them -- one
 *     stream, or an event between them. */
int rips_sort_u64_static(uint64_t* keys_dev, uint64_t* tmp_dev, int64_t n, int lo_bit, int hi_bit, void* stream);

const char* rips_strerror(int code);
/* Text of the last CUDA error seen by this thread's calls ("" if none). */
const char* rips_last_error(void);
void rips_free(rips_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* RIPS_H */
