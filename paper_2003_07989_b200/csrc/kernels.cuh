// kernels.cuh -- host-side launchers of the kernels (definitions in stage1.cu, stage2.cu, dim0.cu,
// init.cu, reduce.cu).  Packed records used throughout the device path:
//
//   column record   (key << lowbits) | verts   key = descending dense rank of the diameter (0 = largest
//                                               distance); verts = the simplex's vertices, v[j] at bit
//                                               j*vbits, vbits = bits of n-1, lowbits = (d+1)*vbits.
//                                               The vertex word orders simplices exactly like cidx does
//                                               (colex order = lexicographic on the decreasing vertex
//                                               tuple, Remark 2), and spares every consumer
//                                               the inverse of Eq. 2.
//   regular pair    (v << tbits) | cidx(t)     v = the cofacet vertex, above every vertex of s (apparent.cuh)
//   irregular pair  (cidx(t) << 3) | j         j = position of the added vertex v inside t
//                                               (number of vertices of s below v); s = t minus that vertex
//
// Both are bijective encodings of the paper's (diameter, cidx) struct and
// (t, s) key-value pair; the fp32 / two-array forms the C ABI exposes are produced
// from them by the unpack kernels.
#pragma once
#include "common.cuh"

#define RIPS_MAX_M 6           // vertices of a column simplex: d+1 <= 6  (dim_max <= 4, scale row d = dim_max+1)
#define RIPS_PAIR_POS_BITS 3

// ------------------------------------------------------------------ init.cu
// rec[e] = (~bits(dist[e]) << 32) | e ; dist canonicalised in place (-0 -> +0); *bad |= 1 on NaN / inf / negative
// (values above the threshold are all ranked as one class, +inf)
// *n_over += number of such edges
cudaError_t launch_prep_edges(float* dist, i64 E, u64* rec, int* bad, float threshold, u64* n_over, cudaStream_t st);
// sorted rec (value descending, e ascending) -> K[e] = dense rank, values[rank]; *n_distinct
cudaError_t launch_rank_edges(const u64* rec_sorted, i64 E, u32* K, float* values, u64* status, u32* ticket,
                              u64* n_distinct, cudaStream_t st);
i64 rank_edges_tiles(i64 E);
// Kf (see common.cuh) from K: n*n entries of u16 (kf_u16 != 0) or u32
cudaError_t launch_build_full_keys(const u32* K, int n, int pitch, void* Kf, int kf_u16, cudaStream_t st);
// Sf[i*spitch + b] = max of Kf[i][32b .. 32b+31] (same entry type as Kf); spitch >= ceil(n / 32).  Built by rips_init
// from SUMMARY_MIN_N points on: below that a scan of all vertices is a few warp steps and the table buys nothing.
#ifdef RIPS_STRESS
constexpr int SUMMARY_MIN_N = 8;     // the small inputs of the stress tests take the summary-guided scan too
#else
constexpr int SUMMARY_MIN_N = 2048;
#endif
cudaError_t launch_build_block_max(const void* Kf, int n, int pitch, void* Sf, int spitch, int kf_u16, cudaStream_t st);

// ------------------------------------------------------------------ dim0.cu
struct Dim0Out {
    u64* pair_ts;   // [n-1] packed (edge cidx << 16) | birth vertex of the dying component, in merge order
    float* death;   // [n-1] diameter of the merging edge
    u32* n_pairs;   // scalar
};
cudaError_t launch_dim0(const u64* rec_sorted, i64 E, int n, u32 thr_bits_inv, u32* parent_maxv /*2n*/, Dim0Out out,
                        cudaStream_t st);

// ------------------------------------------------------------------ stage1.cu
struct ClearSet {
    const u32* bitmap;     // bit idx set <=> idx is a pivot row of dimension d-1 (NULL: use the sorted arrays)
    const u64* layer1;     // sorted packed pair records of dimension d-1 (t = rec >> shift1)
    i64 n1;
    int shift1;
    const u64* layer2;     // sorted t of the reduced pivots
    i64 n2;
};
// digits of a radix sort whose histogram a producer kernel accumulates while it writes the records
struct FusedHist {
    u64* hist;        // [npasses][256] raw counts, zeroed by the caller; NULL = not fused
    int npasses;      // <= 3 for the filtration sort, <= 2 for the pair partition (S1_MAX_FUSED, S1_MAX_FUSED_P)
    int shift[4], bits[4];
};
// Counters written by the fused kernel (u64 each)
enum { S1C_KEPT = 0, S1C_OVER = 1, S1C_CLEARED = 2, S1C_REGULAR = 3, S1C_IRREGULAR = 4, S1C_NONAPP = 5, S1C_STAGE_OVERFLOW = 6 };

struct Stage1Params {
    const void* Kf;   // full key matrix (u16 or u32, see launch_stage1's kf_u16), row pitch `pitch` entries
    int pitch;
    const void* Sf;   // block maxima of Kf's rows (launch_build_block_max), or NULL: the warp scan then reads every vertex
    int spitch;
    BinomTable bt;
    int n;
    u64 total;        // C(n, d+1)
    i64 tiles;        // warp chunks
    int chunk;        // candidates per warp chunk (stage1_chunk)
    int stage_cap;    // compact mode: records a warp can stage per chunk (stage1_stage_cap)
    u32 thr_key;      // keep iff key >= thr_key
    u32 sentinel_key; // key field of the column sentinel (= number of distinct keys, larger than every key)
    int vbits, lowbits;
    int tbits;        // bits of the row index field of a regular pair record (holds C(n, d+2) as well)
    ClearSet clear;
    int compact;      // 0: one slot per candidate, sentinels in the dropped ones (sorted away afterwards);
                      // 1: survivors compacted in increasing index with a decoupled look-back
    int count_only;   // 1: only counters[S1C_KEPT/OVER/CLEARED] are produced
    int fast_visits;  // cofacet vertices each lane tests on its own before the warp takes over its scan (<= 32)
    u64* cols_out;    // packed column records
    u64* pairs_out;   // same slots: regular pair record (v << tbits) | cidx(t), or the pair sentinel (n << tbits)
    u64* irr_out;     // irregular apparent pairs (cidx(t) << 3) | j, unordered; capacity irr_cap
    u64* non_out;     // non-apparent column records, unordered; capacity non_cap
    u64 irr_cap, non_cap;
    u64* status;      // one word per warp chunk, zeroed (compact mode)
    u32* ticket;      // zeroed
    u64* counters;    // S1C_*, zeroed
    FusedHist fh_cols;   // digit histogram of the filtration sort (over every slot written to cols_out)
    FusedHist fh_pairs;  // digit histogram of the partition of pairs_out by v
};
int stage1_chunk(u64 total, int compact, double est_survival, int retry, int sms);
int stage1_stage_cap();
cudaError_t launch_stage1(int M, int kf_u16, const Stage1Params& p, cudaStream_t st);
// the three sorted layers of dimension d-1's pivots, as the clearing bitmap's kernel reads them
struct ClearLayers {
    const u64* reg; i64 n_reg; int reg_tbits; u64 reg_mask, reg_sentinel;   // (v << tbits) | cidx(t); v == sentinel: no pair in this slot
    const u64* irr; i64 n_irr; const u64* n_irr_dev; int irr_shift;         // (cidx(t) << shift) | j; count on the device (may be NULL)
    const u64* red; i64 n_red;                                              // cidx(t)
};
cudaError_t launch_clear_bitmap(u32* bitmap, const ClearLayers& L, int sms, cudaStream_t st);

// ------------------------------------------------------------------ sparse.cu (the sparse path, Algorithm 5)
struct SparseExpand {
    const u64* in;    // simplices of MP vertices as vertex words (NULL for MP = 1: the vertices 0..n_in-1)
    i64 n_in;
    const void* Kf;
    int pitch, vbits;
    u32 thr1;         // an edge is admissible iff its entry of Kf is >= thr1
    const u64* off;   // CSR of the admissible edges: off[n+1], adj ascending per vertex
    const u32* adj;
    u32* cnt;         // [n_in] simplices made from each input simplex (count pass)
    const u64* pos;   // [n_in] exclusive scan of cnt (write pass)
    u64* out;         // simplices of MP+1 vertices, grouped by input simplex, the new (top) vertex ascending
};
struct SparseParams {
    const u64* simp;  // all simplices of M vertices within the threshold, vertex words, increasing combinatorial index
    i64 n_simp;
    const void* Kf;
    int pitch, n;
    BinomTable bt;
    int vbits, lowbits, tbits;
    u32 sentinel_key;
    const u64* off;
    const u32* adj;
    const u64* c_reg; i64 n_reg; u64 reg_mask;   // clearing set: the three sorted layers of dimension d-1's pivots
    const u64* c_irr; i64 n_irr;
    const u64* c_red; i64 n_red;
    u64* cols_out;    // [n_simp] column record or sentinel (slot = position in simp)
    u64* pairs_out;   // [n_simp] regular pair record or sentinel
    u64* irr_out; u64* non_out; u64 irr_cap, non_cap;
    u64* counters;    // S1C_*
};
i64 sparse_scan_tiles(i64 n);
cudaError_t launch_csr_count(const void* Kf, int kf_u16, int n, int pitch, u32 thr1, u32* deg, cudaStream_t st);
cudaError_t launch_csr_scan(const u32* deg, int n, u64* off, cudaStream_t st);
cudaError_t launch_csr_fill(const void* Kf, int kf_u16, int n, int pitch, u32 thr1, const u64* off, u32* adj, cudaStream_t st);
cudaError_t launch_scan_counts(const u32* cnt, i64 n, u64* pos, u64* status, u32* ticket, cudaStream_t st);
cudaError_t launch_expand(int MP, int kf_u16, const SparseExpand& e, bool write, cudaStream_t st);
cudaError_t launch_sparse_apparent(int M, int kf_u16, const SparseParams& p, cudaStream_t st);

// ------------------------------------------------------------------ pair store, unpack, lookup (stage2.cu)
// The two sorted layers of apparent pairs of one dimension (the third layer, the pivots found by the
// reduction, is a pair of plain arrays).
struct PairLayers {
    const u64* reg;   // (v << tbits) | cidx(t), ascending; s = t minus its top vertex v
    i64 n_reg;
    const u64* irr;   // (cidx(t) << 3) | j, ascending
    i64 n_irr;
    int tbits;
};
// packed column records -> diam[], cidx[] (M = vertices of the simplex; cidx by Eq. 2)
cudaError_t launch_unpack_columns(int M, const u64* cols, i64 len, int vbits, BinomTable bt, const float* values,
                                  float* diam, u64* cidx, cudaStream_t st);
// both apparent layers -> t[], s[] ascending by t   (M = vertices of s)
cudaError_t launch_merge_apparent(int M, const PairLayers& L, BinomTable bt, int n, u64* t, u64* s, cudaStream_t st);
// merge of two (t, s) arrays, both ascending by t, all t distinct
cudaError_t launch_merge_ts(const u64* t1, const u64* s1, i64 n1, const u64* t2, const u64* s2, i64 n2, u64* t, u64* s,
                            cudaStream_t st);
cudaError_t launch_pivot_lookup(int M, const PairLayers& L, BinomTable bt, int n, const u64* red_t, const u64* red_s,
                                i64 n2, const u64* query, i64 m, i64* s_out, cudaStream_t st);

// ------------------------------------------------------------------ reduce.cu (not the hot path)
// Reference to a reduced column in the arena: bit 63 = sorted, bits 62..27 = offset (entries), bits 26..0 = length.
#define RD_REF(off, len, sorted) (((u64)(sorted) << 63) | ((u64)(off) << 27) | (u64)(len))
#define RD_REF_OFF(r) (((r) >> 27) & ((1ull << 36) - 1ull))
#define RD_REF_LEN(r) ((r) & ((1ull << 27) - 1ull))
#define RD_REF_SORTED(r) ((r) >> 63)
enum { RDC_ARENA_TOP = 0, RDC_ADDS = 1, RDC_TODO = 2, RDC_TICKET = 3, RDC_STEALS = 4, RDC_PIVOTS = 5, RDC_NBARS = 6, RDC_NESS = 7, RDC_DBG = 8, RDC_COUNT = 14 };
enum { RD_ERR_ARENA = 1, RD_ERR_SORTCAP = 2, RD_ERR_PROTOCOL = 4, RD_ERR_STUCK = 8 };

struct ReduceParams {
    const u64* cols;      // non-apparent column records, coboundary order
    i64 ncols;
    const void* Kf;
    int pitch, n;
    BinomTable bt;
    int vbits, tbits;
    u32 thr_key;          // cofacets with key < thr_key are above the threshold
    PairLayers layers;    // apparent pairs of this dimension (first layer of the pair store)
    u64* piv;             // [ncols] 0 = zero column, ~0 = not reduced yet, else the pivot entry ((key << tbits | cidx(t)) + 1)
    u64* colref;          // [ncols] RD_REF of the column's published reduced column
    unsigned char* todo;  // [ncols] 1 = reduce_kernel has to take the column
    u64* ht_keys;         // second layer of the pair store: open addressing, ~0 = empty
    u32* ht_vals;         // owning column, 0xffffffff = none
    u32 ht_mask;
    u64* arena;           // reduced columns and working buffers
    u64 arena_cap;        // entries
    int sort_cap;         // entries a CTA can sort in shared memory (>= n, >= 2048, a power of two)
    int workers;          // CTAs of reduce_kernel
    u64* counters;        // RDC_*, zeroed
    u32* error;           // RD_ERR_* flags, zeroed
};
size_t reduce_smem_bytes(int sort_cap);
int reduce_sort_cap(int n);
int reduce_workers(int sms, int sort_cap);
// prereduce_kernel, claim_kernel, worklist_kernel, reduce_kernel: afterwards piv[] holds every column's pivot
cudaError_t launch_reduce(int M, int kf_u16, const ReduceParams& p, int sms, cudaStream_t st);
// rec[j] = (cidx(t) << jbits) | j (all ones for a zero column); counters[RDC_PIVOTS] += columns with a pivot
cudaError_t launch_pivot_records(const ReduceParams& p, int jbits, u64* rec, cudaStream_t st);
// rec sorted by t -> t_out[i], s_out[i] = cidx of the column (Eq. 2)
cudaError_t launch_pivot_arrays(int M, const ReduceParams& p, int jbits, const u64* rec, i64 n_piv, u64* t_out, u64* s_out,
                                cudaStream_t st);
// bars (birth, death) in column order, zero-length ones dropped, +inf for zero columns; counts to n_bars / n_essential
cudaError_t launch_bars(const ReduceParams& p, int lowbits, const float* values, float* bars, u64* n_bars, u64* n_essential,
                        cudaStream_t st);
