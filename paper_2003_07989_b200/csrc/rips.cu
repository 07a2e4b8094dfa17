// rips.cu -- context, per-dimension driver and the C ABI of include/rips.h.
// Control flow (Fig. 3(b)): dim 0, then per d: stage 1 (clearing bitmap -> fused
// enumerate / filter / apparent-test kernel -> onesweep sort of the columns), stage 2 (sorts of the two
// small lists, stable partition of the pair slots: on side streams, beside stage 1's sort), reduction
// of the few non-apparent columns (device pre-reduction, serial remainder on the host; not hot path).
#include "../../include/rips.h"

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "kernels.cuh"
#include "radix_sort.cuh"

namespace {

thread_local std::string g_last_error;

int cuda_fail(cudaError_t e, const char* what)
{
    g_last_error = std::string(what) + ": " + cudaGetErrorString(e);
    return RIPS_ECUDA;
}
#define CU(x)                                        \
    do {                                             \
        cudaError_t e__ = (x);                       \
        if (e__ != cudaSuccess) return cuda_fail(e__, #x); \
    } while (0)
#define RC(x)                  \
    do {                       \
        int r__ = (x);         \
        if (r__ != RIPS_OK) return r__; \
    } while (0)

// A device buffer that is reused while large enough; carved from the context's workspace (Pool).
struct DevBuf {
    void* p = nullptr;
    size_t cap = 0;
};

// The workspace: one device allocation (the caller's, or the library's own made by rips_init) managed on the host
// as a list of blocks, first fit, 256-byte granules.  Nothing between rips_init and rips_free calls cudaMalloc /
// cudaFree, unless the library owns the workspace AND a computation needs more than rips_workspace_bytes foresaw
// (the reduced columns of a difficult input, views of thresholded inputs): then a further chunk is added.
struct Pool {
    struct Chunk {
        unsigned char* base = nullptr;
        size_t size = 0;
        bool owned = false;
        struct Blk { size_t off, size; bool used; };
        std::vector<Blk> blks;
    };
    std::vector<Chunk> chunks;
    bool may_grow = false;
    size_t in_use = 0, peak = 0;

    static size_t round(size_t b) { return (b + 255) & ~(size_t)255; }
    void add_chunk(void* base, size_t size, bool owned)
    {
        Chunk ch;
        ch.base = (unsigned char*)base;
        ch.size = size & ~(size_t)255;
        ch.owned = owned;
        ch.blks.push_back({0, ch.size, false});
        chunks.push_back(std::move(ch));
    }
    void* alloc(size_t bytes)
    {
        bytes = round(bytes ? bytes : 1);
        for (Chunk& ch : chunks)
            for (size_t i = 0; i < ch.blks.size(); ++i) {
                Chunk::Blk& b = ch.blks[i];
                if (b.used || b.size < bytes) continue;
                if (b.size > bytes) {
                    Chunk::Blk rest{b.off + bytes, b.size - bytes, false};
                    b.size = bytes;
                    b.used = true;
                    const size_t off = b.off;
                    ch.blks.insert(ch.blks.begin() + (long)i + 1, rest);
                    in_use += bytes;
                    peak = std::max(peak, in_use);
                    return ch.base + off;
                }
                b.used = true;
                in_use += bytes;
                peak = std::max(peak, in_use);
                return ch.base + b.off;
            }
        return nullptr;
    }
    void free(void* p)
    {
        if (!p) return;
        for (Chunk& ch : chunks) {
            if ((unsigned char*)p < ch.base || (unsigned char*)p >= ch.base + ch.size) continue;
            const size_t off = (size_t)((unsigned char*)p - ch.base);
            for (size_t i = 0; i < ch.blks.size(); ++i) {
                if (ch.blks[i].off != off || !ch.blks[i].used) continue;
                ch.blks[i].used = false;
                in_use -= ch.blks[i].size;
                if (i + 1 < ch.blks.size() && !ch.blks[i + 1].used) { ch.blks[i].size += ch.blks[i + 1].size; ch.blks.erase(ch.blks.begin() + (long)i + 1); }
                if (i > 0 && !ch.blks[i - 1].used) { ch.blks[i - 1].size += ch.blks[i].size; ch.blks.erase(ch.blks.begin() + (long)i); }
                return;
            }
        }
    }
    size_t largest_free() const
    {
        size_t m = 0;
        for (const Chunk& ch : chunks)
            for (const Chunk::Blk& b : ch.blks)
                if (!b.used) m = std::max(m, b.size);
        return m;
    }
    size_t total() const
    {
        size_t t = 0;
        for (const Chunk& ch : chunks) t += ch.size;
        return t;
    }
};

thread_local int64_t g_required_bytes = 0;

enum Ev {
    EV_S1_BEGIN, EV_S1_BITMAP, EV_S1_ENUM, EV_S1_SORTBEG, EV_S1_HIST, EV_S1_SORT, EV_S1_END,
    EV_S2_BEGIN, EV_S2_APP, EV_S2_SORTBEG, EV_S2_HIST, EV_S2_SORT, EV_S2_END,
    EV_D0_BEGIN, EV_D0_END, EV_COUNT
};

struct DimState {
    // sizes
    u64 total = 0;   // C(n, d+1)
    int M = 0;       // d + 1
    int cbits = 0, tbits = 0, lowbits = 0;
    int compact = 0;
    // stage 1: column records (sorted), pair slots (unsorted until stage 2), the two small lists
    bool have_s1 = false;
    DevBuf colsA, colsB, s1_status, bitmap, pairsA, pairsB, irrA, irrB, nonA, nonB, pair_scratch, d_cnt;
    u64* h_cnt = nullptr;         // pinned: the fused kernel's counters, copied behind it
    cudaEvent_t ev_cnt = nullptr; // ... and the event of that copy
    bool counts_pending = false;  // h_cnt has not been read yet
    bool cnt_copied = false;      // ev_cnt has been recorded at least once
    bool caps_valid = false;      // a run of this dimension has fitted its lists: the sizes are known to suffice
    u64 irr_cap = 0, non_cap = 0; // capacities of the two small lists (records)
    int chunk_retry = 0, attempts = 0;
    size_t arena_hint = 0;        // reduction: arena size to start from
    DevBuf simpA, simpB;          // sparse path: all simplices of this dimension within the threshold (vertex words)
    const u64* simp = nullptr;    // ... in increasing combinatorial index
    i64 n_simp = -1;
    i64 sparse_over = 0;          // sparse path: candidates never enumerated (diameter above the threshold)
    // stage 1 + stage 2 of this dimension as one CUDA graph (captured once the sizes are known to fit)
    cudaGraphExec_t graph = nullptr;
    u64 graph_sig = 0;
    i64 graph_launches = 0;
    DevBuf rd_piv, rd_colref, rd_todo, rd_htk, rd_htv, rd_arena, rd_cnt, rd_rec, rd_rec2, rd_bars; // reduction
    u64* cols = nullptr; // sorted packed column records (points into colsA or colsB)
    i64 len = 0;         // columns
    i64 exact_kept = -1; // compact mode: columns counted by the first run of this dimension (a constant of the context)
    i64 slots = 0;       // records in the column / pair arrays (len in compact mode, else C(n,d+1) with sentinels)
    SortPlan pair_plan;
    bool pair_fused = false, pairs_fresh = false;
    // stage 2: the sorted layers of the pair store
    bool have_s2 = false;
    u64* reg = nullptr;  // regular pairs, ascending (first n_reg records of the partitioned pair slots)
    u64* irr = nullptr;  // irregular pairs, ascending
    u64* non = nullptr;  // non-apparent columns, coboundary order
    i64 n_reg = 0, n_irr = 0, n_non = 0;
    // reduction (second layer), sorted by t
    bool have_red = false;
    DevBuf red_t, red_s;
    i64 n_red = 0;
    // lazily materialised views
    DevBuf v_fdiam, v_fcidx, v_at, v_as, v_ndiam, v_ncidx, v_pt, v_ps;
    bool has_vf = false, has_va = false, has_vn = false, has_vp = false;
    std::vector<float> bars;
    rips_stats_t stats;
    rips_timings_t tim;
    cudaEvent_t ev[EV_COUNT];
    bool ev_rec[EV_COUNT];
    bool ev_made = false;
};

} // namespace

struct rips_ctx {
    i64 n = 0, E = 0;
    int dim_max = 0;
    float threshold = 0;
    cudaStream_t stream = 0;
    cudaStream_t stream2 = nullptr; // stage 2's sorts run here, beside the filtration sort of stage 1 on `stream`
    cudaStream_t stream3 = nullptr; // the sort of the non-apparent columns, beside the other two
    cudaEvent_t ev_join = nullptr, ev_join3 = nullptr, ev_fused = nullptr;
    int kmax = 0; // binomial table holds C(v,k), k <= kmax
    std::vector<u64> h_binom;
    float* d_dist = nullptr;
    u64* d_edges = nullptr; // sorted edge records (value descending, cidx ascending)
    u32* d_K = nullptr;
    void* d_Kf = nullptr;  // full symmetric matrix of key+1 (common.cuh)
    void* d_Sf = nullptr;  // block maxima of its rows (n >= SUMMARY_MIN_N; kernels.cuh), else NULL
    int sf_pitch = 0;
    int kf_u16 = 0, kf_pitch = 1, vbits = 1;
    int sms = 148;       // multiprocessors of the device
    bool use_graphs = true;  // switched off for the context if a capture fails
    bool capturing = false;
    cudaStream_t cap_stream = nullptr; // captures are made on this stream (the caller's may be the legacy default stream, which cannot capture)
    float* d_values = nullptr;
    u64* d_binom = nullptr;
    u64* d_counters = nullptr; // 16 u64 scratch counters
    u32* d_tickets = nullptr;  // 8 u32
    u64* h_counters = nullptr; // pinned
    u64* h_dimcnt = nullptr;   // pinned: 8 u64 per dimension (DimState::h_cnt)
    u32 n_distinct = 0, thr_key = 0;
    double edge_share = 1.0; // share of the edges the threshold admits
    int mode = 0;            // RIPS_MODE_*
    bool sparse = false, mode_locked = false; // the path stage 1 takes, fixed by the first stage 1
    DevBuf sp_deg, sp_off, sp_adj, sp_cnt, sp_pos, sp_status; // sparse path: CSR of the admissible edges, expansion scratch
    bool have_csr = false;
    int key_bits = 1;
    DevBuf sort_scratch, sort_scratch2, sort_scratch3;
    // dim 0
    DevBuf d0_pairs, d0_death, d0_uf;
    std::vector<DimState> dims; // index d, 0 .. dim_max+1
    Pool pool;
    DevBuf b_dist, b_edges, b_K, b_Kf, b_Sf, b_values, b_binom, b_counters, b_tickets, b_init_tmp, b_init_status;
    i64 launches = 0;
    BinomTable bt() const { return BinomTable{d_binom, (int)(n + 1)}; }
};

namespace {

int ensure(rips_ctx* c, DevBuf& b, size_t bytes)
{
    if (bytes == 0) bytes = 16;
    if (b.cap >= bytes) return RIPS_OK;
    if (b.p) { c->pool.free(b.p); b.p = nullptr; b.cap = 0; }
    void* q = c->pool.alloc(bytes);
    if (!q && c->pool.may_grow) {
        // the library owns the workspace and the estimate fell short: one more chunk
        size_t chunk = std::max<size_t>(Pool::round(bytes), (size_t)256 << 20);
        void* base = nullptr;
        cudaError_t e = cudaMalloc(&base, chunk);
        if (e != cudaSuccess) { cudaGetLastError(); chunk = Pool::round(bytes); e = cudaMalloc(&base, chunk); }
        if (e == cudaSuccess) {
            c->pool.add_chunk(base, chunk, true);
            q = c->pool.alloc(bytes);
        } else
            cudaGetLastError();
    }
    if (!q) {
        g_required_bytes = (int64_t)(c->pool.total() - c->pool.largest_free() + Pool::round(bytes));
        g_last_error = "workspace too small: " + std::to_string(bytes) + " more bytes needed with " + std::to_string(c->pool.in_use) + " of " +
                       std::to_string(c->pool.total()) + " in use (rips_last_required_bytes: " + std::to_string(g_required_bytes) + ")";
        return RIPS_ENOMEM;
    }
    b.p = q;
    b.cap = Pool::round(bytes);
    return RIPS_OK;
}
void release(rips_ctx* c, DevBuf& b)
{
    if (b.p) c->pool.free(b.p);
    b.p = nullptr;
    b.cap = 0;
}

void ev_record(rips_ctx* c, DimState& s, int which, cudaStream_t st = nullptr)
{
    if (!s.ev_made) {
        for (int i = 0; i < EV_COUNT; ++i) { cudaEventCreate(&s.ev[i]); s.ev_rec[i] = false; }
        s.ev_made = true;
    }
    // (inside a capture: an external event node, so that the event can be read from outside the graph)
    if (c->capturing) cudaEventRecordWithFlags(s.ev[which], st ? st : c->stream, cudaEventRecordExternal);
    else cudaEventRecord(s.ev[which], st ? st : c->stream);
    s.ev_rec[which] = true;
}
float ev_ms(DimState& s, int a, int b)
{
    if (!s.ev_made || !s.ev_rec[a] || !s.ev_rec[b]) return 0.f;
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, s.ev[a], s.ev[b]) != cudaSuccess) { cudaGetLastError(); return 0.f; }
    return ms;
}

// saturating binomial table, k-major
bool build_binom(i64 n, int kmax, std::vector<u64>& out)
{
    const size_t stride = (size_t)n + 1;
    out.assign((size_t)(kmax + 1) * stride, 0);
    for (size_t v = 0; v <= (size_t)n; ++v) out[v] = 1; // C(v,0)
    for (int k = 1; k <= kmax; ++k)
        for (size_t v = 1; v <= (size_t)n; ++v) {
            u64 a = out[(size_t)(k - 1) * stride + v - 1], b = out[(size_t)k * stride + v - 1];
            out[(size_t)k * stride + v] = (a > ~0ull - b) ? ~0ull : a + b;
        }
    return true;
}
u64 hbinom(const rips_ctx* c, i64 v, int k)
{
    if (k < 0 || v < 0 || k > c->kmax) return 0;
    return c->h_binom[(size_t)k * (c->n + 1) + v];
}

void invalidate_views(DimState& s, bool f, bool a, bool nn, bool p)
{
    if (f) s.has_vf = false;
    if (a) s.has_va = false;
    if (nn) s.has_vn = false;
    if (p) s.has_vp = false;
}

double now_ms()
{
    using namespace std::chrono;
    return duration<double, std::milli>(steady_clock::now().time_since_epoch()).count();
}

// ------------------------------------------------------------------------------------------ dim 0
int run_dim0(rips_ctx* c)
{
    DimState& s = c->dims[0];
    const i64 n = c->n;
    s.M = 1;
    s.total = (u64)n;
    s.stats = rips_stats_t{};
    s.stats.n_candidates = n;
    s.bars.clear();
    RC(ensure(c, c->d0_pairs, (size_t)n * 8));
    RC(ensure(c, c->d0_death, (size_t)n * 4));
    RC(ensure(c, c->d0_uf, (size_t)n * 8));
    i64 npairs = 0;
    ev_record(c, s, EV_D0_BEGIN);
    if (n >= 2 && c->threshold >= 0.0f) {
        u32 thr_bits;
        float thr = c->threshold;
        memcpy(&thr_bits, &thr, 4);
        CU(cudaMemsetAsync(c->d_counters, 0, 64, c->stream));
        Dim0Out out{(u64*)c->d0_pairs.p, (float*)c->d0_death.p, (u32*)c->d_counters};
        CU(launch_dim0(c->d_edges, c->E, (int)n, ~thr_bits, (u32*)c->d0_uf.p, out, c->stream));
        c->launches += 1;
        ev_record(c, s, EV_D0_END);
        CU(cudaMemcpyAsync(c->h_counters, c->d_counters, 8, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        npairs = (i64)(u32)c->h_counters[0];
    } else {
        ev_record(c, s, EV_D0_END);
    }
    // n-1 items at most: order them by edge index on the host, upload as the (only) pivot layer
    std::vector<u64> ts((size_t)npairs);
    std::vector<float> death((size_t)npairs);
    if (npairs) {
        CU(cudaMemcpy(ts.data(), c->d0_pairs.p, (size_t)npairs * 8, cudaMemcpyDeviceToHost));
        CU(cudaMemcpy(death.data(), c->d0_death.p, (size_t)npairs * 4, cudaMemcpyDeviceToHost));
    }
    std::vector<i64> order((size_t)npairs);
    for (i64 i = 0; i < npairs; ++i) order[i] = i;
    std::sort(order.begin(), order.end(), [&](i64 a, i64 b) { return ts[a] < ts[b]; });
    std::vector<u64> t((size_t)npairs), sv((size_t)npairs);
    for (i64 i = 0; i < npairs; ++i) {
        u64 r = ts[order[i]];
        t[i] = r >> 16;
        sv[i] = r & 0xffffu;
        float dd = death[order[i]];
        if (dd > 0.0f) { s.bars.push_back(0.0f); s.bars.push_back(dd); }
    }
    for (i64 i = 0; i < n - npairs; ++i) { s.bars.push_back(0.0f); s.bars.push_back(INFINITY); }
    RC(ensure(c, s.red_t, (size_t)npairs * 8));
    RC(ensure(c, s.red_s, (size_t)npairs * 8));
    if (npairs) {
        CU(cudaMemcpy(s.red_t.p, t.data(), (size_t)npairs * 8, cudaMemcpyHostToDevice));
        CU(cudaMemcpy(s.red_s.p, sv.data(), (size_t)npairs * 8, cudaMemcpyHostToDevice));
    }
    s.n_red = npairs;
    s.n_reg = s.n_irr = s.n_non = 0;
    s.reg = s.irr = s.non = nullptr;
    s.tbits = 1;
    s.have_s1 = s.have_s2 = s.have_red = true;
    s.caps_valid = true;
    s.counts_pending = false;
    s.slots = 0;
    s.irr_cap = 0;
    s.stats.n_columns = n;
    s.stats.n_reduced_pivots = npairs;
    s.stats.n_essential = n - npairs;
    s.stats.n_bars = (i64)s.bars.size() / 2;
    invalidate_views(s, true, true, true, true);
    return RIPS_OK;
}

// ------------------------------------------------------------------------------------------ stage 1
PairLayers layers_of(const DimState& s)
{
    PairLayers L;
    L.reg = s.reg;
    L.n_reg = s.n_reg;
    L.irr = s.irr;
    L.n_irr = s.n_irr;
    L.tbits = s.tbits;
    return L;
}

// Counters of the fused kernel of dimension d: copied to pinned host memory behind the kernel, read here.
// The first run of a dimension waits for them (the two small lists are provisioned by a rule of thumb and the
// launch is repeated if one overflowed); once a run has fitted, the sizes are known to fit -- they depend only on
// the context's input -- and rips_stage1 / rips_stage2 no longer wait for anything: the host reads the counters
// only when an accessor, rips_stats or rips_reduce asks for them.
int run_stage1(rips_ctx* c, int d);
int run_stage2(rips_ctx* c, int d);

int finish_counts(rips_ctx* c, int d)
{
    DimState& s = c->dims[d];
    if (!s.counts_pending) return RIPS_OK;
    CU(cudaEventSynchronize(s.ev_cnt));
    s.counts_pending = false;
    const u64* h = s.h_cnt;
    const u64 ni = h[S1C_IRREGULAR], nn = h[S1C_NONAPP];
    const bool stage_overflow = h[S1C_STAGE_OVERFLOW] != 0;
    if (ni > s.irr_cap || nn > s.non_cap || stage_overflow) {
        // rare: more irregular pairs / non-apparent columns than provisioned, or a chunk of compact mode kept more than
        // a warp can stage: both stages again with the sizes now known
        if (s.attempts >= 3) { g_last_error = "rips_stage1: list capacities still too small on the third attempt"; return RIPS_ECUDA; }
        ++s.attempts;
        s.irr_cap = std::max(s.irr_cap, ni);
        s.non_cap = std::max(s.non_cap, nn);
        if (stage_overflow) s.chunk_retry = 1;
        s.caps_valid = false;
        const bool had_s2 = s.have_s2;
        CU(cudaStreamSynchronize(c->stream));
        RC(run_stage1(c, d));
        if (had_s2) RC(run_stage2(c, d));
        return finish_counts(c, d);
    }
    s.attempts = 0;
    s.caps_valid = !c->sparse; // (the sparse path sizes its arrays by what it finds, run by run: it stays synchronous)
    s.len = s.compact ? (i64)h[S1C_KEPT] : (i64)(s.total - h[S1C_OVER] - h[S1C_CLEARED]); // slot mode counts what it drops
    s.n_reg = (i64)h[S1C_REGULAR];
    s.n_irr = (i64)ni;
    s.n_non = (i64)nn;
    s.stats.n_columns = s.len;
    s.stats.n_removed_by_diameter = (i64)h[S1C_OVER] + s.sparse_over;
    s.stats.n_cleared = (i64)h[S1C_CLEARED];
    s.stats.n_apparent = s.n_reg + s.n_irr;
    s.stats.n_nonapparent = s.n_non;
    s.stats.n_regular = s.n_reg;
    return RIPS_OK;
}

// ------------------------------------------------------------------------------------------ stage 1, sparse path
int ensure_csr(rips_ctx* c)
{
    if (c->have_csr) return RIPS_OK;
    const int n = (int)c->n;
    const u32 thr1 = c->thr_key + 1u;
    RC(ensure(c, c->sp_deg, (size_t)n * 4));
    RC(ensure(c, c->sp_off, (size_t)(n + 1) * 8));
    CU(launch_csr_count(c->d_Kf, c->kf_u16, n, c->kf_pitch, thr1, (u32*)c->sp_deg.p, c->stream));
    CU(launch_csr_scan((const u32*)c->sp_deg.p, n, (u64*)c->sp_off.p, c->stream));
    CU(cudaMemcpyAsync(c->h_counters, (u64*)c->sp_off.p + n, 8, cudaMemcpyDeviceToHost, c->stream));
    CU(cudaStreamSynchronize(c->stream));
    const u64 total = c->h_counters[0];
    RC(ensure(c, c->sp_adj, (size_t)total * 4));
    CU(launch_csr_fill(c->d_Kf, c->kf_u16, n, c->kf_pitch, thr1, (const u64*)c->sp_off.p, (u32*)c->sp_adj.p, c->stream));
    c->launches += 3;
    c->have_csr = true;
    return RIPS_OK;
}

// Sparse stage 1 (sparse.cu): the simplices of dimension d from those of dimension d-1 and the neighbour lists, in
// increasing combinatorial index; then one thread per simplex (key, clearing, apparent test) writes the records the
// dense kernels write in slot mode, the position in the list being the slot.  The sorts that follow are the dense ones.
int run_stage1_sparse(rips_ctx* c, int d)
{
    DimState& s = c->dims[d];
    DimState& prev = c->dims[d - 1];
    const i64 n = c->n;
    const int pvbits = bits_for((u64)n);
    RC(ensure_csr(c));
    // ---- the simplex list L_d
    const int MP = d; // vertices of the simplices it is made from
    const u64* in = nullptr;
    i64 n_in = n;
    if (d >= 2) {
        if (prev.n_simp < 0 || (prev.n_simp > 0 && !prev.simp)) {
            g_last_error = "rips_stage1: the sparse path needs the previous dimension's simplex list (run its stage 1 in sparse mode)";
            return RIPS_EINVAL;
        }
        in = prev.simp;
        n_in = prev.n_simp;
    }
    i64 total = 0;
    if (n_in > 0) {
        RC(ensure(c, c->sp_cnt, (size_t)n_in * 4));
        RC(ensure(c, c->sp_pos, (size_t)(n_in + 1) * 8));
        RC(ensure(c, c->sp_status, (size_t)sparse_scan_tiles(n_in) * 8 + 64));
        SparseExpand e;
        e.in = in; e.n_in = n_in; e.Kf = c->d_Kf; e.pitch = c->kf_pitch; e.vbits = c->vbits; e.thr1 = c->thr_key + 1u;
        e.off = (const u64*)c->sp_off.p; e.adj = (const u32*)c->sp_adj.p; e.cnt = (u32*)c->sp_cnt.p; e.pos = (const u64*)c->sp_pos.p; e.out = nullptr;
        CU(launch_expand(MP, c->kf_u16, e, false, c->stream));
        CU(cudaMemsetAsync(c->sp_status.p, 0, (size_t)sparse_scan_tiles(n_in) * 8 + 64, c->stream));
        u64* status = (u64*)c->sp_status.p + 8;
        CU(launch_scan_counts((const u32*)c->sp_cnt.p, n_in, (u64*)c->sp_pos.p, status, (u32*)c->sp_status.p, c->stream));
        CU(cudaMemcpyAsync(c->h_counters, (u64*)c->sp_pos.p + n_in, 8, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        total = (i64)c->h_counters[0];
        c->launches += 2;
        if (total > 0) {
            RC(ensure(c, s.simpA, (size_t)total * 8));
            RC(ensure(c, s.simpB, (size_t)total * 8));
            e.out = (u64*)s.simpA.p;
            CU(launch_expand(MP, c->kf_u16, e, true, c->stream));
            c->launches += 1;
            // stable partition by the new (top) vertex: increasing combinatorial index
            SortPlan pp = sort_make_plan(MP * c->vbits, (MP + 1) * c->vbits);
            RC(ensure(c, c->sort_scratch, sort_scratch_bytes(total, pp)));
            u64* res = nullptr;
            CU(sort_u64((u64*)s.simpA.p, (u64*)s.simpB.p, total, pp, c->sort_scratch.p, c->stream, &res, nullptr, &c->launches));
            s.simp = res;
        }
    }
    s.n_simp = total;
    s.sparse_over = (i64)s.total - total;
    s.compact = 1;
    s.slots = total;
    s.stats.n_slots = total;
    ev_record(c, s, EV_S1_BITMAP);
    if (total == 0) {
        ev_record(c, s, EV_S1_ENUM); ev_record(c, s, EV_S1_SORTBEG); ev_record(c, s, EV_S1_HIST); ev_record(c, s, EV_S1_SORT); ev_record(c, s, EV_S1_END);
        s.len = 0; s.n_reg = s.n_irr = s.n_non = 0;
        s.stats.n_removed_by_diameter = (i64)s.total;
        s.irr_cap = s.non_cap = 0;
        s.pair_plan = sort_make_plan(s.tbits, s.tbits + pvbits);
        s.pair_fused = false;
        s.have_s1 = true;
        s.pairs_fresh = true;
        return RIPS_OK;
    }
    RC(ensure(c, s.d_cnt, 128));
    u64* const d_cnt = (u64*)s.d_cnt.p;
    RC(ensure(c, s.colsA, (size_t)total * 8));
    RC(ensure(c, s.colsB, (size_t)total * 8));
    RC(ensure(c, s.pairsA, (size_t)total * 8));
    s.irr_cap = std::max<u64>(s.irr_cap, std::max<u64>(4096, (u64)total / 8));
    s.non_cap = std::max<u64>(s.non_cap, std::max<u64>(4096, (u64)total / 8));
    RC(ensure(c, s.irrA, (size_t)s.irr_cap * 8));
    RC(ensure(c, s.nonA, (size_t)s.non_cap * 8));
    SparseParams p;
    p.simp = s.simp; p.n_simp = total; p.Kf = c->d_Kf; p.pitch = c->kf_pitch; p.n = (int)n; p.bt = c->bt();
    p.vbits = c->vbits; p.lowbits = s.lowbits; p.tbits = s.tbits; p.sentinel_key = c->n_distinct;
    p.off = (const u64*)c->sp_off.p; p.adj = (const u32*)c->sp_adj.p;
    p.c_reg = (d >= 2) ? prev.reg : nullptr; p.n_reg = (d >= 2) ? prev.n_reg : 0;
    p.reg_mask = (prev.tbits >= 64) ? ~0ull : ((1ull << prev.tbits) - 1ull);
    p.c_irr = (d >= 2) ? prev.irr : nullptr; p.n_irr = (d >= 2) ? prev.n_irr : 0;
    p.c_red = (const u64*)prev.red_t.p; p.n_red = prev.n_red;
    p.cols_out = (u64*)s.colsA.p; p.pairs_out = (u64*)s.pairsA.p;
    p.irr_out = (u64*)s.irrA.p; p.non_out = (u64*)s.nonA.p; p.irr_cap = s.irr_cap; p.non_cap = s.non_cap;
    p.counters = d_cnt;
    CU(cudaMemsetAsync(d_cnt, 0, 128, c->stream));
    CU(launch_sparse_apparent(s.M, c->kf_u16, p, c->stream));
    c->launches += 1;
    ev_record(c, s, EV_S1_ENUM);
    {
        cudaStream_t sc = c->stream2 ? c->stream2 : c->stream;
        if (sc != c->stream) {
            CU(cudaEventRecord(c->ev_fused, c->stream));
            CU(cudaStreamWaitEvent(sc, c->ev_fused, 0));
        }
        CU(cudaMemcpyAsync(s.h_cnt, d_cnt, 64, cudaMemcpyDeviceToHost, sc));
        CU(cudaEventRecord(s.ev_cnt, sc));
        s.counts_pending = true;
        s.cnt_copied = true;
    }
    SortPlan plan = sort_make_plan(s.lowbits, s.lowbits + c->key_bits);
    s.pair_plan = sort_make_plan(s.tbits, s.tbits + pvbits);
    s.pair_fused = false;
    RC(ensure(c, c->sort_scratch, sort_scratch_bytes(total, plan)));
    RC(ensure(c, s.pair_scratch, sort_scratch_bytes(total, s.pair_plan)));
    {
        SortTimes st;
        st.enabled = true;
        st.ev[0] = s.ev[EV_S1_SORTBEG]; st.ev[1] = s.ev[EV_S1_HIST]; st.ev[2] = s.ev[EV_S1_SORT];
        s.ev_rec[EV_S1_SORTBEG] = s.ev_rec[EV_S1_HIST] = s.ev_rec[EV_S1_SORT] = true;
        u64* res = nullptr;
        CU(sort_u64((u64*)s.colsA.p, (u64*)s.colsB.p, total, plan, c->sort_scratch.p, c->stream, &res, &st, &c->launches, false,
                    s.M == 2 ? 0xffu : 0u)); // the keys of edges differ inside a warp, those of neighbouring triangles mostly do not
        s.cols = res;
        ev_record(c, s, EV_S1_END);
    }
    s.stats.sort_passes = total > 1 ? plan.npasses : 0;
    s.have_s1 = true;
    s.pairs_fresh = true;
    RC(finish_counts(c, d)); // the sparse path is synchronous: the sizes of the next steps come from these counts
    return RIPS_OK;
}

int run_stage1(rips_ctx* c, int d)
{
    if (d < 1 || d > c->dim_max + 1) return RIPS_EINVAL;
    DimState& s = c->dims[d];
    DimState& prev = c->dims[d - 1];
    if (!prev.have_red || !prev.have_s2) {
        g_last_error = "rips_stage1: pivots of the previous dimension are missing";
        return RIPS_EINVAL;
    }
    if (!prev.caps_valid) RC(finish_counts(c, d - 1)); // (only before the previous dimension's sizes are known to fit)
    const i64 n = c->n;
    s.M = d + 1;
    s.total = hbinom(c, n, d + 1);
    const u64 rows = hbinom(c, n, d + 2);
    if (rows == ~0ull) return RIPS_EOVERFLOW;
    s.cbits = bits_for(s.total ? s.total - 1 : 0);
    s.lowbits = s.M * c->vbits;
    s.tbits = bits_for(rows); // one value more than the row indices, so a field of all ones is never a row
    const int pvbits = bits_for((u64)n); // field of the cofacet vertex; n itself marks the pair sentinel
    if (c->key_bits + s.lowbits > 64 || pvbits + s.tbits > 64 || s.tbits + RIPS_PAIR_POS_BITS > 64) {
        g_last_error = "rips_stage1: a packed 64-bit record cannot hold this (n, dimension)";
        return RIPS_EOVERFLOW;
    }
    // The pivots found by an earlier rips_reduce(d) depend only on the input, so they stay valid
    // (have_red) while stage 1 / stage 2 are re-run; accessors additionally require have_s2.
    s.have_s1 = s.have_s2 = false;
    s.counts_pending = false;
    invalidate_views(s, true, true, true, true);
    rips_stats_t keep_stats = rips_stats_t{};
    if (s.have_red) {
        keep_stats.n_reduced_pivots = s.stats.n_reduced_pivots;
        keep_stats.n_essential = s.stats.n_essential;
        keep_stats.n_additions = s.stats.n_additions;
        keep_stats.n_bars = s.stats.n_bars;
        keep_stats.n_reduce_serial = s.stats.n_reduce_serial;
        keep_stats.n_reduce_displaced = s.stats.n_reduce_displaced;
        keep_stats.reduce_arena_bytes = s.stats.reduce_arena_bytes;
    }
    s.stats = keep_stats;
    s.stats.n_candidates = (i64)s.total;
    s.stats.key_bits = c->key_bits;
    s.stats.index_bits = s.lowbits;
    if (!s.caps_valid) { s.len = 0; s.n_reg = s.n_irr = s.n_non = 0; } // (else: constants of the context, kept for sizing the launches)
    s.slots = 0;
    s.cols = s.reg = s.irr = s.non = nullptr;
    ev_record(c, s, EV_S1_BEGIN);
    if (s.total == 0) {
        ev_record(c, s, EV_S1_BITMAP); ev_record(c, s, EV_S1_ENUM); ev_record(c, s, EV_S1_SORTBEG);
        ev_record(c, s, EV_S1_HIST); ev_record(c, s, EV_S1_SORT); ev_record(c, s, EV_S1_END);
        s.have_s1 = true;
        s.caps_valid = true;
        return RIPS_OK;
    }
    if (s.cnt_copied && c->stream2 && !c->capturing) CU(cudaStreamWaitEvent(c->stream, s.ev_cnt, 0)); // the previous run's copy of the counters
    if (!c->mode_locked) {
        c->sparse = c->mode == RIPS_MODE_SPARSE || (c->mode == RIPS_MODE_AUTO && c->thr_key != 0 && c->edge_share < 0.05 && c->n >= 64);
        c->mode_locked = true;
    }
    if (c->sparse) return run_stage1_sparse(c, d);
    RC(ensure(c, s.d_cnt, 128)); // 8 u64 counters, then the kernel's tickets
    u64* const d_cnt = (u64*)s.d_cnt.p;
    u32* const d_tick = (u32*)(d_cnt + 8);
    // ---- a4: clearing set of dimension d-1 as a bitmap over the candidate indices
    const u64 words = (s.total + 31) / 32;
    const bool use_bitmap = words * 4 <= (8ull << 30);
    ClearSet cs{nullptr, prev.irr, prev.n_irr, RIPS_PAIR_POS_BITS, (const u64*)prev.red_t.p, prev.n_red};
    if (use_bitmap) {
        RC(ensure(c, s.bitmap, (size_t)words * 4));
        CU(cudaMemsetAsync(s.bitmap.p, 0, (size_t)words * 4, c->stream));
        const u64 pmask = (prev.tbits >= 64) ? ~0ull : ((1ull << prev.tbits) - 1ull);
        ClearLayers L;
        const bool lower = d >= 2;
        L.reg = (lower && prev.reg) ? prev.reg : nullptr;
        L.n_reg = L.reg ? prev.slots : 0;
        L.reg_tbits = prev.tbits;
        L.reg_mask = pmask;
        L.reg_sentinel = (u64)n;
        L.irr = (lower && prev.irr) ? prev.irr : nullptr;
        L.n_irr = L.irr ? (i64)prev.irr_cap : 0;
        L.n_irr_dev = L.irr ? (const u64*)prev.d_cnt.p + S1C_IRREGULAR : nullptr;
        L.irr_shift = RIPS_PAIR_POS_BITS;
        L.red = (const u64*)prev.red_t.p;
        L.n_red = prev.n_red;
        CU(launch_clear_bitmap((u32*)s.bitmap.p, L, c->sms, c->stream));
        c->launches += (L.n_reg > 0 || L.n_irr > 0 || L.n_red > 0);
        cs.bitmap = (const u32*)s.bitmap.p;
    } else if (d >= 2) {
        // no bitmap: the kernel searches the sorted layers, which needs their sizes on the host
        RC(finish_counts(c, d - 1));
        cs.n1 = prev.n_irr;
        if (prev.n_reg > 0) {
            g_last_error = "rips_stage1: candidate space too large for the clearing bitmap";
            return RIPS_ENOMEM;
        }
    }
    ev_record(c, s, EV_S1_BITMAP);

    // ---- a3-a5 + a7: the fused kernel
    // mode: without a threshold at least (n-d-1)/n of the candidates survive (only clearing drops
    // any), so every candidate keeps its slot; with one, estimate the surviving share from the share
    // q of admissible edges (q^(edges of the simplex)) and compact when most are dropped
    const double q = c->edge_share;
    const double est_survival = std::pow(q, (double)(s.M * (s.M - 1) / 2));
    s.compact = (c->thr_key != 0 && est_survival < 0.5) ? 1 : 0;
    int chunk = stage1_chunk(s.total, s.compact, est_survival, s.chunk_retry, c->sms);
    i64 tiles = (i64)((s.total + (u64)chunk - 1) / (u64)chunk);
    Stage1Params p;
    p.Kf = c->d_Kf;
    p.pitch = c->kf_pitch;
    p.Sf = c->d_Sf;
    p.spitch = c->sf_pitch;
    p.bt = c->bt();
    p.n = (int)n;
    p.total = s.total;
    p.tiles = tiles;
    p.chunk = chunk;
    p.stage_cap = stage1_stage_cap();
    p.thr_key = c->thr_key;
    p.sentinel_key = c->n_distinct;
    p.vbits = c->vbits;
    p.lowbits = s.lowbits;
    p.tbits = s.tbits;
    p.clear = cs;
    p.compact = s.compact;
    p.count_only = 0;
    p.fast_visits = 16; // swept at cfg 2 (4..32): flat above 12
    p.cols_out = p.pairs_out = p.irr_out = p.non_out = nullptr;
    p.irr_cap = p.non_cap = 0;
    p.status = nullptr;
    p.ticket = d_tick;
    p.counters = d_cnt;
    p.fh_cols.hist = p.fh_pairs.hist = nullptr;
    p.fh_cols.npasses = p.fh_pairs.npasses = 0;

    u64 cap = s.total; // slots of the two record arrays
    if (s.compact) {
        if (s.exact_kept >= 0) cap = (u64)s.exact_kept; // the count is a constant of the context
        else { // first run of this dimension: count, then size the arrays exactly
            CU(cudaMemsetAsync(d_cnt, 0, 128, c->stream));
            p.count_only = 1;
            CU(launch_stage1(s.M, c->kf_u16, p, c->stream));
            c->launches += 1;
            p.count_only = 0;
            CU(cudaMemcpyAsync(c->h_counters, d_cnt, 64, cudaMemcpyDeviceToHost, c->stream));
            CU(cudaStreamSynchronize(c->stream));
            cap = c->h_counters[S1C_KEPT];
            s.exact_kept = (i64)cap;
        }
        RC(ensure(c, s.s1_status, (size_t)tiles * 8));
        p.status = (u64*)s.s1_status.p;
    }
    s.slots = (i64)cap;
    RC(ensure(c, s.colsA, (size_t)cap * 8));
    RC(ensure(c, s.colsB, (size_t)cap * 8));
    RC(ensure(c, s.pairsA, (size_t)cap * 8));
    p.cols_out = (u64*)s.colsA.p;
    p.pairs_out = (u64*)s.pairsA.p;
    // digit histograms of the two sorts are accumulated by the kernel itself
    SortPlan plan = sort_make_plan(s.lowbits, s.lowbits + c->key_bits);
    s.pair_plan = sort_make_plan(s.tbits, s.tbits + pvbits);
    RC(ensure(c, c->sort_scratch, sort_scratch_bytes((i64)cap, plan)));
    RC(ensure(c, s.pair_scratch, sort_scratch_bytes((i64)cap, s.pair_plan)));
    const bool fused = plan.npasses <= 3;           // S1_MAX_FUSED digits
    s.pair_fused = s.pair_plan.npasses <= 2;        // S1_MAX_FUSED_P digits
    // the two small lists: provisioned for (d+1)/n of the columns to hold the top vertices (those pairs are irregular)
    // and as many non-apparent ones; finish_counts repeats the run with the exact sizes if one overflows
    s.irr_cap = std::max<u64>(s.irr_cap, std::max<u64>(4096, cap / 8));
    s.non_cap = std::max<u64>(s.non_cap, std::max<u64>(4096, cap / 8));
    RC(ensure(c, s.irrA, (size_t)s.irr_cap * 8));
    RC(ensure(c, s.nonA, (size_t)s.non_cap * 8));
    p.irr_out = (u64*)s.irrA.p;
    p.non_out = (u64*)s.nonA.p;
    p.irr_cap = s.irr_cap;
    p.non_cap = s.non_cap;
    CU(cudaMemsetAsync(d_cnt, 0, 128, c->stream));
    if (s.compact) CU(cudaMemsetAsync(s.s1_status.p, 0, (size_t)tiles * 8, c->stream));
    if (fused) {
        CU(sort_prepare_fused(c->sort_scratch.p, (i64)cap, plan, c->stream));
        p.fh_cols.hist = sort_hist_ptr(c->sort_scratch.p);
        p.fh_cols.npasses = plan.npasses;
        for (int r = 0; r < plan.npasses; ++r) { p.fh_cols.shift[r] = plan.shift[r]; p.fh_cols.bits[r] = plan.bits[r]; }
    }
    if (s.pair_fused) {
        CU(sort_prepare_fused(s.pair_scratch.p, (i64)cap, s.pair_plan, c->stream));
        p.fh_pairs.hist = sort_hist_ptr(s.pair_scratch.p);
        p.fh_pairs.npasses = s.pair_plan.npasses;
        for (int r = 0; r < s.pair_plan.npasses; ++r) {
            p.fh_pairs.shift[r] = s.pair_plan.shift[r];
            p.fh_pairs.bits[r] = s.pair_plan.bits[r];
        }
    }
    CU(launch_stage1(s.M, c->kf_u16, p, c->stream));
    c->launches += 1;
    ev_record(c, s, EV_S1_ENUM);
    // the counters follow the kernel to the host on the second stream (nobody waits for them here)
    {
        cudaStream_t sc = c->stream2 ? c->stream2 : c->stream;
        if (sc != c->stream) {
            CU(cudaEventRecord(c->ev_fused, c->stream));
            CU(cudaStreamWaitEvent(sc, c->ev_fused, 0));
        }
        CU(cudaMemcpyAsync(s.h_cnt, d_cnt, 64, cudaMemcpyDeviceToHost, sc));
        if (c->capturing) CU(cudaEventRecordWithFlags(s.ev_cnt, sc, cudaEventRecordExternal));
        else CU(cudaEventRecord(s.ev_cnt, sc));
        s.counts_pending = true;
        s.cnt_copied = true;
    }
    // ---- a6: sort by key (diameter descending); stable, so cidx stays ascending inside equal keys, and the
    // sentinels of the dropped candidates (largest key) end up behind the len columns
    {
        SortTimes st;
        st.enabled = true;
        st.external = c->capturing;
        st.ev[0] = s.ev[EV_S1_SORTBEG]; st.ev[1] = s.ev[EV_S1_HIST]; st.ev[2] = s.ev[EV_S1_SORT];
        s.ev_rec[EV_S1_SORTBEG] = s.ev_rec[EV_S1_HIST] = s.ev_rec[EV_S1_SORT] = true;
        u64* res = nullptr;
        CU(sort_u64((u64*)s.colsA.p, (u64*)s.colsB.p, (i64)cap, plan, c->sort_scratch.p, c->stream, &res, &st, &c->launches, fused,
                    s.M == 2 ? 0xffu : 0u)); // the keys of edges differ inside a warp, those of neighbouring triangles mostly do not
        s.cols = res;
        ev_record(c, s, EV_S1_END);
    }
    s.stats.n_slots = s.slots;
    s.stats.sort_passes = s.slots > 1 ? plan.npasses : 0;
    s.have_s1 = true;
    s.pairs_fresh = true;
    if (!s.caps_valid) RC(finish_counts(c, d)); // first run of this dimension: make sure the lists fitted
    return RIPS_OK;
}

// ------------------------------------------------------------------------------------------ stage 2
int run_stage2(rips_ctx* c, int d)
{
    if (d < 1 || d > c->dim_max + 1) return RIPS_EINVAL;
    DimState& s = c->dims[d];
    if (!s.have_s1) { g_last_error = "rips_stage2: rips_stage1 has not run for this dimension"; return RIPS_EINVAL; }
    if (s.have_s2 && !s.pairs_fresh) return RIPS_OK; // nothing new to partition: the pair store is current
    s.have_s2 = false;
    invalidate_views(s, false, true, true, true);
    if (s.total == 0) { s.have_s2 = true; s.pairs_fresh = false; return RIPS_OK; }
    // The pair partition follows the filtration sort on the main stream (two HBM-bound kernels gain nothing from
    // sharing the memory system; measured: 0.755 ms overlapped against 0.78 ms one after the other at config 2).  The
    // sorts of the two small lists are short chains of small passes, bound by launch latency: they run beside all
    // that, on the second and third stream, right behind the fused kernel.  Their sizes stay on the device (the fused
    // kernel's counters); once a run of this dimension has been checked they are constants of the context and the
    // launches are sized by them, before that by the capacities.
    cudaStream_t st2 = c->stream2 ? c->stream2 : c->stream;
    cudaStream_t st3 = (c->stream3 && st2 != c->stream) ? c->stream3 : st2;
    const u64* d_cnt = (const u64*)s.d_cnt.p;
    const i64 irr_n = s.caps_valid ? std::max<i64>(s.n_irr, 1) : (i64)s.irr_cap;
    const i64 non_n = s.caps_valid ? std::max<i64>(s.n_non, 1) : (i64)s.non_cap;
    ev_record(c, s, EV_S2_BEGIN, st2);
    if (st3 != st2) { // the third stream starts behind the fused kernel as well
        CU(cudaEventRecord(c->ev_join3, st2));
        CU(cudaStreamWaitEvent(st3, c->ev_join3, 0));
    }
    // ---- a9: stable partition of the pair slots by the cofacet vertex v: the regular pairs come out
    // ascending by cidx(t), the sentinels (v = n) behind them
    {
        s.stats.pair_sort_passes = s.slots > 1 ? s.pair_plan.npasses : 0;
        RC(ensure(c, s.pairsB, (size_t)s.slots * 8));
        SortTimes st;
        st.enabled = true;
        st.external = c->capturing;
        st.ev[0] = s.ev[EV_S2_SORTBEG]; st.ev[1] = s.ev[EV_S2_HIST]; st.ev[2] = s.ev[EV_S2_SORT];
        s.ev_rec[EV_S2_SORTBEG] = s.ev_rec[EV_S2_HIST] = s.ev_rec[EV_S2_SORT] = true;
        u64* res = nullptr;
        CU(sort_u64((u64*)s.pairsA.p, (u64*)s.pairsB.p, s.slots, s.pair_plan, s.pair_scratch.p, c->stream, &res, &st,
                    &c->launches, s.pair_fused, 0u)); // cofacet vertices: a few values per warp
        s.reg = res;
    }
    // ---- a8: the two small out-of-order lists: irregular pairs by cidx(t), non-apparent columns by
    // (key, vertices), which is the coboundary order
    {
        SortPlan pi = sort_make_plan(RIPS_PAIR_POS_BITS, RIPS_PAIR_POS_BITS + s.tbits);
        RC(ensure(c, s.irrB, (size_t)s.irr_cap * 8));
        RC(ensure(c, c->sort_scratch2, sort_scratch_bytes((i64)s.irr_cap, pi)));
        u64* res = nullptr;
        CU(sort_u64((u64*)s.irrA.p, (u64*)s.irrB.p, irr_n, pi, c->sort_scratch2.p, st2, &res, nullptr, &c->launches, false, 0u,
                    d_cnt + S1C_IRREGULAR));
        s.irr = res;
        SortPlan pn = sort_make_plan(0, s.lowbits + c->key_bits);
        RC(ensure(c, s.nonB, (size_t)s.non_cap * 8));
        RC(ensure(c, c->sort_scratch3, sort_scratch_bytes((i64)s.non_cap, pn)));
        CU(sort_u64((u64*)s.nonA.p, (u64*)s.nonB.p, non_n, pn, c->sort_scratch3.p, st3, &res, nullptr, &c->launches, false, 0u,
                    d_cnt + S1C_NONAPP));
        if (st3 != st2) { // join the third stream into the second
            CU(cudaEventRecord(c->ev_join3, st3));
            CU(cudaStreamWaitEvent(st2, c->ev_join3, 0));
        }
        s.non = res;
    }
    ev_record(c, s, EV_S2_APP, st2);
    if (st2 != c->stream) { // join: whatever follows on the main stream sees stage 2's results
        CU(cudaEventRecord(c->ev_join, st2));
        CU(cudaStreamWaitEvent(c->stream, c->ev_join, 0));
    }
    ev_record(c, s, EV_S2_END);
    s.pairs_fresh = false;
    s.have_s2 = true;
    return RIPS_OK;
}

// ------------------------------------------------------------------------------------------ reduction (not hot path)
int run_reduce(rips_ctx* c, int d)
{
    if (d < 1 || d > c->dim_max + 1) return RIPS_EINVAL;
    DimState& s = c->dims[d];
    if (!s.have_s2) { g_last_error = "rips_reduce: rips_stage2 has not run for this dimension"; return RIPS_EINVAL; }
    RC(finish_counts(c, d));
    s.have_red = false;
    invalidate_views(s, false, false, false, true);
    s.bars.clear();
    s.tim.reduce_host_ms = s.tim.reduce_xfer_ms = s.tim.reduce_device_ms = 0.f;
    i64 n_piv = 0, n_ess = 0, n_adds = 0;
    if (s.n_non > 0) {
        const double t0 = now_ms();
        const i64 nn = s.n_non;
        const int jbits = bits_for((u64)(nn - 1));
        if (s.tbits + jbits > 64 || c->key_bits + s.tbits > 63) {
            g_last_error = "rips_reduce: (key, row) entries or (row, column) records do not fit 64 bits";
            return RIPS_EOVERFLOW;
        }
        u32 ht_cap = 1024;
        while ((u64)ht_cap < 2ull * (u64)nn) ht_cap <<= 1;
        const int sort_cap = reduce_sort_cap((int)c->n);
        if (reduce_smem_bytes(sort_cap) > 200u * 1024u) {
            g_last_error = "rips_reduce: more points than a CTA can sort the coboundary of in shared memory (n <= 16384)";
            return RIPS_EOVERFLOW;
        }
        const int workers = reduce_workers(c->sms, sort_cap);
        RC(ensure(c, s.rd_piv, (size_t)nn * 8));
        RC(ensure(c, s.rd_colref, (size_t)nn * 8));
        RC(ensure(c, s.rd_todo, (size_t)nn));
        RC(ensure(c, s.rd_htk, (size_t)ht_cap * 8));
        RC(ensure(c, s.rd_htv, (size_t)ht_cap * 4));
        RC(ensure(c, s.rd_cnt, (size_t)(RDC_COUNT + 1) * 8));
        RC(ensure(c, s.rd_rec, (size_t)nn * 8));
        RC(ensure(c, s.rd_rec2, (size_t)nn * 8));
        RC(ensure(c, s.rd_bars, (size_t)nn * 8));
        // what follows the reduction is reserved before the arena is sized (the arena may take all that is left)
        RC(ensure(c, s.red_t, (size_t)nn * 8));
        RC(ensure(c, s.red_s, (size_t)nn * 8));
        RC(ensure(c, c->sort_scratch2, sort_scratch_bytes(nn, sort_make_plan(jbits, jbits + s.tbits))));
        // the arena holds every reduced column and the working buffers; how much the columns fill in depends on
        // the input, so a run that exhausts it is repeated with a larger one
        // (library-owned workspace: a further chunk; caller's workspace: RIPS_ENOMEM with the size the next attempt
        // would have asked for).  First attempt: the largest free block of the workspace, at most 64 bytes per slot.
        size_t arena_bytes = s.arena_hint; // (what the last reduction of this dimension used, plus a quarter)
        if (!arena_bytes) {
            const size_t want = std::max<size_t>((size_t)256 << 20, (size_t)s.slots * 64);
            const size_t have = c->pool.largest_free();
            arena_bytes = std::min(want, have);
            if (arena_bytes < ((size_t)16 << 20)) arena_bytes = want;
        }
        ReduceParams p;
        for (int attempt = 0;; ++attempt) {
            // what the arena can be at most: after giving back the one it has, the largest free block of the workspace,
            // or (library-owned workspace) a new chunk of 90 % of the device memory still free
            size_t limit = ~(size_t)0;
            if (arena_bytes > s.rd_arena.cap) {
                release(c, s.rd_arena);
                limit = c->pool.largest_free();
                if (c->pool.may_grow) {
                    size_t free_b = 0, total_b = 0;
                    cudaMemGetInfo(&free_b, &total_b);
                    limit = std::max(limit, (size_t)((double)free_b * 0.9) & ~(size_t)255);
                }
                if (arena_bytes > limit && limit >= ((size_t)16 << 20)) arena_bytes = limit;
            }
            RC(ensure(c, s.rd_arena, arena_bytes));
            p.cols = s.non;
            p.ncols = nn;
            p.Kf = c->d_Kf;
            p.pitch = c->kf_pitch;
            p.n = (int)c->n;
            p.bt = c->bt();
            p.vbits = c->vbits;
            p.tbits = s.tbits;
            p.thr_key = c->thr_key;
            p.layers = layers_of(s);
            p.piv = (u64*)s.rd_piv.p;
            p.colref = (u64*)s.rd_colref.p;
            p.todo = (unsigned char*)s.rd_todo.p;
            p.ht_keys = (u64*)s.rd_htk.p;
            p.ht_vals = (u32*)s.rd_htv.p;
            p.ht_mask = ht_cap - 1;
            p.arena = (u64*)s.rd_arena.p;
            p.arena_cap = (u64)(s.rd_arena.cap / 8);
            p.sort_cap = sort_cap;
            p.workers = workers;
            p.counters = (u64*)s.rd_cnt.p;
            p.error = (u32*)((u64*)s.rd_cnt.p + RDC_COUNT);
            CU(cudaMemsetAsync(s.rd_cnt.p, 0, (size_t)(RDC_COUNT + 1) * 8, c->stream));
            CU(cudaMemsetAsync(s.rd_colref.p, 0, (size_t)nn * 8, c->stream));
            CU(cudaMemsetAsync(s.rd_htk.p, 0xff, (size_t)ht_cap * 8, c->stream));
            CU(cudaMemsetAsync(s.rd_htv.p, 0xff, (size_t)ht_cap * 4, c->stream));
            CU(launch_reduce(s.M, c->kf_u16, p, c->sms, c->stream));
            c->launches += 4;
            CU(cudaMemcpyAsync(c->h_counters, s.rd_cnt.p, (size_t)(RDC_COUNT + 1) * 8, cudaMemcpyDeviceToHost, c->stream));
            CU(cudaStreamSynchronize(c->stream));
            const u32 err = (u32)c->h_counters[RDC_COUNT];
            if (!err) break;
            if ((err & RD_ERR_ARENA) && attempt < 4 && arena_bytes < limit) { arena_bytes *= 8; continue; }
            if (err & RD_ERR_ARENA) {
                g_last_error = "rips_reduce: the reduced columns do not fit the device memory left (" + std::to_string(arena_bytes) + " bytes of arena)";
                return RIPS_ENOMEM;
            }
            g_last_error = (err & RD_ERR_SORTCAP) ? "rips_reduce: a coboundary exceeds the CTA's sort capacity"
                                                  : "rips_reduce: internal error " + std::to_string(err) + " at column " + std::to_string(c->h_counters[RDC_DBG]) +
                                                        " length " + std::to_string(c->h_counters[RDC_DBG + 1]) + " pivot " + std::to_string(c->h_counters[RDC_DBG + 2]) +
                                                        " work item " + std::to_string(c->h_counters[RDC_DBG + 3]);
            return RIPS_ECUDA;
        }
#ifdef RIPS_REDUCE_PROFILE
        fprintf(stderr, "reduce d=%d: cycles summed over CTAs: peek %llu apparent %llu coboundary+sort %llu add %llu other-add %llu; flushes %llu merge tiles %llu\n", d,
                (unsigned long long)c->h_counters[RDC_DBG], (unsigned long long)c->h_counters[RDC_DBG + 1], (unsigned long long)c->h_counters[RDC_DBG + 2],
                (unsigned long long)c->h_counters[RDC_DBG + 3], (unsigned long long)c->h_counters[RDC_DBG + 4],
                (unsigned long long)(c->h_counters[RDC_DBG + 5] >> 40), (unsigned long long)(c->h_counters[RDC_DBG + 5] & ((1ull << 40) - 1)));
#endif
        n_adds = (i64)c->h_counters[RDC_ADDS];
        s.stats.n_reduce_serial = (i64)c->h_counters[RDC_TODO];
        s.stats.n_reduce_displaced = (i64)c->h_counters[RDC_STEALS];
        s.stats.reduce_arena_bytes = (i64)c->h_counters[RDC_ARENA_TOP] * 8;
        s.arena_hint = std::max<size_t>((size_t)16 << 20, ((size_t)s.stats.reduce_arena_bytes + (size_t)s.stats.reduce_arena_bytes / 4 + 255) & ~(size_t)255);
        // ---- second layer of the pair store as sorted arrays (t ascending), and the bars in column order
        CU(launch_pivot_records(p, jbits, (u64*)s.rd_rec.p, c->stream));
        SortPlan plan = sort_make_plan(jbits, jbits + s.tbits);
        RC(ensure(c, c->sort_scratch2, sort_scratch_bytes(nn, plan)));
        u64* sorted = nullptr;
        CU(sort_u64((u64*)s.rd_rec.p, (u64*)s.rd_rec2.p, nn, plan, c->sort_scratch2.p, c->stream, &sorted, nullptr, &c->launches));
        CU(launch_bars(p, s.lowbits, c->d_values, (float*)s.rd_bars.p, p.counters + RDC_NBARS, p.counters + RDC_NESS, c->stream));
        c->launches += 2;
        CU(cudaMemcpyAsync(c->h_counters, s.rd_cnt.p, (size_t)RDC_COUNT * 8, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        n_piv = (i64)c->h_counters[RDC_PIVOTS];
        n_ess = (i64)c->h_counters[RDC_NESS];
        const i64 n_bars = (i64)c->h_counters[RDC_NBARS];
        RC(ensure(c, s.red_t, (size_t)n_piv * 8));
        RC(ensure(c, s.red_s, (size_t)n_piv * 8));
        CU(launch_pivot_arrays(s.M, p, jbits, sorted, n_piv, (u64*)s.red_t.p, (u64*)s.red_s.p, c->stream));
        c->launches += n_piv > 0;
        const double t1 = now_ms();
        s.bars.resize((size_t)n_bars * 2);
        if (n_bars) CU(cudaMemcpyAsync(s.bars.data(), s.rd_bars.p, (size_t)n_bars * 8, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        const double t2 = now_ms();
        s.tim.reduce_device_ms = (float)(t1 - t0);
        s.tim.reduce_xfer_ms = (float)(t2 - t1);
        release(c, s.rd_arena); // scratch of the reduction only: the next dimension may need the room
    } else {
        RC(ensure(c, s.red_t, 16));
        RC(ensure(c, s.red_s, 16));
    }
    s.n_red = n_piv;
    s.stats.n_reduced_pivots = n_piv;
    s.stats.n_essential = n_ess;
    s.stats.n_additions = n_adds;
    s.stats.n_bars = (i64)s.bars.size() / 2;
    s.have_red = true;
    return RIPS_OK;
}

int check_dim(rips_ctx* c, int d, int lo)
{
    if (!c) return RIPS_EINVAL;
    if (d < lo || d > c->dim_max + 1) return RIPS_EINVAL;
    return RIPS_OK;
}

void free_dim(rips_ctx* c, DimState& s)
{
    DevBuf* all[] = {&s.colsA, &s.colsB, &s.s1_status, &s.bitmap, &s.pairsA, &s.pairsB, &s.irrA, &s.irrB, &s.nonA, &s.nonB,
                     &s.pair_scratch, &s.d_cnt, &s.simpA, &s.simpB, &s.rd_piv, &s.rd_colref, &s.rd_todo, &s.rd_htk, &s.rd_htv, &s.rd_arena, &s.rd_cnt,
                     &s.rd_rec, &s.rd_rec2, &s.rd_bars, &s.red_t,
                     &s.red_s, &s.v_fdiam, &s.v_fcidx, &s.v_at, &s.v_as, &s.v_ndiam, &s.v_ncidx, &s.v_pt, &s.v_ps};
    for (DevBuf* b : all) release(c, *b);
    if (s.ev_made) for (int i = 0; i < EV_COUNT; ++i) cudaEventDestroy(s.ev[i]);
    s.ev_made = false;
    if (s.graph) { cudaGraphExecDestroy(s.graph); s.graph = nullptr; }
}

int init_device_tables(rips_ctx* c, const float* dist_lower)
{
    const i64 E = c->E, n = c->n;
    RC(ensure(c, c->b_counters, 256));
    RC(ensure(c, c->b_tickets, 32));
    c->d_counters = (u64*)c->b_counters.p;
    c->d_tickets = (u32*)c->b_tickets.p;
    CU(cudaMallocHost(&c->h_counters, 256));
    RC(ensure(c, c->b_binom, c->h_binom.size() * 8));
    c->d_binom = (u64*)c->b_binom.p;
    CU(cudaMemcpyAsync(c->d_binom, c->h_binom.data(), c->h_binom.size() * 8, cudaMemcpyHostToDevice, c->stream));
    const size_t eb = (size_t)(E ? E : 1);
    RC(ensure(c, c->b_dist, eb * 4));
    RC(ensure(c, c->b_edges, eb * 8));
    RC(ensure(c, c->b_K, eb * 4));
    RC(ensure(c, c->b_values, eb * 4));
    c->d_dist = (float*)c->b_dist.p;
    c->d_edges = (u64*)c->b_edges.p;
    c->d_K = (u32*)c->b_K.p;
    c->d_values = (float*)c->b_values.p;
    c->n_distinct = 0;
    if (E > 0) {
        CU(cudaMemcpyAsync(c->d_dist, dist_lower, (size_t)E * 4, cudaMemcpyDefault, c->stream));
        RC(ensure(c, c->b_init_tmp, (size_t)E * 8));
        CU(cudaMemsetAsync(c->d_counters, 0, 64, c->stream));
        CU(cudaMemsetAsync(c->d_tickets, 0, 32, c->stream));
        CU(launch_prep_edges(c->d_dist, E, c->d_edges, (int*)(c->d_counters + 1), c->threshold, c->d_counters + 2, c->stream));
        SortPlan plan = sort_make_plan(32, 64);
        RC(ensure(c, c->sort_scratch, sort_scratch_bytes(E, plan)));
        u64* res = nullptr;
        CU(sort_u64(c->d_edges, (u64*)c->b_init_tmp.p, E, plan, c->sort_scratch.p, c->stream, &res, nullptr, &c->launches, false,
                    0x7u)); // fp32 bits: the mantissa bytes differ inside a warp, the exponent byte does not
        if (res != c->d_edges) { std::swap(c->b_edges, c->b_init_tmp); c->d_edges = (u64*)c->b_edges.p; }
        RC(ensure(c, c->b_init_status, (size_t)rank_edges_tiles(E) * 8));
        CU(cudaMemsetAsync(c->b_init_status.p, 0, (size_t)rank_edges_tiles(E) * 8, c->stream));
        CU(launch_rank_edges(c->d_edges, E, c->d_K, c->d_values, (u64*)c->b_init_status.p, c->d_tickets, c->d_counters, c->stream));
        c->launches += 2;
        CU(cudaMemcpyAsync(c->h_counters, c->d_counters, 24, cudaMemcpyDeviceToHost, c->stream));
        CU(cudaStreamSynchronize(c->stream));
        c->edge_share = E ? (double)(E - (i64)c->h_counters[2]) / (double)E : 1.0;
        // keys are ranks in descending value order: thr_key = number of distinct values above the threshold, and
        // prep_edges_kernel made ONE value (+inf) of all of them -- so the table of values stays on the device
        // (800 MB at n = 20000, which the host never needs)
        c->thr_key = c->h_counters[2] != 0 ? 1u : 0u;
        release(c, c->b_init_tmp);
        release(c, c->b_init_status);
        if ((int)c->h_counters[1] != 0) {
            g_last_error = "rips_init: the distance matrix holds a NaN, negative or infinite entry";
            return RIPS_EINVAL;
        }
        c->n_distinct = (u32)c->h_counters[0];
        c->kf_u16 = c->n_distinct <= 65535u; // entries are key+1 <= n_distinct
    }
    {
        // row pitch: an odd number of 32-bit words, so the rows of consecutive vertices start in
        // different shared-memory banks (lanes of the fused kernel read column v of rows x, x+1, ...)
        int pitch = (int)n;
        if (c->kf_u16) { while ((pitch & 3) != 2) ++pitch; }
        else if ((pitch & 1) == 0) ++pitch;
        c->kf_pitch = pitch;
        const size_t kf_bytes = (((size_t)n * (size_t)pitch * (c->kf_u16 ? 2 : 4)) + 15) & ~(size_t)15;
        RC(ensure(c, c->b_Kf, kf_bytes));
        c->d_Kf = c->b_Kf.p;
        CU(cudaMemsetAsync(c->d_Kf, 0, kf_bytes, c->stream));
        CU(launch_build_full_keys(c->d_K, (int)n, pitch, c->d_Kf, c->kf_u16, c->stream));
        c->launches += 1;
        if (n >= SUMMARY_MIN_N) {
            c->sf_pitch = (int)((n + 31) / 32);
            RC(ensure(c, c->b_Sf, (size_t)n * (size_t)c->sf_pitch * (c->kf_u16 ? 2 : 4)));
            c->d_Sf = c->b_Sf.p;
            CU(launch_build_block_max(c->d_Kf, (int)n, pitch, c->d_Sf, c->sf_pitch, c->kf_u16, c->stream));
            c->launches += 1;
        }
        c->vbits = bits_for((u64)(n - 1));
    }
    c->key_bits = bits_for(c->n_distinct); // the value n_distinct itself is the key of the column sentinel
    return RIPS_OK;
}

// Device bytes rips_init holds for n points (distances, edge records and their sort buffer, keys, values, the full
// key matrix as u32, binomial table, counters, the edge sort's scratch): an upper bound.
size_t setup_bytes(i64 n, int kmax)
{
    const size_t E = (size_t)(n * (n - 1) / 2) + 1;
    SortPlan plan = sort_make_plan(32, 64);
    return E * (4 + 8 + 8 + 4 + 4) + (size_t)n * (size_t)(n + 4) * 4 + (n >= SUMMARY_MIN_N ? (size_t)n * (size_t)(n / 32 + 2) * 4 : 0) +
           (size_t)(kmax + 1) * (size_t)(n + 1) * 8 + sort_scratch_bytes((i64)E, plan) +
           (E / 2048 + 1) * 8 + (size_t)n * 20 + (1 << 16);
}

// Device bytes one dimension with `cand` candidates can hold when a share `keep` of them survives the threshold:
// column records and pair slots with their ping-pong buffers (4 x 8), the irregular-pair and non-apparent lists with
// theirs (4 lists of max(4096, slots / 8) records), the clearing bitmap over ALL candidates, the look-back words of
// three sorts (2048 bytes per tile of 5120 records) and their heads, the views the accessors materialise (filtration
// 12, apparent pairs 16, pivots 16, non-apparent columns 12 / 8 bytes per column), the reduction's per-column words
// (at most slots / 8 non-apparent columns) and its default arena.
long double dim_bytes(long double cand, long double keep)
{
    const long double slots = std::max<long double>(4096.0L, cand * keep);
    const long double lists = std::max<long double>(4096.0L, slots / 8);
    return slots * 32 + lists * 8 * 4 + cand / 8 + 64 + 8 * ((slots / 5120 + 2) * 2048) + 16 * ((lists / 5120 + 2) * 2048) + 5 * (1 << 15) +
           slots * (12 + 16 + 16) + lists * 12 +
           lists * 96 + std::max<long double>((long double)(256u << 20), slots * 64);
}

} // namespace

// =============================================================================================== C ABI
extern "C" {

const char* rips_strerror(int code)
{
    switch (code) {
    case RIPS_OK: return "ok";
    case RIPS_EINVAL: return "invalid argument";
    case RIPS_EOVERFLOW: return "sizes overflow the 64-bit packed records";
    case RIPS_ENOMEM: return "out of memory";
    case RIPS_ECUDA: return "CUDA error";
    default: return "unknown error";
    }
}

const char* rips_last_error(void) { return g_last_error.c_str(); }

int rips_workspace_bytes(int64_t n, int dim_max, int64_t* bytes)
{
    g_last_error.clear();
    if (!bytes || n < 1 || dim_max < 0 || dim_max > 4) return RIPS_EINVAL;
    if (n > 46340) return RIPS_EOVERFLOW;
    std::vector<u64> b;
    build_binom(n, dim_max + 3, b);
    if (b[(size_t)(dim_max + 2) * (n + 1) + n] >> 62) return RIPS_EOVERFLOW;
    long double total = (long double)setup_bytes(n, dim_max + 3);
    for (int d = 1; d <= dim_max; ++d) total += dim_bytes((long double)b[(size_t)(d + 1) * (n + 1) + n], 1.0L);
    total += total / 64 + (16 << 20); // granules of 256 bytes, holes left by lists that had to grow
    if (total > 9.0e18L) return RIPS_EOVERFLOW;
    *bytes = (int64_t)total;
    return RIPS_OK;
}

int64_t rips_last_required_bytes(void) { return g_required_bytes; }

int rips_init(rips_ctx** out, const float* dist_lower, int64_t n, int dim_max, float threshold, void* workspace_dev,
              int64_t workspace_bytes, void* stream)
{
    g_last_error.clear();
    g_required_bytes = 0;
    if (!out) return RIPS_EINVAL;
    *out = nullptr;
    if (n < 1 || dim_max < 0 || dim_max > 4 || std::isnan(threshold)) return RIPS_EINVAL;
    if (n > 46340) return RIPS_EOVERFLOW; // the kernels index the n x n key matrix with 32-bit integers
    if (n > 1 && !dist_lower) return RIPS_EINVAL;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        g_last_error = "no usable CUDA device: this library has no CPU fallback";
        return RIPS_ECUDA;
    }
    rips_ctx* c = new (std::nothrow) rips_ctx();
    if (!c) return RIPS_ENOMEM;
    c->n = n;
    c->E = n * (n - 1) / 2;
    c->dim_max = dim_max;
    c->threshold = threshold;
    c->stream = (cudaStream_t)stream;
    c->kmax = dim_max + 3;
    {
        int dev = 0;
        if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev);
        if (c->sms < 1) c->sms = 1;
    }
    if (cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); c->cap_stream = nullptr; }
    if (cudaStreamCreateWithFlags(&c->stream2, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); c->stream2 = nullptr; }
    if (cudaStreamCreateWithFlags(&c->stream3, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); c->stream3 = nullptr; }
    if (cudaEventCreateWithFlags(&c->ev_join3, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); c->ev_join3 = nullptr; c->stream3 = nullptr; }
    if (cudaEventCreateWithFlags(&c->ev_fused, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); c->ev_fused = nullptr; c->stream2 = nullptr; }
    if (cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); c->ev_join = nullptr; c->stream2 = nullptr; }
    build_binom(n, c->kmax, c->h_binom);
    if (hbinom(c, n, dim_max + 2) >> 62) { delete c; return RIPS_EOVERFLOW; }
    c->dims.resize((size_t)dim_max + 2);
    if (cudaMallocHost(&c->h_dimcnt, c->dims.size() * 64) != cudaSuccess) { cudaGetLastError(); delete c; return RIPS_ENOMEM; }
    memset(c->h_dimcnt, 0, c->dims.size() * 64);
    for (size_t i = 0; i < c->dims.size(); ++i) {
        c->dims[i].h_cnt = c->h_dimcnt + 8 * i;
        if (cudaEventCreateWithFlags(&c->dims[i].ev_cnt, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); c->dims[i].ev_cnt = nullptr; }
    }
    int r = RIPS_OK;
    if (workspace_dev) {
        if (workspace_bytes < 4096 || ((uintptr_t)workspace_dev & 255)) {
            g_last_error = "rips_init: the workspace must be 256-byte aligned and at least 4096 bytes";
            delete c;
            return RIPS_EINVAL;
        }
        c->pool.add_chunk(workspace_dev, (size_t)workspace_bytes, false);
    } else {
        // the library's own workspace: first what the set-up needs (known from n), the rest once the threshold's
        // share of admissible edges is known
        void* base = nullptr;
        const size_t sb = Pool::round(setup_bytes(n, c->kmax));
        cudaError_t e2 = cudaMalloc(&base, sb);
        if (e2 != cudaSuccess) { cudaGetLastError(); g_last_error = "rips_init: cudaMalloc of the set-up workspace failed"; delete c; return RIPS_ENOMEM; }
        c->pool.add_chunk(base, sb, true);
        c->pool.may_grow = true;
    }
    r = init_device_tables(c, dist_lower);
    if (r == RIPS_OK && !workspace_dev) {
        const double q = c->edge_share;
        long double rest = 0;
        for (int d = 1; d <= dim_max; ++d) {
            const double surv = std::pow(q, (double)((d + 1) * d / 2));
            const bool compact = c->thr_key != 0 && surv < 0.5; // the rule of run_stage1
            rest += dim_bytes((long double)hbinom(c, n, d + 1), compact ? std::min(1.0, 2.0 * surv) : 1.0);
        }
        rest += rest / 64 + (16 << 20);
        size_t free_b = 0, total_b = 0;
        cudaMemGetInfo(&free_b, &total_b);
        if (rest > (long double)free_b * 0.9L) rest = (long double)free_b * 0.9L;
        void* base = nullptr;
        if (cudaMalloc(&base, (size_t)rest) == cudaSuccess) c->pool.add_chunk(base, (size_t)rest, true);
        else cudaGetLastError(); // chunks are added as the computation asks for them
    }
    if (r == RIPS_OK) {
        // the widest record of the requested dimensions must fit 64 bits
        int lb = (dim_max + 1) * c->vbits;
        int tb = bits_for(hbinom(c, n, dim_max + 2));
        // (the reduction's entries, key and row index in one word, are checked by rips_reduce: stage 1 and stage 2 do not need them)
        if ((dim_max >= 1 && c->key_bits + lb > 64) || bits_for((u64)n) + tb > 64)
            r = RIPS_EOVERFLOW;
    }
    if (r != RIPS_OK) { rips_free(c); return r; }
    *out = c;
    return RIPS_OK;
}

void rips_free(rips_ctx* c)
{
    if (!c) return;
    if (c->stream3) { cudaStreamSynchronize(c->stream3); cudaStreamDestroy(c->stream3); }
    if (c->ev_join3) cudaEventDestroy(c->ev_join3);
    if (c->stream2) { cudaStreamSynchronize(c->stream2); cudaStreamDestroy(c->stream2); }
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    for (DimState& s : c->dims) free_dim(c, s);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->ev_fused) cudaEventDestroy(c->ev_fused);
    release(c, c->sort_scratch);
    release(c, c->sort_scratch2);
    release(c, c->sort_scratch3);
    release(c, c->d0_pairs);
    release(c, c->d0_death);
    release(c, c->d0_uf);
    if (c->stream) cudaStreamSynchronize(c->stream);
    else cudaDeviceSynchronize();
    for (Pool::Chunk& ch : c->pool.chunks)
        if (ch.owned) cudaFree(ch.base);
    if (c->h_counters) cudaFreeHost(c->h_counters);
    if (c->h_dimcnt) cudaFreeHost(c->h_dimcnt);
    for (DimState& s : c->dims) if (s.ev_cnt) cudaEventDestroy(s.ev_cnt);
    cudaGetLastError();
    delete c;
}

int rips_dim0(rips_ctx* c) { return c ? run_dim0(c) : RIPS_EINVAL; }

int rips_set_mode(rips_ctx* c, int mode)
{
    if (!c || mode < RIPS_MODE_AUTO || mode > RIPS_MODE_SPARSE) return RIPS_EINVAL;
    if (c->mode_locked) { g_last_error = "rips_set_mode: a stage 1 has already run on this context"; return RIPS_EINVAL; }
    c->mode = mode;
    return RIPS_OK;
}
// Stage 1 + stage 2 of a dimension whose sizes are known to fit are one CUDA graph: ~45 kernels, memsets and copies on
// three streams whose launch parameters no longer change (the counts they depend on are read on the device).  The
// graph is captured by the first rips_stage1 call that finds the dimension in that state and replayed by the later
// ones (it covers stage 2 as well, so the rips_stage2 that follows finds its work done); a change of any buffer it
// uses (a list that had to grow, other pivots of the previous dimension) makes a new capture.
static u64 graph_signature(rips_ctx* c, int d)
{
    const DimState& s = c->dims[d];
    const DimState& q = c->dims[d - 1];
    const void* ptrs[] = {s.colsA.p, s.colsB.p, s.pairsA.p, s.pairsB.p, s.irrA.p, s.irrB.p, s.nonA.p, s.nonB.p, s.bitmap.p, s.s1_status.p,
                          s.pair_scratch.p, s.d_cnt.p, c->sort_scratch.p, c->sort_scratch2.p, c->sort_scratch3.p, q.reg, q.irr, q.red_t.p,
                          q.d_cnt.p, c->d_Kf};
    u64 h = 1469598103934665603ull;
    auto mix = [&](u64 x) { h = (h ^ x) * 1099511628211ull; };
    for (const void* p : ptrs) mix((u64)(uintptr_t)p);
    mix((u64)q.n_red); mix((u64)q.slots); mix(q.irr_cap); mix(s.irr_cap); mix(s.non_cap); mix((u64)s.n_irr); mix((u64)s.n_non);
    mix((u64)s.exact_kept); mix((u64)s.chunk_retry);
    return h;
}

static int run_stage12_graph(rips_ctx* c, int d)
{
    DimState& s = c->dims[d];
    const u64 sig = graph_signature(c, d);
    if (s.graph && s.graph_sig == sig) {
        CU(cudaGraphLaunch(s.graph, c->stream));
        c->launches += s.graph_launches;
        s.have_s1 = s.have_s2 = true;
        s.pairs_fresh = false;
        s.counts_pending = true;
        invalidate_views(s, true, true, true, true);
        return RIPS_OK;
    }
    if (s.graph) { cudaGraphExecDestroy(s.graph); s.graph = nullptr; }
    const i64 l0 = c->launches;
    if (!c->cap_stream || cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
        cudaGetLastError();
        c->use_graphs = false;
        return run_stage1(c, d);
    }
    cudaStream_t callers = c->stream;
    c->stream = c->cap_stream;
    c->capturing = true;
    int r = run_stage1(c, d);
    if (r == RIPS_OK) r = run_stage2(c, d);
    c->capturing = false;
    c->stream = callers;
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(c->cap_stream, &g);
    if (r == RIPS_OK && e == cudaSuccess && g) {
        cudaGraphExec_t ex = nullptr;
        e = cudaGraphInstantiate(&ex, g, 0);
        cudaGraphDestroy(g);
        if (e == cudaSuccess) {
            s.graph = ex;
            s.graph_sig = graph_signature(c, d);
            s.graph_launches = c->launches - l0;
            CU(cudaGraphLaunch(s.graph, c->stream));
            return RIPS_OK;
        }
    } else if (g)
        cudaGraphDestroy(g);
    // the capture did not work out: this context runs its stages launch by launch from now on
    cudaGetLastError();
    c->use_graphs = false;
    c->launches = l0;
    s.have_s1 = s.have_s2 = false;
    s.counts_pending = false;
    RC(run_stage1(c, d));
    return RIPS_OK;
}

int rips_stage1(rips_ctx* c, int d)
{
    RC(check_dim(c, d, 1));
    DimState& s = c->dims[d];
    if (c->use_graphs && c->stream2 && c->stream3 && s.caps_valid && c->dims[d - 1].caps_valid && c->dims[d - 1].have_red &&
        c->dims[d - 1].have_s2 && hbinom(c, c->n, d + 1) > 0)
        return run_stage12_graph(c, d);
    return run_stage1(c, d);
}
int rips_stage2(rips_ctx* c, int d) { RC(check_dim(c, d, 1)); return run_stage2(c, d); }
int rips_reduce(rips_ctx* c, int d) { RC(check_dim(c, d, 1)); return run_reduce(c, d); }

int rips_import_pivots(rips_ctx* c, int d, const uint64_t* t_host, const uint64_t* s_host, int64_t count)
{
    RC(check_dim(c, d, 1));
    if (count < 0 || (count > 0 && (!t_host || !s_host))) return RIPS_EINVAL;
    DimState& s = c->dims[d];
    if (!s.have_s2) { g_last_error = "rips_import_pivots: rips_stage2 has not run for this dimension"; return RIPS_EINVAL; }
    RC(finish_counts(c, d));
    for (int64_t i = 1; i < count; ++i)
        if (t_host[i] <= t_host[i - 1]) return RIPS_EINVAL;
    s.have_red = false;
    invalidate_views(s, false, false, false, true);
    RC(ensure(c, s.red_t, (size_t)count * 8));
    RC(ensure(c, s.red_s, (size_t)count * 8));
    if (count) {
        CU(cudaMemcpyAsync(s.red_t.p, t_host, (size_t)count * 8, cudaMemcpyHostToDevice, c->stream));
        CU(cudaMemcpyAsync(s.red_s.p, s_host, (size_t)count * 8, cudaMemcpyHostToDevice, c->stream));
        CU(cudaStreamSynchronize(c->stream));
    }
    s.n_red = count;
    s.bars.clear();
    s.stats.n_reduced_pivots = count;
    s.stats.n_essential = 0;
    s.stats.n_additions = 0;
    s.stats.n_bars = 0;
    s.have_red = true;
    return RIPS_OK;
}

int rips_compute(rips_ctx* c)
{
    if (!c) return RIPS_EINVAL;
    RC(run_dim0(c));
    for (int d = 1; d <= c->dim_max; ++d) {
        RC(run_stage1(c, d));
        RC(run_stage2(c, d));
        RC(run_reduce(c, d));
    }
    return RIPS_OK;
}

int rips_barcodes(rips_ctx* c, int d, const float** birth_death_host, int64_t* count)
{
    if (!c || !birth_death_host || !count || d < 0 || d > c->dim_max + 1) return RIPS_EINVAL;
    DimState& s = c->dims[d];
    if (!s.have_red || !s.have_s2) return RIPS_EINVAL;
    *birth_death_host = s.bars.data();
    *count = (int64_t)s.bars.size() / 2;
    return RIPS_OK;
}

int rips_filtration(rips_ctx* c, int d, const float** diam_dev, const uint64_t** cidx_dev, int64_t* len)
{
    RC(check_dim(c, d, 1));
    if (!diam_dev || !cidx_dev || !len) return RIPS_EINVAL;
    DimState& s = c->dims[d];
    if (!s.have_s1) return RIPS_EINVAL;
    RC(finish_counts(c, d));
    if (!s.has_vf) {
        RC(ensure(c, s.v_fdiam, (size_t)s.len * 4));
        RC(ensure(c, s.v_fcidx, (size_t)s.len * 8));
        CU(launch_unpack_columns(s.M, s.cols, s.len, c->vbits, c->bt(), c->d_values, (float*)s.v_fdiam.p, (u64*)s.v_fcidx.p, c->stream));
        c->launches += s.len > 0;
        CU(cudaStreamSynchronize(c->stream));
        s.has_vf = true;
    }
    *diam_dev = (const float*)s.v_fdiam.p;
    *cidx_dev = (const u64*)s.v_fcidx.p;
    *len = s.len;
    return RIPS_OK;
}

int rips_apparent_pairs(rips_ctx* c, int d, const uint64_t** t_dev, const uint64_t** s_dev, int64_t* n_app)
{
    RC(check_dim(c, d, 1));
    if (!t_dev || !s_dev || !n_app) return RIPS_EINVAL;
    DimState& s = c->dims[d];
    if (!s.have_s2) return RIPS_EINVAL;
    RC(finish_counts(c, d));
    if (!s.has_va) {
        RC(ensure(c, s.v_at, (size_t)(s.n_reg + s.n_irr) * 8));
        RC(ensure(c, s.v_as, (size_t)(s.n_reg + s.n_irr) * 8));
        CU(launch_merge_apparent(s.M, layers_of(s), c->bt(), (int)c->n, (u64*)s.v_at.p, (u64*)s.v_as.p, c->stream));
        c->launches += (s.n_reg + s.n_irr) > 0;
        CU(cudaStreamSynchronize(c->stream));
        s.has_va = true;
    }
    *t_dev = (const u64*)s.v_at.p;
    *s_dev = (const u64*)s.v_as.p;
    *n_app = s.n_reg + s.n_irr;
    return RIPS_OK;
}

int rips_nonapparent(rips_ctx* c, int d, const float** diam_dev, const uint64_t** cidx_dev, int64_t* n_non)
{
    RC(check_dim(c, d, 1));
    if (!diam_dev || !cidx_dev || !n_non) return RIPS_EINVAL;
    DimState& s = c->dims[d];
    if (!s.have_s2) return RIPS_EINVAL;
    RC(finish_counts(c, d));
    if (!s.has_vn) {
        RC(ensure(c, s.v_ndiam, (size_t)s.n_non * 4));
        RC(ensure(c, s.v_ncidx, (size_t)s.n_non * 8));
        CU(launch_unpack_columns(s.M, s.non, s.n_non, c->vbits, c->bt(), c->d_values, (float*)s.v_ndiam.p,
                                 (u64*)s.v_ncidx.p, c->stream));
        c->launches += s.n_non > 0;
        CU(cudaStreamSynchronize(c->stream));
        s.has_vn = true;
    }
    *diam_dev = (const float*)s.v_ndiam.p;
    *cidx_dev = (const u64*)s.v_ncidx.p;
    *n_non = s.n_non;
    return RIPS_OK;
}

int rips_pivots(rips_ctx* c, int d, const uint64_t** t_dev, const uint64_t** s_dev, int64_t* n_piv)
{
    RC(check_dim(c, d, 0));
    if (!t_dev || !s_dev || !n_piv) return RIPS_EINVAL;
    DimState& s = c->dims[d];
    if (!s.have_red || !s.have_s2) return RIPS_EINVAL;
    RC(finish_counts(c, d));
    const i64 na = s.n_reg + s.n_irr, np = na + s.n_red;
    if (!s.has_vp) {
        if (!s.has_va) { // the apparent layers as (t, s) arrays first
            RC(ensure(c, s.v_at, (size_t)na * 8));
            RC(ensure(c, s.v_as, (size_t)na * 8));
            CU(launch_merge_apparent(s.M, layers_of(s), c->bt(), (int)c->n, (u64*)s.v_at.p, (u64*)s.v_as.p, c->stream));
            c->launches += na > 0;
            s.has_va = true;
        }
        RC(ensure(c, s.v_pt, (size_t)np * 8));
        RC(ensure(c, s.v_ps, (size_t)np * 8));
        CU(launch_merge_ts((const u64*)s.v_at.p, (const u64*)s.v_as.p, na, (const u64*)s.red_t.p, (const u64*)s.red_s.p,
                           s.n_red, (u64*)s.v_pt.p, (u64*)s.v_ps.p, c->stream));
        c->launches += np > 0;
        CU(cudaStreamSynchronize(c->stream));
        s.has_vp = true;
    }
    *t_dev = (const u64*)s.v_pt.p;
    *s_dev = (const u64*)s.v_ps.p;
    *n_piv = np;
    return RIPS_OK;
}

int rips_pivot_lookup(rips_ctx* c, int d, const uint64_t* t_query_dev, int64_t m, int64_t* s_out_dev)
{
    RC(check_dim(c, d, 0));
    if (m < 0 || (m > 0 && (!t_query_dev || !s_out_dev))) return RIPS_EINVAL;
    DimState& s = c->dims[d];
    if (!s.have_s2) return RIPS_EINVAL;
    RC(finish_counts(c, d));
    CU(launch_pivot_lookup(s.M, layers_of(s), c->bt(), (int)c->n, (const u64*)s.red_t.p, (const u64*)s.red_s.p,
                           s.have_red ? s.n_red : 0, t_query_dev, m, s_out_dev, c->stream));
    c->launches += m > 0;
    CU(cudaStreamSynchronize(c->stream));
    return RIPS_OK;
}

int rips_stats(rips_ctx* c, int d, rips_stats_t* out)
{
    RC(check_dim(c, d, 0));
    if (!out) return RIPS_EINVAL;
    RC(finish_counts(c, d));
    *out = c->dims[d].stats;
    return RIPS_OK;
}

int rips_timings(rips_ctx* c, int d, rips_timings_t* out)
{
    RC(check_dim(c, d, 0));
    if (!out) return RIPS_EINVAL;
    DimState& s = c->dims[d];
    CU(cudaStreamSynchronize(c->stream));
    rips_timings_t t = s.tim;
    t.clear_bitmap_ms = ev_ms(s, EV_S1_BEGIN, EV_S1_BITMAP);
    t.enumerate_ms = ev_ms(s, EV_S1_BITMAP, EV_S1_ENUM);
    t.sort_hist_ms = ev_ms(s, EV_S1_SORTBEG, EV_S1_HIST);
    t.sort_pass_ms = ev_ms(s, EV_S1_HIST, EV_S1_SORT);
    t.stage1_ms = ev_ms(s, EV_S1_BEGIN, EV_S1_END);
    t.apparent_ms = ev_ms(s, EV_S2_BEGIN, EV_S2_APP);
    t.pair_hist_ms = ev_ms(s, EV_S2_SORTBEG, EV_S2_HIST);
    t.pair_sort_ms = ev_ms(s, EV_S2_HIST, EV_S2_SORT);
    t.stage2_ms = ev_ms(s, EV_S2_BEGIN, EV_S2_END);
    t.dim0_ms = ev_ms(s, EV_D0_BEGIN, EV_D0_END);
    *out = t;
    return RIPS_OK;
}

int rips_device_bytes(rips_ctx* c, int64_t* bytes)
{
    if (!c || !bytes) return RIPS_EINVAL;
    *bytes = (int64_t)c->pool.total();
    return RIPS_OK;
}

int rips_workspace_in_use(rips_ctx* c, int64_t* bytes, int64_t* peak)
{
    if (!c || !bytes) return RIPS_EINVAL;
    *bytes = (int64_t)c->pool.in_use;
    if (peak) *peak = (int64_t)c->pool.peak;
    return RIPS_OK;
}

int rips_kernel_launches(rips_ctx* c, int64_t* launches)
{
    if (!c || !launches) return RIPS_EINVAL;
    *launches = c->launches;
    return RIPS_OK;
}

int rips_sort_u64(uint64_t* keys_dev, uint64_t* tmp_dev, int64_t n, int lo_bit, int hi_bit, void* stream)
{
    g_last_error.clear();
    if (n < 0 || lo_bit < 0 || hi_bit > 64 || lo_bit >= hi_bit || (n > 0 && (!keys_dev || !tmp_dev))) return RIPS_EINVAL;
    if (n <= 1) return RIPS_OK;
    cudaStream_t st = (cudaStream_t)stream;
    SortPlan plan = sort_make_plan(lo_bit, hi_bit);
    void* scratch = nullptr;
    cudaError_t e = cudaMalloc(&scratch, sort_scratch_bytes(n, plan));
    if (e != cudaSuccess) { cudaGetLastError(); return RIPS_ENOMEM; }
    u64* res = nullptr;
    e = sort_u64(keys_dev, tmp_dev, n, plan, scratch, st, &res, nullptr, nullptr);
    if (e == cudaSuccess && res != keys_dev)
        e = cudaMemcpyAsync(keys_dev, res, (size_t)n * 8, cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    cudaFree(scratch);
    if (e != cudaSuccess) return cuda_fail(e, "rips_sort_u64");
    return RIPS_OK;
}

int rips_sort_u64_static(uint64_t* keys_dev, uint64_t* tmp_dev, int64_t n, int lo_bit, int hi_bit, void* stream)
{
    g_last_error.clear();
    if (n < 0 || lo_bit < 0 || hi_bit > 64 || lo_bit >= hi_bit || (n > 0 && (!keys_dev || !tmp_dev))) return RIPS_EINVAL;
    if (n > RIPS_SORT_STATIC_MAX_RECORDS) {
        g_last_error = "rips_sort_u64_static: " + std::to_string(n) + " records exceed the maximum of " +
                       std::to_string((long long)RIPS_SORT_STATIC_MAX_RECORDS) + " the static scratch is sized for (use rips_sort_u64)";
        return RIPS_EINVAL;
    }
    if (n <= 1) return RIPS_OK;
    cudaStream_t st = (cudaStream_t)stream;
    SortPlan plan = sort_make_plan(lo_bit, hi_bit);
    void* scratch = nullptr;
    size_t bytes = 0;
    cudaError_t e = sort_static_scratch(&scratch, &bytes);
    if (e != cudaSuccess) return cuda_fail(e, "rips_sort_u64_static: address of the static scratch");
    if (sort_scratch_bytes(n, plan) > bytes) { // (cannot happen in the product build: the maximum above is what the array holds)
        g_last_error = "rips_sort_u64_static: " + std::to_string(n) + " records need " + std::to_string(sort_scratch_bytes(n, plan)) +
                       " bytes of scratch, the static array holds " + std::to_string(bytes);
        return RIPS_EINVAL;
    }
    u64* res = nullptr;
    e = sort_u64(keys_dev, tmp_dev, n, plan, scratch, st, &res, nullptr, nullptr);
    if (e == cudaSuccess && res != keys_dev)
        e = cudaMemcpyAsync(keys_dev, res, (size_t)n * 8, cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) return cuda_fail(e, "rips_sort_u64_static");
    return RIPS_OK;
}

} // extern "C"
