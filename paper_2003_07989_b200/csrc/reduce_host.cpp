// reduce_host.cpp -- see reduce_host.h.  Implicit cohomology reduction over Z/2 (PAPER.md:127,
// :168-170, :210) of the non-apparent columns the device could not finish on its own (reduce.cu): those
// whose pivot, after reduction against the apparent columns, another non-apparent column owns.  Pair
// store as in PAPER.md:555-561: pivots found here go to a hash map; whether a row belongs to an apparent
// pair is evaluated from Definition 5 (apparent_lookup) instead of searching the device arrays.  Column
// entries are packed (key << tbits) | cidx(t); the pivot of a column is the cofacet that comes first in
// the filtration order (smallest diameter = LARGEST key, then largest cidx), i.e. simply
// the largest packed entry.
#include "reduce_host.h"

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <functional>
#include <memory>
#include <unordered_map>

namespace {

struct Ctx {
    const HostReduceIn& in;
    int M; // vertices of a column simplex
    std::vector<uint32_t> Kfull; // n x n symmetric copy of the keys (diagonal unused): branch-free, row-contiguous reads
    explicit Ctx(const HostReduceIn& i) : in(i), M(i.d + 1), Kfull((size_t)i.n * i.n, 0xffffffffu)
    {
        for (int a = 1; a < in.n; ++a)
            for (int b = 0; b < a; ++b)
                Kfull[(size_t)a * in.n + b] = Kfull[(size_t)b * in.n + a] = in.K[(size_t)a * (a - 1) / 2 + b];
    }
    uint64_t C(int v, int k) const { return in.binom[(size_t)k * in.bstride + v]; }
    uint32_t key(int a, int b) const { return Kfull[(size_t)a * in.n + b]; }
    void decode(uint64_t idx, int m, int* v) const
    { // v[m-1] > ... > v[0]
        int hi = in.n - 1;
        for (int k = m; k >= 1; --k) {
            int lo = k - 1, h = hi;
            while (lo < h) {
                int mid = (lo + h + 1) >> 1;
                if (C(mid, k) <= idx) lo = mid;
                else h = mid - 1;
            }
            v[k - 1] = lo;
            idx -= C(lo, k);
            hi = lo - 1;
        }
    }
    // First-layer lookup: s of the apparent pair whose row is t, or false.  Evaluated directly from
    // the definition (Definition 5) instead of searching the device array, which
    // spares the host a copy of ~C(n-1,d+1) records: s must be the youngest facet of t -- the facet of
    // diameter diam(t) with the smallest index (facets in increasing index = vertices removed in
    // decreasing order, Algorithm 6) -- and t the oldest cofacet of s of that diameter (cofacets in
    // decreasing index = added vertex decreasing, first hit).  An apparent s is a birth simplex, so it
    // is never cleared and (s, t) is in the pair store.
    bool apparent_lookup(uint64_t t, uint64_t* s_out) const
    {
        int tv[17];
        decode(t, M + 1, tv);
        uint32_t key_t = 0xffffffffu;
        for (int a = 1; a <= M; ++a)
            for (int b = 0; b < a; ++b) { uint32_t k = key(tv[a], tv[b]); if (k < key_t) key_t = k; }
        for (int drop = M; drop >= 0; --drop) {
            int s[16], m = 0;
            for (int i = 0; i <= M; ++i) if (i != drop) s[m++] = tv[i];
            uint32_t key_s = 0xffffffffu;
            for (int a = 1; a < M; ++a)
                for (int b = 0; b < a; ++b) { uint32_t k = key(s[a], s[b]); if (k < key_s) key_s = k; }
            if (M == 1) key_s = 0xffffffffu; // a vertex has no edge: never of the diameter of an edge t
            if (key_s != key_t) continue;
            // s is the youngest facet of t; is t the oldest cofacet of s with that diameter?
            for (int v = in.n - 1; v >= 0; --v) {
                bool member = false, ok = true;
                for (int j = 0; j < M; ++j) {
                    if (s[j] == v) { member = true; break; }
                    if (key(v, s[j]) < key_s) { ok = false; break; }
                }
                if (member || !ok) continue;
                if (v != tv[drop]) return false;
                uint64_t r = 0;
                for (int i = 0; i < M; ++i) r += C(s[i], i + 1);
                *s_out = r;
                return true;
            }
            return false;
        }
        return false;
    }
    // push the coboundary of the column simplex s (cofacets with diameter <= threshold)
    template <class Heap>
    uint32_t push_coboundary(Heap& h, uint64_t cidx_s) const
    {
        int s[16];
        decode(cidx_s, M, s);
        uint32_t key_s = 0xffffffffu;
        for (int a = 1; a < M; ++a)
            for (int b = 0; b < a; ++b) { uint32_t k = key(s[a], s[b]); if (k < key_s) key_s = k; }
        uint64_t low[17], high[17]; // low[g] = sum_{i<g} C(s[i], i+1); high[g] = sum_{i>=g} C(s[i], i+2)
        low[0] = 0;
        for (int i = 0; i < M; ++i) low[i + 1] = low[i] + C(s[i], i + 1);
        high[M] = 0;
        for (int i = M - 1; i >= 0; --i) high[i] = high[i + 1] + C(s[i], i + 2);
        const uint32_t* rows[16];
        for (int j = 0; j < M; ++j) rows[j] = Kfull.data() + (size_t)s[j] * in.n;
        for (int seg = M; seg >= 0; --seg) {
            int hi = (seg == M) ? in.n - 1 : s[seg] - 1;
            int lo = (seg == 0) ? 0 : s[seg - 1] + 1;
            const uint64_t* Crow = in.binom + (size_t)(seg + 1) * in.bstride;
            const uint64_t fixed = low[seg] + high[seg];
            for (int v = hi; v >= lo; --v) {
                uint32_t kt = key_s;
                for (int j = 0; j < M; ++j) { uint32_t k = rows[j][v]; if (k < kt) kt = k; }
                if (kt < in.thr_key) continue;
                h.push(((uint64_t)kt << in.tbits) | (fixed + Crow[v]));
            }
        }
        return key_s;
    }
};

// Working column of the reduction: a multiset of packed entries (key << tbits | cidx(t)) with "largest
// first" access.  The pivots of a column come out in (almost always) decreasing order -- whatever an
// addition brings in lies later in the filtration than the pivot it cancels, except for the unreduced
// column of an earlier non-apparent owner -- so instead of one big heap the entries are kept in buckets
// of neighbouring keys: only the bucket at the sweep position is a heap (small, cache-resident), the
// others are plain vectors that are heapified when the sweep reaches them.
class KeyedColumn {
public:
    // one bucket per 64 consecutive keys: few enough vectors to stay in cache while a coboundary is pushed
    KeyedColumn(uint32_t n_keys, int tbits) : tbits_(tbits + 6), buckets_((n_keys >> 6) + 2) {}
    void clear()
    {
        for (uint32_t k : touched_) buckets_[k].clear();
        touched_.clear();
        cur_ = -1;
        max_key_ = 0;
        size_ = 0;
    }
    void push(uint64_t e)
    {
        const int64_t k = (int64_t)(e >> tbits_);
        std::vector<uint64_t>& b = buckets_[(size_t)k];
        if (b.empty()) touched_.push_back((uint32_t)k);
        b.push_back(e);
        ++size_;
        if (k == cur_) std::push_heap(b.begin(), b.end());
        else if (k > cur_) cur_ = -1; // an entry above the sweep position: find the top again at the next access
        if (k > max_key_) max_key_ = k;
    }
    bool empty() { return !settle(); }
    uint64_t top() { settle(); return buckets_[(size_t)cur_].front(); }
    void pop()
    {
        settle();
        std::vector<uint64_t>& b = buckets_[(size_t)cur_];
        std::pop_heap(b.begin(), b.end());
        b.pop_back();
        --size_;
    }
    size_t size() const { return size_; }

private:
    // make cur_ the largest key with a non-empty bucket, its bucket a heap; false if the column is empty
    bool settle()
    {
        if (cur_ >= 0 && !buckets_[(size_t)cur_].empty()) return true;
        if (size_ == 0) return false;
        int64_t k = (cur_ >= 0) ? cur_ : max_key_;
        while (k >= 0 && buckets_[(size_t)k].empty()) --k;
        if (k < 0) { // entries only above the old position (cannot happen when cur_ < 0)
            k = max_key_;
            while (buckets_[(size_t)k].empty()) --k;
        }
        if (cur_ < 0) max_key_ = k;
        cur_ = k;
        std::make_heap(buckets_[(size_t)k].begin(), buckets_[(size_t)k].end());
        return true;
    }
    int tbits_;
    std::vector<std::vector<uint64_t>> buckets_;
    std::vector<uint32_t> touched_;
    int64_t cur_ = -1, max_key_ = 0;
    size_t size_ = 0;
};

template <class Heap>
bool pop_pivot(Heap& h, uint64_t* piv)
{
    while (!h.empty()) {
        uint64_t p = h.top();
        h.pop();
        if (!h.empty() && h.top() == p) { h.pop(); continue; } // equal entries cancel over Z/2
        *piv = p;
        return true;
    }
    return false;
}

} // namespace

// Oblivious column reduction (Algorithm 2) of the columns in coboundary order.  A
// column the device has already reduced against the apparent columns (in.pre) and whose pivot no
// earlier column owns is final at once; the others -- the conflicts between non-apparent columns, a
// fraction of a per cent of the columns at the paper-shaped workloads -- are reduced here (KeyedColumn as
// the working column), adding D_{lookup[low]} whether the pivot's owner is an apparent column or one
// reduced earlier (Lemma 3: same result as adding R_i).
void host_reduce_columns(const HostReduceIn& in, HostReduceOut& out)
{
    Ctx cx(in);
    const uint64_t cmask = (in.cbits >= 64) ? ~0ull : ((1ull << in.cbits) - 1ull);
    const uint64_t tmask = (1ull << in.tbits) - 1ull;
    typedef KeyedColumn Heap;
    std::unordered_map<uint64_t, uint64_t> owner; // second layer: t -> cidx(s) of the column that owns the pivot
    owner.reserve((size_t)in.ncols * 2 + 16);
    auto finalize = [&](int64_t j, uint64_t piv, uint64_t cidx_s, uint32_t key_s) {
        owner.emplace(piv & tmask, cidx_s);
        out.piv_t.push_back(piv & tmask);
        out.piv_s.push_back(cidx_s);
        out.piv_key_t.push_back((uint32_t)(piv >> in.tbits));
        out.piv_key_s.push_back(key_s);
        out.piv_col.push_back(j);
    };
    // Reduction-matrix technique for the rare column on which the oblivious form runs
    // away (it re-adds, pivot by pivot, every column an owner's reduction had added): V_i = the columns
    // whose coboundaries sum to R_i, kept per reduced column, so that adding R_i is one step and the
    // additions cancel in V over Z/2.  V of a column that was reduced obliviously (or on the device) is
    // recomputed on demand by reducing it again this way; a pivot owned by a later column cannot come up
    // while doing so, because the earlier column would have claimed it.
    std::unordered_map<uint64_t, std::vector<uint64_t>> vstore; // cidx(s) of a reduced column -> V (cidx of columns)
    int64_t n_vmode = 0;
    std::function<const std::vector<uint64_t>&(uint64_t, uint64_t*)> reduce_v =
        [&](uint64_t cidx_s, uint64_t* piv_out) -> const std::vector<uint64_t>& {
        Heap h(in.n_keys, in.tbits);
        std::unordered_map<uint64_t, int> par; // column -> parity in V
        auto add_col = [&](uint64_t c) { cx.push_coboundary(h, c); par[c] ^= 1; };
        add_col(cidx_s);
        uint64_t piv = 0;
        bool zero = true;
        for (;;) {
            if (!pop_pivot(h, &piv)) break;
            const uint64_t t = piv & tmask;
            auto it = owner.find(t);
            if (it != owner.end() && it->second == cidx_s) { zero = false; break; } // its own, already known pivot
            uint64_t s2 = 0;
            if (it != owner.end()) {
                const uint64_t own = it->second;
                auto vs = vstore.find(own);
                h.push(piv);
                if (vs == vstore.end()) {
                    uint64_t dummy;
                    const std::vector<uint64_t>& v = reduce_v(own, &dummy);
                    std::vector<uint64_t> copy(v); // reduce_v may rehash vstore
                    for (uint64_t c : copy) add_col(c);
                } else {
                    std::vector<uint64_t> copy(vs->second);
                    for (uint64_t c : copy) add_col(c);
                }
                ++out.additions;
                continue;
            }
            if (cx.apparent_lookup(t, &s2)) { h.push(piv); add_col(s2); ++out.additions; continue; }
            zero = false;
            break; // a new pivot
        }
        if (piv_out) *piv_out = zero ? ~0ull : piv;
        std::vector<uint64_t> v;
        for (auto& kv : par) if (kv.second) v.push_back(kv.first);
        return vstore[cidx_s] = std::move(v);
    };
    // Stored reduced columns (the standard form, Algorithm 1; Lemma 3) for
    // inputs on which restarts keep coming -- flag complexes of random graphs, many equal diameters: the
    // reduced columns fill in, and both the oblivious form and the V technique re-derive them through
    // coboundaries again and again.  Once `stored_after` columns have been restarted, every further column
    // that needs reducing keeps its reduced column R_j (packed entries, first = pivot) and a pivot whose
    // owner has a stored column costs one pass over that column.  R of an owner finalised before the
    // switch (or at once, from the device pre-reduction) is computed when first asked for, by reducing it
    // again against the store -- a pivot of a later column cannot come up, as above.
    const int64_t stored_after = 16;
    const int stored_max_depth = 512; // nesting of on-demand recomputations; deeper owners are added as D_i (Algorithm 2)
    std::unordered_map<uint64_t, std::vector<uint64_t>> rstore; // cidx(s) -> R_s
    std::vector<std::unique_ptr<Heap>> heaps;                   // one working column per nesting level
    int64_t n_stored = 0;
    std::function<uint64_t(uint64_t, int)> reduce_r = [&](uint64_t cidx_s, int depth) -> uint64_t {
        if ((size_t)depth >= heaps.size()) heaps.emplace_back(new Heap(in.n_keys, in.tbits));
        Heap& w = *heaps[(size_t)depth];
        w.clear();
        cx.push_coboundary(w, cidx_s);
        for (;;) {
            uint64_t piv;
            if (!pop_pivot(w, &piv)) return ~0ull; // a zero column is never an owner: nothing to keep
            const uint64_t t = piv & tmask;
            auto it = owner.find(t);
            if (it == owner.end() || it->second != cidx_s) {
                if (it != owner.end()) {
                    const uint64_t own = it->second;
                    auto rs = rstore.find(own);
                    if (rs == rstore.end() && depth < stored_max_depth) {
                        reduce_r(own, depth + 1);
                        rs = rstore.find(own);
                    }
                    w.push(piv); // the added column holds t as well: the two cancel
                    if (rs != rstore.end()) for (uint64_t e : rs->second) w.push(e);
                    else cx.push_coboundary(w, own);
                    ++out.additions;
                    continue;
                }
                uint64_t s2 = 0;
                if (cx.apparent_lookup(t, &s2)) { w.push(piv); cx.push_coboundary(w, s2); ++out.additions; continue; }
            }
            // a new pivot, or the one this column is already known to own: keep the reduced column
            std::vector<uint64_t> r;
            r.push_back(piv);
            uint64_t e;
            while (pop_pivot(w, &e)) r.push_back(e);
            rstore[cidx_s] = std::move(r);
            ++n_stored;
            return piv;
        }
    };
    const int64_t oblivious_budget = 256; // additions before a column is restarted with the V technique
    int64_t n_fast = 0, n_slow = 0, n_def = 0, n_own_adds = 0;
    Heap h(in.n_keys, in.tbits);
    for (int64_t j = 0; j < in.ncols; ++j) {
        const uint64_t cidx_s = in.cols[j] & cmask;
        const uint32_t key_s = (uint32_t)(in.cols[j] >> in.cbits);
        if (in.pre && in.pre[j] == ~0ull) ++n_def;
        if (in.pre && in.pre[j] != ~0ull) {
            if (in.pre[j] == 0) {
                out.ess_s.push_back(cidx_s);
                out.ess_key.push_back(key_s);
                out.ess_col.push_back(j);
                continue;
            }
            const uint64_t piv = in.pre[j] - 1;
            ++out.lookups;
            if (owner.find(piv & tmask) == owner.end()) { finalize(j, piv, cidx_s, key_s); ++n_fast; continue; }
        }
        ++n_slow;
        if (n_vmode >= stored_after) {
            const uint64_t pv = reduce_r(cidx_s, 0);
            if (pv == ~0ull) {
                out.ess_s.push_back(cidx_s);
                out.ess_key.push_back(key_s);
                out.ess_col.push_back(j);
            } else
                finalize(j, pv, cidx_s, key_s);
            continue;
        }
        const int64_t adds0 = out.additions;
        h.clear();
        cx.push_coboundary(h, cidx_s);
        for (;;) {
            uint64_t piv;
            if (!pop_pivot(h, &piv)) {
                out.ess_s.push_back(cidx_s);
                out.ess_key.push_back(key_s);
                out.ess_col.push_back(j);
                break;
            }
            const uint64_t t = piv & tmask;
            uint64_t s2 = 0;
            bool hit = false;
            ++out.lookups;
            auto it = owner.find(t);
            if (it != owner.end()) { hit = true; s2 = it->second; }
            else hit = cx.apparent_lookup(t, &s2);
            if (!hit) { finalize(j, piv, cidx_s, key_s); break; }
            if (it != owner.end()) ++n_own_adds;
            if (out.additions - adds0 >= oblivious_budget) { // runaway: start over with the V technique
                out.additions = adds0;
                ++n_vmode;
                uint64_t pv = 0;
                reduce_v(cidx_s, &pv);
                if (pv == ~0ull) {
                    out.ess_s.push_back(cidx_s);
                    out.ess_key.push_back(key_s);
                    out.ess_col.push_back(j);
                } else
                    finalize(j, pv, cidx_s, key_s);
                break;
            }
            h.push(piv); // the column of s2 contains t as well: the two cancel
            cx.push_coboundary(h, s2);
            ++out.additions;
        }
    }
    if (getenv("RIPS_DEBUG"))
        fprintf(stderr, "host_reduce d=%d: cols %lld final at once %lld reduced here %lld (not pre-reduced %lld), additions of reduced columns %lld, restarted with V %lld, reduced columns stored %lld\n", in.d,
                (long long)in.ncols, (long long)n_fast, (long long)n_slow, (long long)n_def, (long long)n_own_adds, (long long)n_vmode, (long long)n_stored);
}
