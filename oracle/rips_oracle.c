/* ORACLE tiers O2 and O3 -- plain C, written from PAPER.md.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * load this.  It shares no code, header, table or constant generator with the CUDA path under
 * paper_2003_07989_b200/csrc, and neither side includes the other.
 *
 * What it computes (every array below is uniquely determined by the input):
 *   oracle_stage1  Filtration construction with clearing, Algorithms 7-8:
 *                  every candidate d-simplex by combinatorial index (Eq. 2), its
 *                  diameter (Eq. 1), keep iff diam <= threshold and the simplex is
 *                  not the death simplex of a pair of dimension d-1 (clearing, PAPER.md:146-154,
 *                  reading R2 of DESIGN.md), sort by diameter descending, cidx ascending
 *                  (PAPER.md:607-608).
 *   oracle_stage2  Algorithm 3 literally, per column: scan cofacets in
 *                  decreasing cidx (vertex v = n-1 .. 0, reading R4), stop at the first with
 *                  diam(t) == diam(s) (the oldest cofacet, Lemma 7), list the
 *                  facets of t by removing vertices in decreasing order (Algorithm 6,
 *                  PAPER.md:443-469, increasing cidx), stop at the first with diam == diam(s);
 *                  apparent iff that facet is s (reading R3).
 *   oracle_dim0    H_0 by union-find over edges in filtration order.
 *   oracle_reduce  Implicit cohomology reduction of coboundary columns over Z/2, columns = cofacets
 *                  with diam <= threshold: the standard reduction R_j <- R_j + R_i of Algorithm 1
 *                  (PAPER.md:99-121), which Lemma 3 proves equivalent to the oblivious
 *                  Algorithm 2; the reduced columns are kept because the oblivious
 *                  form, which re-adds D_i, needs orders of magnitude more additions on "difficult"
 *                  inputs such as config 3's random matrices.
 *   oracle_reduce_explicit  the same reduction as Algorithm 1 verbatim on the explicit
 *                  coboundary matrix (rows ranked in reverse filtration order, working column a bit
 *                  array, R_j <- R_j + R_i an exclusive or): same pairs; used where the heap of
 *                  oracle_reduce is too slow (config 3, dimension 1).
 *
 * No blocking, fusion or reordering beyond what those passages state.  The only concession to
 * run time is `#pragma omp parallel for` over independent simplices (Corollary 8)
 * and a binary heap for the working column of oracle_reduce.
 *
 * Pinned by tests/test_oracle_*.py against oracle/brute.py (definitions only), the paper's
 * worked examples and closed forms (tests/golden/).  Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef uint64_t u64;
typedef int64_t i64;

#define MAXV 16 /* max vertices of a simplex handled (dimension <= 15) */

/* ------------------------------------------------------------------ binomials, Eq. 2 */

typedef struct {
    int n, K;
    u64 *c; /* c[v*(K+1)+k] = C(v,k), saturating at UINT64_MAX */
} binom_t;

static u64 sat_add(u64 a, u64 b) { return (a > UINT64_MAX - b) ? UINT64_MAX : a + b; }

static void binom_init(binom_t *b, int n, int K)
{
    b->n = n;
    b->K = K;
    b->c = (u64 *)calloc((size_t)(n + 1) * (K + 1), sizeof(u64));
    for (int v = 0; v <= n; ++v) {
        b->c[(size_t)v * (K + 1)] = 1;
        for (int k = 1; k <= K && k <= v; ++k) /* Pascal's rule */
            b->c[(size_t)v * (K + 1) + k] =
                sat_add(b->c[(size_t)(v - 1) * (K + 1) + k - 1], (k <= v - 1) ? b->c[(size_t)(v - 1) * (K + 1) + k] : 0);
    }
}
static void binom_free(binom_t *b) { free(b->c); }
static u64 C(const binom_t *b, int v, int k)
{
    if (k < 0 || v < 0 || k > v) return 0;
    return b->c[(size_t)v * (b->K + 1) + k];
}

u64 oracle_binomial(int n, int k)
{
    binom_t b;
    if (k < 0 || n < 0 || k > n) return 0;
    binom_init(&b, n, k);
    u64 r = C(&b, n, k);
    binom_free(&b);
    return r;
}

/* distance between two points; dist_lower holds (i>j) at i(i-1)/2+j */
static float dist(const float *D, int i, int j)
{
    if (i == j) return 0.0f;
    if (i < j) { int t = i; i = j; j = t; }
    return D[(size_t)i * (i - 1) / 2 + j];
}

/* Eq. 2, simplex -> index.  verts decreasing: verts[0] > verts[1] > ... > verts[m-1]. */
static u64 encode(const binom_t *b, const int *verts, int m)
{
    u64 idx = 0;
    for (int p = 0; p < m; ++p) idx += C(b, verts[p], m - p); /* v_k with k = m-1-p gets C(v_k, k+1) */
    return idx;
}

/* Eq. 2, index -> simplex: for k = m..1 the largest v with C(v,k) <= rest.  verts decreasing. */
static void decode(const binom_t *b, u64 idx, int m, int n, int *verts)
{
    int v = n - 1;
    for (int k = m; k >= 1; --k) {
        while (C(b, v, k) > idx) --v;
        verts[m - k] = v;
        idx -= C(b, v, k);
        --v;
    }
}

/* Eq. 1 */
static float diameter(const float *D, const int *verts, int m)
{
    float dm = 0.0f;
    for (int a = 0; a < m; ++a)
        for (int c = a + 1; c < m; ++c) {
            float x = dist(D, verts[a], verts[c]);
            if (x > dm) dm = x;
        }
    return dm;
}

/* ------------------------------------------------------------------ exported helpers */

void oracle_free(void *p) { free(p); }

/* bench.py's cpu_baseline times the same sample at all cores and at one thread */
void oracle_set_threads(int t)
{
#ifdef _OPENMP
    if (t >= 1) omp_set_num_threads(t);
#else
    (void)t;
#endif
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* decode / encode / diameter exposed so the tests can pin them one by one */
void oracle_decode(u64 idx, int m, int n, int *verts)
{
    binom_t b;
    binom_init(&b, n, m);
    decode(&b, idx, m, n, verts);
    binom_free(&b);
}
u64 oracle_encode(const int *verts_decreasing, int m, int n)
{
    binom_t b;
    binom_init(&b, n, m);
    u64 r = encode(&b, verts_decreasing, m);
    binom_free(&b);
    return r;
}
float oracle_diameter(const float *D, u64 idx, int m, int n)
{
    int verts[MAXV];
    binom_t b;
    binom_init(&b, n, m);
    decode(&b, idx, m, n, verts);
    binom_free(&b);
    return diameter(D, verts, m);
}

/* ------------------------------------------------------------------ stage 1 (Algorithms 7-8) */

typedef struct { float diam; u64 cidx; } col_t;

static int cmp_coboundary_order(const void *pa, const void *pb)
{   /* decreasing diameters, increasing combinatorial indices */
    const col_t *a = (const col_t *)pa, *b = (const col_t *)pb;
    if (a->diam > b->diam) return -1;
    if (a->diam < b->diam) return 1;
    if (a->cidx < b->cidx) return -1;
    if (a->cidx > b->cidx) return 1;
    return 0;
}

static int is_member(const u64 *sorted, i64 n, u64 x)
{
    i64 lo = 0, hi = n;
    while (lo < hi) {
        i64 mid = lo + (hi - lo) / 2;
        if (sorted[mid] < x) lo = mid + 1; else hi = mid;
    }
    return lo < n && sorted[lo] == x;
}

/* Candidates idx in [idx_lo, idx_hi) (pass 0, C(n,d+1) for all of them).  cleared: ascending cidx of
 * the death simplices of dimension d-1 (the keys t of P_{d-1}).  do_sort = 0 leaves the survivors in
 * increasing cidx.  Outputs are malloc'ed; free with oracle_free.  counts[0..2] = kept, removed by
 * diameter, cleared (a simplex over the threshold counts as removed by diameter).  Returns 0. */
int oracle_stage1(const float *D, int n, int d, float threshold, const u64 *cleared, i64 n_cleared,
                  u64 idx_lo, u64 idx_hi, int do_sort, float **out_diam, u64 **out_cidx, i64 *out_len,
                  i64 *counts)
{
    int m = d + 1;
    binom_t b;
    binom_init(&b, n, m);
    u64 total = idx_hi - idx_lo;
    float *dm = (float *)malloc(sizeof(float) * (total ? total : 1));
    unsigned char *flag = (unsigned char *)malloc(total ? total : 1); /* flagarray of Alg. 7 */
#pragma omp parallel for schedule(static)
    for (i64 i = 0; i < (i64)total; ++i) {
        int verts[MAXV];
        u64 idx = idx_lo + (u64)i;           /* cidx(s) <- tid */
        decode(&b, idx, m, n, verts);
        float x = diameter(D, verts, m);
        dm[i] = x;
        if (!(x <= threshold)) flag[i] = 2;  /* removed by diameter */
        else if (is_member(cleared, n_cleared, idx)) flag[i] = 1; /* cleared */
        else flag[i] = 0;
    }
    i64 kept = 0, over = 0, clr = 0;
    for (u64 i = 0; i < total; ++i) { kept += flag[i] == 0; over += flag[i] == 2; clr += flag[i] == 1; }
    col_t *cols = (col_t *)malloc(sizeof(col_t) * (kept ? kept : 1));
    i64 w = 0;
    for (u64 i = 0; i < total; ++i)
        if (flag[i] == 0) { cols[w].diam = dm[i]; cols[w].cidx = idx_lo + i; ++w; }
    free(dm);
    free(flag);
    if (do_sort) qsort(cols, (size_t)kept, sizeof(col_t), cmp_coboundary_order);
    float *od = (float *)malloc(sizeof(float) * (kept ? kept : 1));
    u64 *oc = (u64 *)malloc(sizeof(u64) * (kept ? kept : 1));
    for (i64 i = 0; i < kept; ++i) { od[i] = cols[i].diam; oc[i] = cols[i].cidx; }
    free(cols);
    binom_free(&b);
    *out_diam = od; *out_cidx = oc; *out_len = kept;
    if (counts) { counts[0] = kept; counts[1] = over; counts[2] = clr; }
    return 0;
}

/* ------------------------------------------------------------------ stage 2 (Algorithm 3) */

/* One column.  Returns 1 and *t_out = cidx(t) if (s,t) is an apparent pair, else 0.
 * *visited (optional) = number of cofacets whose diameter was evaluated. */
static int apparent_column(const float *D, const binom_t *b, int n, int d, float diam_s, u64 cidx_s,
                           u64 *t_out, int *visited)
{
    int m = d + 1;
    int V[MAXV], T[MAXV + 1], F[MAXV];
    decode(b, cidx_s, m, n, V);                       /* line 2: V <- vertices(s) */
    int seen = 0;
    for (int v = n - 1; v >= 0; --v) {                /* line 3: cofacets, lexicographically decreasing */
        int in_s = 0;
        for (int p = 0; p < m; ++p) in_s |= (V[p] == v);
        if (in_s) continue;
        float dt = diam_s;                            /* line 4: diam(t) <- max(dist(v',v), diam(s)) */
        for (int p = 0; p < m; ++p) { float x = dist(D, V[p], v); if (x > dt) dt = x; }
        ++seen;
        if (dt == diam_s) {                           /* line 5: t is the oldest cofacet of s */
            int q = 0, placed = 0;                    /* vertices of t, decreasing */
            for (int p = 0; p < m; ++p) {
                if (!placed && v > V[p]) { T[q++] = v; placed = 1; }
                T[q++] = V[p];
            }
            if (!placed) T[q++] = v;
            u64 cidx_t = encode(b, T, m + 1);
            /* lines 6-8: facets of t by removing vertices in decreasing order = increasing cidx (Alg. 6) */
            int result = 0;
            for (int r = 0; r <= m; ++r) {
                int f = 0;
                for (int p = 0; p <= m; ++p) if (p != r) F[f++] = T[p];
                float df = diameter(D, F, m);
                if (df == diam_s) {                   /* line 9 */
                    result = (encode(b, F, m) == cidx_s); /* line 10: s is the youngest facet of t */
                    break;                            /* line 13: exit either way */
                }
            }
            if (visited) *visited = seen;
            *t_out = cidx_t;
            return result;                            /* the outer loop never resumes (reading R3) */
        }
    }
    if (visited) *visited = seen;
    return 0;
}

/* Columns (diam[i], cidx[i]), i < len, in any order (the result per column does not depend on it).
 * flag[i] = 1 iff apparent; t[i] = cidx of the oldest cofacet when apparent, else UINT64_MAX.
 * visits (optional, may be NULL) = cofacets evaluated per column. */
int oracle_stage2(const float *D, int n, int d, const float *diam, const u64 *cidx, i64 len,
                  unsigned char *flag, u64 *t, int *visits)
{
    binom_t b;
    binom_init(&b, n, d + 2);
#pragma omp parallel for schedule(dynamic, 1024)
    for (i64 i = 0; i < len; ++i) {
        u64 tt = UINT64_MAX;
        int seen = 0;
        int a = apparent_column(D, &b, n, d, diam[i], cidx[i], &tt, &seen);
        flag[i] = (unsigned char)a;
        t[i] = a ? tt : UINT64_MAX;
        if (visits) visits[i] = seen;
    }
    binom_free(&b);
    return 0;
}

/* ------------------------------------------------------------------ dimension 0 */

typedef struct { float diam; u64 cidx; int a, b; } edge_t;

static int cmp_filtration_order_edges(const void *pa, const void *pb)
{   /* increasing diameter, then decreasing combinatorial index */
    const edge_t *x = (const edge_t *)pa, *y = (const edge_t *)pb;
    if (x->diam < y->diam) return -1;
    if (x->diam > y->diam) return 1;
    if (x->cidx > y->cidx) return -1;
    if (x->cidx < y->cidx) return 1;
    return 0;
}

static int uf_find(int *parent, int x)
{
    while (parent[x] != x) { parent[x] = parent[parent[x]]; x = parent[x]; }
    return x;
}

/* Union-find over the edges with diam <= threshold in filtration order.  Every edge that merges two
 * components is the death simplex of an H_0 class; the class that dies is the younger one, i.e. the
 * component whose first vertex in the filtration order comes later.  Vertices all have diameter 0 and
 * are ordered by decreasing index, so a component is born with its LARGEST vertex and
 * the dying component is the one with the smaller largest-vertex.
 * Outputs (malloc'ed, ascending by edge cidx): pair_t = cidx of the merging edge, pair_s = the vertex
 * that gave birth to the dying class, pair_death = diameter of the edge.  n_components = classes that
 * never die.  */
int oracle_dim0(const float *D, int n, float threshold, u64 **pair_t, u64 **pair_s, float **pair_death,
                i64 *n_pairs, i64 *n_components)
{
    size_t E = (size_t)n * (n - 1) / 2;
    edge_t *edges = (edge_t *)malloc(sizeof(edge_t) * (E ? E : 1));
    size_t ne = 0;
    for (int i = 1; i < n; ++i)
        for (int j = 0; j < i; ++j) {
            float x = dist(D, i, j);
            if (x <= threshold) {
                edges[ne].diam = x; edges[ne].cidx = (u64)i * (i - 1) / 2 + j; edges[ne].a = i; edges[ne].b = j;
                ++ne;
            }
        }
    qsort(edges, ne, sizeof(edge_t), cmp_filtration_order_edges);
    int *parent = (int *)malloc(sizeof(int) * (n ? n : 1));
    int *oldest = (int *)malloc(sizeof(int) * (n ? n : 1));
    for (int i = 0; i < n; ++i) { parent[i] = i; oldest[i] = i; }
    col_t *tmp = (col_t *)malloc(sizeof(col_t) * (n ? n : 1));
    u64 *ss = (u64 *)malloc(sizeof(u64) * (n ? n : 1));
    i64 np = 0;
    for (size_t e = 0; e < ne; ++e) {
        int ra = uf_find(parent, edges[e].a), rb = uf_find(parent, edges[e].b);
        if (ra == rb) continue;
        int dying = (oldest[ra] < oldest[rb]) ? ra : rb;
        int living = (dying == ra) ? rb : ra;
        tmp[np].diam = edges[e].diam; tmp[np].cidx = edges[e].cidx; ss[np] = (u64)oldest[dying];
        ++np;
        parent[dying] = living;
    }
    /* ascending by edge cidx (insertion sort keeps (cidx, vertex, diam) together; n-1 items at most) */
    for (i64 i = 1; i < np; ++i) {
        col_t c = tmp[i]; u64 s = ss[i]; i64 j = i - 1;
        while (j >= 0 && tmp[j].cidx > c.cidx) { tmp[j + 1] = tmp[j]; ss[j + 1] = ss[j]; --j; }
        tmp[j + 1] = c; ss[j + 1] = s;
    }
    *pair_t = (u64 *)malloc(sizeof(u64) * (np ? np : 1));
    *pair_s = (u64 *)malloc(sizeof(u64) * (np ? np : 1));
    *pair_death = (float *)malloc(sizeof(float) * (np ? np : 1));
    for (i64 i = 0; i < np; ++i) { (*pair_t)[i] = tmp[i].cidx; (*pair_s)[i] = ss[i]; (*pair_death)[i] = tmp[i].diam; }
    *n_pairs = np;
    *n_components = (i64)n - np;
    free(tmp); free(ss); free(parent); free(oldest); free(edges);
    return 0;
}

/* ------------------------------------------------------------------ O3: cohomology reduction */

/* working-column entry; "comes first in the filtration order": smaller diameter, then LARGER cidx */
static int entry_before(const col_t *a, const col_t *b)
{
    if (a->diam != b->diam) return a->diam < b->diam;
    return a->cidx > b->cidx;
}

typedef struct { col_t *a; size_t n, cap; } heap_t;

static void heap_push(heap_t *h, col_t x)
{
    if (h->n == h->cap) { h->cap = h->cap ? 2 * h->cap : 256; h->a = (col_t *)realloc(h->a, h->cap * sizeof(col_t)); }
    size_t i = h->n++;
    while (i > 0) {
        size_t p = (i - 1) / 2;
        if (!entry_before(&x, &h->a[p])) break;
        h->a[i] = h->a[p];
        i = p;
    }
    h->a[i] = x;
}
static col_t heap_pop(heap_t *h)
{
    col_t top = h->a[0];
    col_t x = h->a[--h->n];
    size_t i = 0;
    for (;;) {
        size_t l = 2 * i + 1, r = l + 1, c;
        if (l >= h->n) break;
        c = (r < h->n && entry_before(&h->a[r], &h->a[l])) ? r : l;
        if (!entry_before(&h->a[c], &x)) break;
        h->a[i] = h->a[c];
        i = c;
    }
    if (h->n) h->a[i] = x;
    return top;
}
/* the pivot of the working column over Z/2: equal entries cancel in pairs */
static int heap_pop_pivot(heap_t *h, col_t *out)
{
    while (h->n) {
        col_t p = heap_pop(h);
        if (h->n && h->a[0].cidx == p.cidx && h->a[0].diam == p.diam) { heap_pop(h); continue; }
        *out = p;
        return 1;
    }
    return 0;
}

/* open-addressing map cidx(t) -> cidx(s) for pivots found during the reduction */
typedef struct { u64 *k, *v; size_t cap, n; } map_t;
static size_t map_slot(const map_t *m, u64 key)
{
    size_t i = (size_t)((key * 0x9E3779B97F4A7C15ull) >> 17) & (m->cap - 1);
    while (m->k[i] != UINT64_MAX && m->k[i] != key) i = (i + 1) & (m->cap - 1);
    return i;
}
static void map_put(map_t *m, u64 key, u64 val);
static void map_grow(map_t *m)
{
    map_t o = *m;
    m->cap = o.cap ? 2 * o.cap : 1024;
    m->k = (u64 *)malloc(m->cap * sizeof(u64));
    m->v = (u64 *)malloc(m->cap * sizeof(u64));
    memset(m->k, 0xff, m->cap * sizeof(u64));
    m->n = 0;
    for (size_t i = 0; i < o.cap; ++i) if (o.k[i] != UINT64_MAX) map_put(m, o.k[i], o.v[i]);
    free(o.k); free(o.v);
}
static void map_put(map_t *m, u64 key, u64 val)
{
    if (2 * (m->n + 1) > m->cap) map_grow(m);
    size_t i = map_slot(m, key);
    if (m->k[i] == UINT64_MAX) { m->k[i] = key; ++m->n; }
    m->v[i] = val;
}
static int map_get(const map_t *m, u64 key, u64 *val)
{
    if (!m->cap) return 0;
    size_t i = map_slot(m, key);
    if (m->k[i] == UINT64_MAX) return 0;
    *val = m->v[i];
    return 1;
}

/* push the coboundary of the d-simplex s: its cofacets with diam <= threshold (reading R15) */
static void push_coboundary(heap_t *h, const float *D, const binom_t *b, int n, int d, u64 cidx_s, float threshold)
{
    int m = d + 1, V[MAXV], T[MAXV + 1];
    decode(b, cidx_s, m, n, V);
    float ds = diameter(D, V, m);
    for (int v = n - 1; v >= 0; --v) {
        int in_s = 0;
        for (int p = 0; p < m; ++p) in_s |= (V[p] == v);
        if (in_s) continue;
        float dt = ds;
        for (int p = 0; p < m; ++p) { float x = dist(D, V[p], v); if (x > dt) dt = x; }
        if (!(dt <= threshold)) continue;
        int q = 0, placed = 0;
        for (int p = 0; p < m; ++p) {
            if (!placed && v > V[p]) { T[q++] = v; placed = 1; }
            T[q++] = V[p];
        }
        if (!placed) T[q++] = v;
        col_t e; e.diam = dt; e.cidx = encode(b, T, m + 1);
        heap_push(h, e);
    }
}

/* Columns in coboundary order (col_cidx[i], i < ncols).  known_t/known_s: pivots already known (the
 * apparent pairs, ascending by t); pass n_known = 0 and ALL uncleared columns to reduce everything.
 * With n_known > 0 pass only the non-apparent columns.  Outputs (malloc'ed):
 *   piv_t, piv_s, n_piv : pivots found here, in the order the columns were processed
 *   ess_s, n_ess        : columns that reduce to zero (essential classes)
 *   additions           : number of column additions performed (statistics) */
int oracle_reduce(const float *D, int n, int d, float threshold, const u64 *col_cidx, i64 ncols,
                  const u64 *known_t, const u64 *known_s, i64 n_known,
                  u64 **piv_t, u64 **piv_s, i64 *n_piv, u64 **ess_s, i64 *n_ess, i64 *additions)
{
    binom_t b;
    binom_init(&b, n, d + 2);
    map_t map = {0, 0, 0, 0};      /* cidx(t) -> position j of the column that owns the pivot */
    heap_t h = {0, 0, 0};
    u64 *pt = (u64 *)malloc(sizeof(u64) * (ncols ? ncols : 1));
    u64 *ps = (u64 *)malloc(sizeof(u64) * (ncols ? ncols : 1));
    u64 *es = (u64 *)malloc(sizeof(u64) * (ncols ? ncols : 1));
    /* R_j of the columns reduced here, kept as Algorithm 1 keeps them: the entries of
     * the working column when its pivot was found, equal entries cancelled in pairs. */
    col_t **Rcol = (col_t **)calloc((size_t)(ncols ? ncols : 1), sizeof(col_t *));
    size_t *Rlen = (size_t *)calloc((size_t)(ncols ? ncols : 1), sizeof(size_t));
    i64 np = 0, ne = 0, adds = 0;
    for (i64 j = 0; j < ncols; ++j) {
        h.n = 0;
        push_coboundary(&h, D, &b, n, d, col_cidx[j], threshold);     /* R_j <- D_j */
        for (;;) {
            col_t piv;
            if (!heap_pop_pivot(&h, &piv)) { es[ne++] = col_cidx[j]; break; }   /* zero column */
            u64 owner;
            if (map_get(&map, piv.cidx, &owner)) {                    /* R_j <- R_j + R_i, i = lookup[low(R_j)] */
                heap_push(&h, piv);
                for (size_t e = 0; e < Rlen[owner]; ++e) heap_push(&h, Rcol[owner][e]);
                ++adds;
                continue;
            }
            int found = 0;
            u64 s2 = 0;
            if (n_known) {
                i64 lo = 0, hi = n_known;
                while (lo < hi) { i64 mid = lo + (hi - lo) / 2; if (known_t[mid] < piv.cidx) lo = mid + 1; else hi = mid; }
                if (lo < n_known && known_t[lo] == piv.cidx) { found = 1; s2 = known_s[lo]; }
            }
            if (found) {              /* an apparent column needs no additions: R_i = D_i */
                heap_push(&h, piv);
                push_coboundary(&h, D, &b, n, d, s2, threshold);
                ++adds;
                continue;
            }
            map_put(&map, piv.cidx, (u64)j);                          /* lookup[low(R_j)] <- j */
            pt[np] = piv.cidx; ps[np] = col_cidx[j]; ++np;
            Rcol[j] = (col_t *)malloc(sizeof(col_t) * (h.n + 1));
            Rcol[j][0] = piv;
            Rlen[j] = 1;
            {   /* the rest of the column, equal entries cancelled in pairs */
                col_t e;
                while (heap_pop_pivot(&h, &e)) Rcol[j][Rlen[j]++] = e;
            }
            break;
        }
    }
    for (i64 j = 0; j < ncols; ++j) free(Rcol[j]);
    free(Rcol); free(Rlen);
    free(h.a); free(map.k); free(map.v);
    binom_free(&b);
    *piv_t = pt; *piv_s = ps; *n_piv = np; *ess_s = es; *n_ess = ne;
    if (additions) *additions = adds;
    return 0;
}

/* ------------------------------------------------------------------ O3b: Algorithm 1 on explicit columns */

/* A second, plainer reduction for inputs on which the reduced columns fill in ("difficult datasets",
 * PAPER.md:210; config 3's random matrices): the standard persistence algorithm, Algorithm 1
 * (PAPER.md:99-121), on the EXPLICIT coboundary matrix.  Rows = the
 * (d+1)-simplices of diameter <= threshold, indexed like the matrix of PAPER.md:127 in the reverse of the
 * filtration order (diameter descending, cidx ascending: the comparator of stage 1), so that low(R_j),
 * the largest row index of a nonzero entry, is the cofacet that comes FIRST in the filtration order.  The
 * working column R_j is a bit array over the rows, R_j <- R_j + R_i is an exclusive or; the reduced
 * columns are kept as lists of row indices.  Same interface and same (unique) pairs as oracle_reduce;
 * memory = one word per possible row (the index of cidx -> row) + the stored columns. */
int oracle_reduce_explicit(const float *D, int n, int d, float threshold, const u64 *col_cidx, i64 ncols,
                           const u64 *known_t, const u64 *known_s, i64 n_known,
                           u64 **piv_t, u64 **piv_s, i64 *n_piv, u64 **ess_s, i64 *n_ess, i64 *additions)
{
    int m = d + 1;
    binom_t b;
    binom_init(&b, n, d + 2);
    /* rows: every (d+1)-simplex within the threshold, in coboundary order */
    u64 total_rows = C(&b, n, d + 2);
    col_t *rows = (col_t *)malloc(sizeof(col_t) * (total_rows ? total_rows : 1));
    i64 nrows = 0;
    for (u64 idx = 0; idx < total_rows; ++idx) {
        int verts[MAXV + 1];
        decode(&b, idx, m + 1, n, verts);
        float x = diameter(D, verts, m + 1);
        if (x <= threshold) { rows[nrows].diam = x; rows[nrows].cidx = idx; ++nrows; }
    }
    qsort(rows, (size_t)nrows, sizeof(col_t), cmp_coboundary_order);
    i64 *row_of = (i64 *)malloc(sizeof(i64) * (total_rows ? total_rows : 1)); /* cidx(t) -> row index, -1 = above the threshold */
    for (u64 i = 0; i < total_rows; ++i) row_of[i] = -1;
    for (i64 r = 0; r < nrows; ++r) row_of[rows[r].cidx] = r;
    i64 nwords = (nrows + 63) / 64 + 1;
    u64 *w = (u64 *)calloc((size_t)nwords, sizeof(u64));           /* the working column R_j */
    i64 *owner = (i64 *)malloc(sizeof(i64) * (nrows ? nrows : 1)); /* lookup[row] = j, -1 = none (Alg. 1 line 1) */
    for (i64 r = 0; r < nrows; ++r) owner[r] = -1;
    i64 **Rcol = (i64 **)calloc((size_t)(ncols ? ncols : 1), sizeof(i64 *));
    i64 *Rlen = (i64 *)calloc((size_t)(ncols ? ncols : 1), sizeof(i64));
    u64 *pt = (u64 *)malloc(sizeof(u64) * (ncols ? ncols : 1));
    u64 *ps = (u64 *)malloc(sizeof(u64) * (ncols ? ncols : 1));
    u64 *es = (u64 *)malloc(sizeof(u64) * (ncols ? ncols : 1));
    i64 np = 0, ne = 0, adds = 0;
    int V[MAXV], T[MAXV + 1];
    for (i64 j = 0; j < ncols; ++j) {
        /* R_j <- D_j: the coboundary of the column's simplex */
        i64 top = -1; /* no bit is set above row `top` */
#define XOR_COBOUNDARY(CIDX)                                                                     \
        do {                                                                                     \
            decode(&b, (CIDX), m, n, V);                                                         \
            for (int v = 0; v < n; ++v) {                                                        \
                int in_s = 0;                                                                    \
                for (int p = 0; p < m; ++p) in_s |= (V[p] == v);                                 \
                if (in_s) continue;                                                              \
                int q = 0, placed = 0;                                                           \
                for (int p = 0; p < m; ++p) {                                                    \
                    if (!placed && v > V[p]) { T[q++] = v; placed = 1; }                         \
                    T[q++] = V[p];                                                               \
                }                                                                                \
                if (!placed) T[q++] = v;                                                         \
                i64 r = row_of[encode(&b, T, m + 1)];                                            \
                if (r < 0) continue; /* cofacet above the threshold (reading R15) */             \
                w[r >> 6] ^= 1ull << (r & 63);                                                   \
                if (r > top) top = r;                                                            \
            }                                                                                    \
        } while (0)
        XOR_COBOUNDARY(col_cidx[j]);
        for (;;) {
            /* low(R_j): the largest row index with a nonzero entry */
            i64 low = -1;
            for (i64 wd = top >> 6; top >= 0 && wd >= 0; --wd)
                if (w[wd]) {
                    int bit = 63;
                    while (!((w[wd] >> bit) & 1)) --bit;
                    low = wd * 64 + bit;
                    break;
                }
            top = low;
            if (low < 0) { es[ne++] = col_cidx[j]; break; }                       /* zero column */
            if (owner[low] >= 0) {                                                /* R_j <- R_j + R_i, i = lookup[low] */
                i64 i = owner[low];
                for (i64 e = 0; e < Rlen[i]; ++e) w[Rcol[i][e] >> 6] ^= 1ull << (Rcol[i][e] & 63);
                ++adds;
                continue;
            }
            int found = 0;
            u64 s2 = 0;
            if (n_known) {                                                        /* an apparent column: R_i = D_i */
                u64 ct = rows[low].cidx;
                i64 lo = 0, hi = n_known;
                while (lo < hi) { i64 mid = lo + (hi - lo) / 2; if (known_t[mid] < ct) lo = mid + 1; else hi = mid; }
                if (lo < n_known && known_t[lo] == ct) { found = 1; s2 = known_s[lo]; }
            }
            if (found) { XOR_COBOUNDARY(s2); top = low; ++adds; continue; }
            owner[low] = j;                                                       /* lookup[low(R_j)] <- j */
            pt[np] = rows[low].cidx; ps[np] = col_cidx[j]; ++np;
            i64 cnt = 0;
            for (i64 wd = 0; wd <= (low >> 6); ++wd) cnt += __builtin_popcountll(w[wd]);
            Rcol[j] = (i64 *)malloc(sizeof(i64) * (size_t)cnt);
            for (i64 wd = low >> 6; wd >= 0; --wd)                                /* keep R_j, clear the working column */
                while (w[wd]) {
                    int bit = 63 - __builtin_clzll(w[wd]);
                    Rcol[j][Rlen[j]++] = wd * 64 + bit;
                    w[wd] &= ~(1ull << bit);
                }
            break;
        }
#undef XOR_COBOUNDARY
    }
    for (i64 j = 0; j < ncols; ++j) free(Rcol[j]);
    free(Rcol); free(Rlen); free(owner); free(w); free(row_of); free(rows);
    binom_free(&b);
    *piv_t = pt; *piv_s = ps; *n_piv = np; *ess_s = es; *n_ess = ne;
    if (additions) *additions = adds;
    return 0;
}
