"""Pins of the oracle (CPU only).  Each test checks oracle/brute.py (O1, definitions) and/or
oracle/rips_oracle.c (O2/O3, the paper's algorithms) against something OTHER than themselves:
values the paper prints (tests/golden/), closed forms, invariants, brute force.
Pin numbers P1..P14 refer to SURVEY.md section 8(c) / DESIGN.md "Pins"."""
from itertools import combinations
from math import comb, gamma, inf, lgamma, exp, sqrt, pi

import numpy as np
import pytest

from oracle import brute, oracle
from paper_2003_07989_b200 import inputs


def pairs_ts(o, d):
    return list(zip((int(x) for x in o[d]["app_t"]), (int(x) for x in o[d]["app_s"])))


def bars_sorted(b):
    return sorted((float(x), float(y)) for x, y in b)


# ---------------------------------------------------------------- Eq. 2: combinatorial number system

@pytest.mark.parametrize("n,m", [(7, 1), (7, 2), (9, 3), (8, 4), (10, 5)])
def test_cidx_is_the_colex_rank(n, m):
    """Eq. 2 is a bijection onto 0..C(n,m)-1 and orders simplices colexicographically
    (Remark 2): brute-force enumeration."""
    sx = sorted(combinations(range(n), m), key=lambda s: tuple(reversed(s)))   # colex order
    assert len(sx) == comb(n, m) == oracle.binomial(n, m)
    for rank, s in enumerate(sx):
        dec = list(reversed(s))
        assert brute.cidx(s) == rank
        assert oracle.encode(dec, n) == rank
        assert oracle.decode(rank, m, n) == dec


def test_binomial_against_math_comb():
    for n in (0, 1, 5, 50, 192, 400, 1000, 1088):
        for k in range(0, 7):
            assert oracle.binomial(n, k) == comb(n, k)


def test_edge_cidx_is_the_lower_triangle_offset():
    """The layout of rips_init's matrix: element (i>j) at i(i-1)/2+j, which is cidx of the edge (i j)."""
    for i in range(1, 30):
        for j in range(i):
            assert brute.cidx((i, j)) == i * (i - 1) // 2 + j


# ---------------------------------------------------------------- P1: the paper's worked example

def test_P1_unit_square(golden_lines):
    lines = golden_lines("fig1_unit_square.txt")
    k = lines.index("H1")
    pts = np.array([[float(x) for x in ln.split()] for ln in lines[:k]], dtype=np.float32)
    want = [tuple(np.float32(float(x)) for x in ln.split()) for ln in lines[k + 1:]]
    low = inputs.euclidean_lower(pts)
    for relabel in ([0, 1, 2, 3], [2, 0, 3, 1], [3, 2, 1, 0]):       # vertex numbering must not matter
        lw = inputs.euclidean_lower(pts[relabel])
        b = brute.persistence(lw, 4, 1)
        o = oracle.barcodes(lw, 4, 1)
        assert bars_sorted(b[1]["bars"]) == [tuple(float(x) for x in w) for w in want]
        assert bars_sorted(o[1]["bars"]) == bars_sorted(b[1]["bars"])
        assert bars_sorted(o[0]["bars"]) == [(0.0, 1.0)] * 3 + [(0.0, inf)]
    # exact integer version: cyclic metric on 4 points -> [1,2)
    o = oracle.barcodes(inputs.cyclic_lower(4), 4, 1)
    assert bars_sorted(o[1]["bars"]) == [(1.0, 2.0)]
    assert low.shape == (6,)


# ---------------------------------------------------------------- P2, P4: all diameters equal (Thm. 12)

@pytest.mark.parametrize("n,dim_max", [(5, 1), (6, 3), (9, 2), (12, 2)])
def test_P2_all_equal_staircase(n, dim_max):
    """with all diameters equal the apparent pairs are exactly (s, (n-1,s)), s on
    {0..n-2}: C(n-1,d+1) of them (Fig. 5: 6 of 10 for n=5, d=1); T(n)=C(n-1,2)."""
    low = inputs.constant_lower(n, 1.0)
    o = oracle.barcodes(low, n, dim_max)
    for d in range(1, dim_max + 1):
        want = sorted((brute.cidx(s + (n - 1,)), brute.cidx(s)) for s in combinations(range(n - 1), d + 1))
        assert pairs_ts(o, d) == want
        assert len(want) == comb(n - 1, d + 1)
        if n <= 9:
            assert brute.apparent_pairs(low, n, d) == want
        # after clearing every column is apparent, nothing is left to reduce, no bars
        assert o[d]["non_cidx"].size == 0 and o[d]["bars"].size == 0
        assert o[d]["filt_cidx"].size == comb(n - 1, d + 1)
    assert bars_sorted(o[0]["bars"]) == [(0.0, 1.0)] * (n - 1) + [(0.0, inf)]
    # tie-break direction inside equal diameters: cidx ascending in coboundary order
    assert list(o[1]["filt_cidx"]) == sorted(int(c) for c in o[1]["filt_cidx"])


# ---------------------------------------------------------------- P3: Figure 6

def test_P3_fig6_descending(golden_lines):
    lines = golden_lines("fig6_descending_n5.txt")
    k = lines.index("PAIRS")
    rows = [[float(x) for x in ln.split()] for ln in lines[:k]]
    low = np.array([x for r in rows for x in r], dtype=np.float32)
    assert np.array_equal(low, inputs.descending_lower(5))
    want = []
    for ln in lines[k + 1:]:
        s, t = ln.split("|")
        want.append((brute.cidx(tuple(int(x) for x in t.split())), brute.cidx(tuple(int(x) for x in s.split()))))
    want.sort()
    assert brute.apparent_pairs(low, 5, 1) == want
    assert pairs_ts(oracle.barcodes(low, 5, 1), 1) == want
    for n in (6, 8, 11):                                            # same staircase for any n
        o = oracle.barcodes(inputs.descending_lower(n), n, 1)
        assert pairs_ts(o, 1) == sorted((brute.cidx((a, b, n - 1)), brute.cidx((a, b)))
                                        for a, b in combinations(range(n - 1), 2))


# ---------------------------------------------------------------- P5: a single (d+1)-simplex

@pytest.mark.parametrize("d", [1, 2, 3, 4])
def test_P5_single_simplex_has_one_apparent_pair(d):
    """n = d+2 points: exactly one apparent pair of dimension (d,d+1), ties or not."""
    n = d + 2
    for seed, gen in enumerate((inputs.random_matrix_lower, inputs.small_integer_lower, None)):
        low = inputs.constant_lower(n) if gen is None else gen(n, seed)
        s1 = oracle.stage1(low, n, d)
        s2 = oracle.stage2(low, n, d, s1[0], s1[1])
        assert s2["app_t"].size == 1 and int(s2["app_t"][0]) == 0
        assert brute.apparent_pairs(low, n, d) == [(0, int(s2["app_s"][0]))]


# ---------------------------------------------------------------- P13 (+P6, P7, P9, P10): brute force

def _regimes(n, seed):
    yield "distinct", inputs.random_matrix_lower(n, seed)
    yield "ties", inputs.small_integer_lower(n, seed)
    yield "points", inputs.euclidean_lower(inputs.cube_points(n, 2, seed))


@pytest.mark.parametrize("n,dim_max", [(2, 1), (3, 2), (5, 2), (6, 3), (7, 2), (8, 2), (9, 1)])
def test_P13_c_oracle_equals_brute_force(n, dim_max):
    for seed in range(3):
        for name, low in _regimes(n, seed):
            thresholds = [inf, float(np.float32(np.quantile(low, 0.6))), inputs.enclosing_radius(low, n)]
            for thr in thresholds:
                b = brute.persistence(low, n, dim_max, thr)
                o_app = oracle.barcodes(low, n, dim_max, thr, use_apparent=True)
                o_all = oracle.barcodes(low, n, dim_max, thr, use_apparent=False)
                for d in range(dim_max + 1):
                    for o in (o_app, o_all):
                        got = sorted(zip((int(x) for x in o[d]["pivot_s"]), (int(x) for x in o[d]["pivot_t"])))
                        assert got == b[d]["pairs"], (name, thr, d)
                        assert bars_sorted(o[d]["bars"]) == b[d]["bars"], (name, thr, d)
                    if d == 0:
                        continue
                    assert sorted(int(x) for x in o_app[d]["essential"]) == b[d]["essential"]
                    # Definition 5 literally == Algorithm 3 (this is the test of Lemma 7)
                    assert pairs_ts(o_app, d) == brute.apparent_pairs(low, n, d, thr), (name, thr, d)
                    # filtration with clearing == the definition
                    cleared = [t for (_, t) in b[d - 1]["pairs"]]
                    want = brute.coboundary_columns(low, n, d, thr, cleared)
                    got = list(zip((float(x) for x in o_app[d]["filt_diam"]), (int(x) for x in o_app[d]["filt_cidx"])))
                    assert got == want, (name, thr, d)
                    # P6: apparent pairs are persistence pairs of zero persistence (Eq. 4)
                    allp = set(zip((int(x) for x in o_all[d]["pivot_t"]), (int(x) for x in o_all[d]["pivot_s"])))
                    for (t, s) in pairs_ts(o_app, d):
                        assert (t, s) in allp
                        assert oracle.diameter(low, t, d + 2, n) == oracle.diameter(low, s, d + 1, n)
                    # P10: bookkeeping (Table 5's identity)
                    c = o_app[d]["counts"]
                    assert c["kept"] + c["removed_by_diameter"] + c["cleared"] == comb(n, d + 1)
                    # P9: full complex: C(n-1,d+1) columns, every one gets a pivot, no essential class
                    if thr == inf:
                        assert c["kept"] == comb(n - 1, d + 1) == o_app[d]["pivot_t"].size
                        assert o_app[d]["essential"].size == 0


@pytest.mark.parametrize("n,dim_max", [(3, 2), (6, 3), (8, 2), (9, 1)])
def test_P13_explicit_reduction_equals_brute_force(n, dim_max):
    """oracle_reduce_explicit (Algorithm 1 on the explicit coboundary matrix) against the
    brute-force boundary-matrix reduction, with and without the apparent pairs as known pivots."""
    for seed in range(3):
        for name, low in _regimes(n, seed):
            for thr in (inf, float(np.float32(np.quantile(low, 0.6)))):
                b = brute.persistence(low, n, dim_max, thr)
                for use_apparent in (True, False):
                    o = oracle.barcodes(low, n, dim_max, thr, use_apparent=use_apparent, explicit=True)
                    for d in range(1, dim_max + 1):
                        got = sorted(zip((int(x) for x in o[d]["pivot_s"]), (int(x) for x in o[d]["pivot_t"])))
                        assert got == b[d]["pairs"], (name, thr, d, use_apparent)
                        assert bars_sorted(o[d]["bars"]) == b[d]["bars"], (name, thr, d, use_apparent)
                        assert sorted(int(x) for x in o[d]["essential"]) == b[d]["essential"]


@pytest.mark.parametrize("k,n", [(1, 26), (2, 22), (3, 30), (4, 40), (5, 28)])
def test_explicit_and_heap_reductions_agree(k, n):
    """The two reductions of the oracle (implicit columns + heap; explicit matrix + bit array) on the shadow
    configs: same pivots in the same processing order, same essential columns."""
    w = inputs.config(k, n)
    thr = w.threshold if k not in (4, 5) else (inputs.enclosing_radius(w.dist, n) if k == 5 else float(np.float32(np.quantile(w.dist, 0.3))))
    a = oracle.barcodes(w.dist, n, w.dim_max, thr)
    e = oracle.barcodes(w.dist, n, w.dim_max, thr, explicit=True)
    for d in range(1, w.dim_max + 1):
        for key in ("red_t", "red_s", "essential", "pivot_t", "pivot_s"):
            assert np.array_equal(a[d][key], e[d][key]), (d, key)
        assert np.array_equal(a[d]["bars"].view(np.uint32), e[d]["bars"].view(np.uint32))


# ---------------------------------------------------------------- the slice mode of stage 1, the visit counts of stage 2

@pytest.mark.parametrize("k,n,d", [(1, 20, 2), (2, 16, 3), (3, 24, 1), (4, 30, 2), (5, 18, 2)])
def test_stage1_slices_concatenate_to_the_whole(k, n, d):
    """oracle_stage1 with idx_lo/idx_hi and do_sort = 0 (what the full-size GPU tests and bench.py call): the
    survivors of consecutive slices, concatenated, are the survivors of the whole index range in increasing
    cidx, and re-sorted they are the filtration array; against the definition (brute.coboundary_columns)."""
    w = inputs.config(k, n)
    thr = inf if k not in (4, 5) else float(np.float32(np.quantile(w.dist, 0.5)))
    prev = oracle.barcodes(w.dist, n, d - 1, thr) if d > 1 else {0: oracle.barcodes(w.dist, n, 0, thr)[0]}
    cleared = prev[d - 1]["pivot_t"]
    total = comb(n, d + 1)
    fd, fc, counts = oracle.stage1(w.dist, n, d, thr, cleared)                    # whole range, sorted
    ud, uc, ucounts = oracle.stage1(w.dist, n, d, thr, cleared, sort=False)        # whole range, cidx order
    assert ucounts == counts and list(uc) == sorted(int(c) for c in fc)
    cuts = [0, 1, total // 7, total // 7 + 1, total // 2, total - 3, total]
    cd, cc, tot = [], [], {"kept": 0, "removed_by_diameter": 0, "cleared": 0}
    for lo, hi in zip(cuts[:-1], cuts[1:]):
        sd, sc, c = oracle.stage1(w.dist, n, d, thr, cleared, lo, hi, sort=False)
        assert all(lo <= int(x) < hi for x in sc)
        assert c["kept"] + c["removed_by_diameter"] + c["cleared"] == hi - lo
        cd.append(sd); cc.append(sc)
        for key in tot:
            tot[key] += c[key]
    cd, cc = np.concatenate(cd), np.concatenate(cc)
    assert tot == counts
    assert np.array_equal(cc, uc) and np.array_equal(cd.view(np.uint32), ud.view(np.uint32))
    # against the definition: brute force columns (coboundary order), re-sorted by cidx
    if n <= 20:
        b = brute.persistence(w.dist, n, d - 1, thr) if d > 1 else brute.persistence(w.dist, n, 0, thr)
        want = brute.coboundary_columns(w.dist, n, d, thr, [t for (_, t) in b[d - 1]["pairs"]])
        assert sorted((c, dm) for dm, c in want) == list(zip((int(x) for x in cc), (float(x) for x in cd)))
    # an empty slice and a slice of one
    sd, sc, c = oracle.stage1(w.dist, n, d, thr, cleared, 5, 5, sort=False)
    assert sc.size == 0 and c == {"kept": 0, "removed_by_diameter": 0, "cleared": 0}


@pytest.mark.parametrize("k,n,d", [(1, 18, 1), (2, 14, 2), (3, 20, 1), (3, 12, 3)])
def test_stage2_visit_counts(k, n, d):
    """oracle_stage2's `visits` output: the number of cofacets evaluated per column = position (counted over
    the vertices not in s, from n-1 down) of the first cofacet of equal diameter, or n-d-1 if there is none;
    re-derived with numpy from the square matrix."""
    w = inputs.config(k, n)
    sq = inputs.square_from_lower(w.dist, n)
    fd, fc, _ = oracle.stage1(w.dist, n, d)
    s2 = oracle.stage2(w.dist, n, d, fd, fc, want_visits=True)
    for i in range(fc.size):
        verts = oracle.decode(int(fc[i]), d + 1, n)
        others = [v for v in range(n - 1, -1, -1) if v not in verts]
        dt = np.maximum(fd[i], sq[np.ix_(others, verts)].max(axis=1))
        hit = np.nonzero(dt == fd[i])[0]
        assert s2["visits"][i] == (hit[0] + 1 if hit.size else n - d - 1)
        if not hit.size:
            assert s2["flag"][i] == 0


@pytest.mark.parametrize("n,d", [(6, 1), (7, 2), (8, 1), (8, 3)])
def test_P7_apparent_set_unchanged_by_clearing(n, d):
    """Proposition 10: Alg. 3 over ALL d-simplices finds the same pairs as over the cleared columns."""
    for seed in range(3):
        for _, low in _regimes(n, seed):
            o = oracle.barcodes(low, n, d)
            fd, fc, _ = oracle.stage1(low, n, d, inf, cleared=())
            s2 = oracle.stage2(low, n, d, fd, fc)
            assert list(zip(s2["app_t"], s2["app_s"])) == list(zip(o[d]["app_t"], o[d]["app_s"]))


# ---------------------------------------------------------------- P8: enclosing radius (Prop. 4)

@pytest.mark.parametrize("k,n", [(1, 24), (2, 20), (5, 22), (3, 16)])
def test_P8_enclosing_radius_keeps_nonzero_bars(k, n):
    w = inputs.config(k, n)
    r = inputs.enclosing_radius(w.dist, n)
    full = oracle.barcodes(w.dist, n, 2, inf)
    trunc = oracle.barcodes(w.dist, n, 2, r)
    for d in (1, 2):
        assert bars_sorted(full[d]["bars"]) == bars_sorted(trunc[d]["bars"])
        assert all(np.isfinite(full[d]["bars"][:, 1])) if full[d]["bars"].size else True
    assert bars_sorted(full[0]["bars"]) == bars_sorted(trunc[0]["bars"])


# ---------------------------------------------------------------- P9, P10 on the tables' identities

def test_P9_table1_all_pairs_identity(golden_lines):
    for ln in golden_lines("table1_all_pairs.txt"):
        name, n, d, allp = ln.split()
        n, d, allp = int(n), int(d), int(allp)
        assert sum(oracle.binomial(n - 1, k + 1) for k in range(1, d + 1)) == allp, name
    # and the same identity holds for what the oracle actually computes on a small full complex
    w = inputs.config(2, 14)
    o = oracle.barcodes(w.dist, 14, 3)
    assert sum(o[d]["pivot_t"].size for d in (1, 2, 3)) == sum(comb(13, k + 1) for k in (1, 2, 3))


def test_P10_table5_counts_identity(golden_lines):
    for ln in golden_lines("table5_simplex_counts.txt"):
        name, n, d, possible, kept, removed, cleared = ln.split()
        n, d = int(n), int(d)
        assert int(possible) == int(kept) + int(removed) + int(cleared), name
        assert int(possible) == sum(oracle.binomial(n, k + 1) for k in range(1, d + 1)), name


# ---------------------------------------------------------------- P11: random permutation matrices, dim 1

def _expected_fraction(n):
    """E[apparent fraction] = 1 - (sqrt(pi)/2) Gamma(n-1)/Gamma(n-1/2) (derivation in DESIGN.md, pin P11)."""
    return 1.0 - (sqrt(pi) / 2.0) * exp(lgamma(n - 1) - lgamma(n - 0.5))


def test_P11_closed_form_reproduces_the_papers_numbers(golden_lines):
    for ln in golden_lines("sec66_apparent_fraction.txt"):
        n, frac = ln.split()
        assert abs(_expected_fraction(int(n)) - float(frac)) < 2e-5


def _dim1_apparent_by_definition(low, n):
    """Tie-free inputs: the edge ab is apparent iff some c has max(D[a,c],D[b,c]) < D[a,b]; its partner is
    ab + the LARGEST such c.  An independent O(n^3) numpy check of A_1 (pin P11)."""
    sq = inputs.square_from_lower(low, n).astype(np.float64)
    np.fill_diagonal(sq, np.inf)
    out = []
    for a in range(1, n):
        for b in range(a):
            m = np.maximum(sq[a], sq[b])
            cs = np.nonzero(m < sq[a, b])[0]
            if cs.size:
                out.append((brute.cidx((a, b, int(cs.max()))), a * (a - 1) // 2 + b))
    return sorted(out)


def test_P11_dim1_apparent_pairs_on_random_permutation_matrices():
    fr = []
    for seed in range(4):
        n = 120
        low = inputs.permutation_matrix_lower(n, seed)
        fd, fc, _ = oracle.stage1(low, n, 1)
        s2 = oracle.stage2(low, n, 1, fd, fc)
        assert list(zip((int(x) for x in s2["app_t"]), (int(x) for x in s2["app_s"]))) == _dim1_apparent_by_definition(low, n)
        fr.append(s2["app_t"].size / comb(n, 2))
    assert abs(np.mean(fr) - _expected_fraction(120)) < 0.01
    assert np.mean(fr) <= (120 - 2) / 120           # Theorem 12 upper bound


def test_theorem12_bounds_hold_when_its_condition_holds():
    """if every d-simplex containing vertex n-1 has diameter <= every d-simplex without it,
    the apparent fraction lies in [1/(d+2), (n-d-1)/n]."""
    n = 9
    rng = np.random.default_rng(5)
    sq = rng.random((n, n)).astype(np.float32) + 1.0
    sq = np.maximum(sq, sq.T)
    sq[n - 1, :] = sq[:, n - 1] = 0.5                # edges at vertex n-1 are the shortest
    low = inputs.lower_from_square(sq)
    fd, fc, _ = oracle.stage1(low, n, 1)
    frac = oracle.stage2(low, n, 1, fd, fc)["app_t"].size / comb(n, 2)
    assert 1 / 3 <= frac <= (n - 2) / n


# ---------------------------------------------------------------- P12: n-gons and cross-polytopes

@pytest.mark.parametrize("n", [4, 5, 6, 7, 9, 12])
def test_P12_cyclic_ngon_brute(n):
    low = inputs.cyclic_lower(n)
    b = brute.persistence(low, n, 2 if n <= 9 else 1)
    assert b[1]["bars"] == [(1.0, float(-(-n // 3)))]
    if n % 3 == 0 and n <= 9:
        assert b[2]["bars"] == [(n / 3.0, n / 3.0 + 1.0)] * (n // 3 - 1)


@pytest.mark.parametrize("n", [12, 21, 30])
def test_P12_cyclic_ngon_c_oracle(n):
    o = oracle.barcodes(inputs.cyclic_lower(n), n, 2)
    assert bars_sorted(o[1]["bars"]) == [(1.0, float(-(-n // 3)))]
    want2 = [(n / 3.0, n / 3.0 + 1.0)] * (n // 3 - 1) if n % 3 == 0 else []
    assert bars_sorted(o[2]["bars"]) == want2


@pytest.mark.parametrize("m", [2, 3, 4])
def test_P12_cross_polytope(m):
    n = 2 * m
    low = inputs.cross_polytope_lower(m)
    o = oracle.barcodes(low, n, m - 1)
    b = brute.persistence(low, n, m - 1)
    for d in range(1, m):
        want = [(1.0, 2.0)] if d == m - 1 else []
        assert bars_sorted(o[d]["bars"]) == want
        assert b[d]["bars"] == want


# ---------------------------------------------------------------- P14: Betti_0

@pytest.mark.parametrize("k,n", [(1, 30), (4, 60), (3, 25)])
def test_P14_betti0_is_the_number_of_components(k, n):
    w = inputs.config(k, n)
    for thr in (inf, float(np.float32(np.quantile(w.dist, 0.05))), float(np.float32(np.quantile(w.dist, 0.3)))):
        z = oracle.dim0(w.dist, n, thr)
        assert z["n_components"] == brute.connected_components(w.dist, n, thr)
        assert z["t"].size == n - z["n_components"]
        if thr == inf:
            assert z["n_components"] == 1
        assert list(z["t"]) == sorted(z["t"])


# ---------------------------------------------------------------- degenerate inputs

def test_degenerate_inputs():
    # one point, two points, threshold below every distance, duplicate points (zero distances)
    o = oracle.barcodes(np.zeros(0, dtype=np.float32), 1, 2)
    assert bars_sorted(o[0]["bars"]) == [(0.0, inf)] and o[1]["filt_cidx"].size == 0
    o = oracle.barcodes(np.array([3.0], dtype=np.float32), 2, 1)
    assert bars_sorted(o[0]["bars"]) == [(0.0, 3.0), (0.0, inf)] and o[1]["filt_cidx"].size == 0
    low = inputs.random_matrix_lower(6, 1) + 1.0
    o = oracle.barcodes(low, 6, 2, 0.5)
    assert bars_sorted(o[0]["bars"]) == [(0.0, inf)] * 6 and o[1]["filt_cidx"].size == 0
    pts = np.array([[0, 0], [0, 0], [1, 0], [1, 0], [0, 1]], dtype=np.float32)
    low = inputs.euclidean_lower(pts)
    o, b = oracle.barcodes(low, 5, 2), brute.persistence(low, 5, 2)
    for d in (0, 1, 2):
        assert bars_sorted(o[d]["bars"]) == b[d]["bars"]
    assert len(b[0]["bars"]) == 3                      # two zero-length bars dropped (reading R11)
