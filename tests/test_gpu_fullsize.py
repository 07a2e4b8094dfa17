"""GPU parity at BASELINE.json's full sizes, in the launch configuration bench.py times
(rips_compute / rips_stage1 + rips_stage2 through the C ABI on the whole workload).

The oracle cannot produce every array of configs 2-5 in seconds, so the comparison is on SAMPLED index
ranges that the oracle computes one by one (Algorithms 7-8 and 3 over a slice [lo, hi) of the candidate
indices, with the oracle's own clearing set), each compared element by element for equality with the
part of the GPU's arrays that falls in that slice, plus properties that hold at any size:
  * the bookkeeping identity candidates = kept + removed by diameter + cleared (Table 5)
  * without a threshold: columns = C(n-1, d+1) (Table 1's "all pairs")
  * filtration sorted by (diameter descending, cidx ascending)
  * apparent pairs strictly ascending in t, diam(s) = diam(t) on a sample
"""
from math import comb, inf

import numpy as np
import pytest

from oracle import oracle
from paper_2003_07989_b200 import inputs

pytestmark = pytest.mark.gpu

SLICE = 150_000


@pytest.fixture(scope="module")
def R():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2003_07989_b200 import rips
    rips.lib()
    return rips


def oracle_clearing_sets(w, explicit=False):
    """Pivot rows of every dimension below the top one, from the oracle's own pipeline (the TRUE clearing sets:
    apparent pairs united with the pivots of the reduction).  explicit: the oracle's second reduction (Algorithm 1
    on the explicit matrix), for config 3's random matrix, whose reduced columns fill in."""
    z = oracle.dim0(w.dist, w.n, w.threshold)
    cleared = {1: z["t"]}
    for d in range(1, w.dim_max):
        fd, fc, _ = oracle.stage1(w.dist, w.n, d, w.threshold, cleared[d])
        s2 = oracle.stage2(w.dist, w.n, d, fd, fc)
        red = oracle.reduce_columns(w.dist, w.n, d, w.threshold, s2["non_cidx"], s2["app_t"], s2["app_s"], explicit=explicit)
        cleared[d + 1] = np.sort(np.concatenate([s2["app_t"], red["t"]]))
    return cleared


def slices_of(total):
    """beginning, middle, and the end (the end holds the rows of the top vertices: the irregular pairs)"""
    if total <= 3 * SLICE:
        return [(0, total)]
    mid = total // 2
    return [(0, SLICE), (mid, mid + SLICE), (total - SLICE, total)]


def check_top_dimension(R, w, explicit=False):
    import torch
    D, n = w.dim_max, w.n
    cleared = oracle_clearing_sets(w, explicit)
    with R.Rips(w.dist, n, D, w.threshold) as g:
        g.dim0()
        for d in range(1, D):
            g.stage1(d); g.stage2(d)
            g.reduce(d)
        g.stage1(D); g.stage2(D)          # (the barcodes of the top dimension: test_full_size_barcodes)
        st = g.stats(D)
        total = comb(n, D + 1)
        assert st["n_candidates"] == total
        assert st["n_columns"] + st["n_removed_by_diameter"] + st["n_cleared"] == total
        if w.threshold == inf:
            assert st["n_columns"] == comb(n - 1, D + 1) and st["n_removed_by_diameter"] == 0
        assert st["n_apparent"] + st["n_nonapparent"] == st["n_columns"]
        fd, fc = g.filtration(D)
        assert fd.numel() == st["n_columns"]
        if fd.numel() > 1:
            dd = fd[1:] - fd[:-1]
            assert bool((dd <= 0).all())
            assert bool((fc[1:][dd == 0] > fc[:-1][dd == 0]).all())
        at, as_ = g.apparent_pairs(D)
        assert at.numel() == st["n_apparent"]
        if at.numel() > 1:
            assert bool((at[1:] > at[:-1]).all())
        nd, nc = g.nonapparent(D)
        assert nc.numel() == st["n_nonapparent"]
        for lo, hi in slices_of(total):
            tag = f"{w.name} d={D} slice [{lo},{hi})"
            od, oc, counts = oracle.stage1(w.dist, n, D, w.threshold, cleared[D], lo, hi, sort=False)
            # --- filtration: the GPU's records whose cidx falls in the slice, in cidx order
            m = (fc >= lo) & (fc < hi)
            gc, order = torch.sort(fc[m])
            gd = fd[m][order]
            assert np.array_equal(gc.cpu().numpy().astype(np.uint64), oc), tag
            assert np.array_equal(gd.cpu().numpy().view(np.uint32), od.view(np.uint32)), tag
            # --- apparent pairs and non-apparent columns of the slice
            s2 = oracle.stage2(w.dist, n, D, od, oc)
            m = (as_ >= lo) & (as_ < hi)
            gs, order = torch.sort(as_[m])
            gt = at[m][order]
            o_order = np.argsort(s2["app_s"], kind="stable")
            assert np.array_equal(gs.cpu().numpy().astype(np.uint64), s2["app_s"][o_order]), tag
            assert np.array_equal(gt.cpu().numpy().astype(np.uint64), s2["app_t"][o_order]), tag
            m = (nc >= lo) & (nc < hi)
            gn, order = torch.sort(nc[m])
            o_order = np.argsort(s2["non_cidx"], kind="stable")
            assert np.array_equal(gn.cpu().numpy().astype(np.uint64), s2["non_cidx"][o_order]), tag
            assert np.array_equal(nd[m][order].cpu().numpy().view(np.uint32),
                                  s2["non_diam"][o_order].view(np.uint32)), tag
            # --- a10: lookups of the slice's rows
            if s2["app_t"].size:
                q = s2["app_t"][:: max(1, s2["app_t"].size // 300)]
                got = g.pivot_lookup(D, q.astype(np.int64)).cpu().numpy()
                want = s2["app_s"][:: max(1, s2["app_t"].size // 300)].astype(np.int64)
                assert np.array_equal(got, want), tag
                # apparent pairs have zero persistence
                for t, s in list(zip(q, want))[:20]:
                    assert oracle.diameter(w.dist, int(t), D + 2, n) == oracle.diameter(w.dist, int(s), D + 1, n)


@pytest.mark.parametrize("k", [2, 3, 4, 5])
def test_full_size_sampled(R, k):
    check_top_dimension(R, inputs.config(k), explicit=(k == 3))


def _compare_dimension(g, o, d, tag):
    pt, ps = g.pivots(d)
    assert np.array_equal(pt.cpu().numpy().astype(np.uint64), o[d]["pivot_t"]), tag
    assert np.array_equal(ps.cpu().numpy().astype(np.uint64), o[d]["pivot_s"]), tag
    assert np.array_equal(g.barcodes(d).view(np.uint32), o[d]["bars"].reshape(-1, 2).view(np.uint32)), tag
    if d == 0:
        return
    fd, fc = g.filtration(d)
    assert np.array_equal(fc.cpu().numpy().astype(np.uint64), o[d]["filt_cidx"]), tag
    assert np.array_equal(fd.cpu().numpy().view(np.uint32), o[d]["filt_diam"].view(np.uint32)), tag
    at, as_ = g.apparent_pairs(d)
    assert np.array_equal(at.cpu().numpy().astype(np.uint64), o[d]["app_t"]), tag
    assert np.array_equal(as_.cpu().numpy().astype(np.uint64), o[d]["app_s"]), tag
    nd, nc = g.nonapparent(d)
    assert np.array_equal(nc.cpu().numpy().astype(np.uint64), o[d]["non_cidx"]), tag
    st = g.stats(d)
    assert st["n_essential"] == o[d]["essential"].size and st["n_reduced_pivots"] == o[d]["red_t"].size, tag


def test_columns_with_more_than_2048_cofacets(R):
    """2200 points, no threshold, dimension 1: every column has 2198 cofacets -- more than a warp's working column of
    prereduce_kernel holds (2048 entries; round 1 wrote such columns off as zero columns) and more than the
    shared-memory accumulator of reduce_kernel takes in one addition, so every non-apparent column goes through the
    CTA-level reduction with coboundaries as runs of their own.  Every array against the oracle."""
    w = inputs.config(1, 2200)
    o = oracle.barcodes(w.dist, w.n, 1, w.threshold)
    with R.Rips(w.dist, w.n, 1, w.threshold) as g:
        g.compute()
        for d in (0, 1):
            _compare_dimension(g, o, d, f"{w.name} d={d}")
        st = g.stats(1)
        assert st["n_essential"] == 0 and st["n_reduce_serial"] == st["n_nonapparent"] == o[1]["non_cidx"].size
        assert st["n_additions"] >= o[1]["additions"] > 0


def test_block_maxima_guide_the_scan_in_both_fused_kernels(R):
    """From 2048 points on rips_init builds the block maxima of the key matrix's rows and the fused kernels' warp scan
    for a cofacet of equal diameter reads only the blocks of 32 vertices they leave open (stage1.cu, summary_scan).
    2300 points in dimension 1: without a threshold (slot mode, enumerate_slot_kernel) and with one that admits 40 %
    of the edges (compact mode, enumerate_apparent_kernel), the dense path forced.  Every array against the oracle."""
    w = inputs.config(1, 2300)
    thr = float(np.quantile(w.dist, 0.4))
    for threshold in (w.threshold, thr):
        o = oracle.barcodes(w.dist, w.n, 1, threshold)
        with R.Rips(w.dist, w.n, 1, threshold) as g:
            g.set_mode("dense")
            g.compute()
            for d in (0, 1):
                _compare_dimension(g, o, d, f"{w.name} thr={threshold} d={d}")
            st = g.stats(1)
            assert st["n_candidates"] == comb(w.n, 2)
            if threshold == thr:
                assert 0.39 * comb(w.n, 2) < st["n_columns"] + st["n_cleared"] < 0.41 * comb(w.n, 2)


def test_dimension0_with_vertex_numbers_beyond_15_bits(R):
    """33,000 points on a line at distinct integer positions (fp32-exact distances, many of them equal): dim0_kernel
    keeps its forest as 16-bit vertex numbers in shared memory for every n rips_init admits.  The finite bars of
    dimension 0 are the edges of a minimum spanning tree, whose multiset of weights is unique whatever the ties: the
    gaps between neighbours on the line (a closed form, not the oracle: its dimension 0 needs minutes at this size).
    The pivots must be edges of that weight, and every vertex but one must die exactly once."""
    n = 33000
    rng = np.random.default_rng(11)
    pos = rng.choice(1 << 23, n, replace=False).astype(np.float32)
    low = np.empty(n * (n - 1) // 2, dtype=np.float32)
    for i in range(1, n):
        low[i * (i - 1) // 2: i * (i + 1) // 2] = np.abs(pos[i] - pos[:i])
    gaps = np.sort(np.diff(np.sort(pos)))
    with R.Rips(low, n, 0) as g:
        g.dim0()
        bars = g.barcodes(0)
        assert bars.shape[0] == n                                    # n - 1 finite bars and the essential one
        fin = bars[np.isfinite(bars[:, 1])]
        assert fin.shape[0] == n - 1 and np.all(fin[:, 0] == 0)
        assert np.array_equal(np.sort(fin[:, 1]), gaps)
        pt, ps = g.pivots(0)                                         # (edge, vertex that dies with it)
        e = pt.cpu().numpy().astype(np.int64)
        v = ps.cpu().numpy().astype(np.int64)
        assert np.array_equal(np.sort(low[e]), gaps)
        assert np.unique(v).size == n - 1 and v.min() >= 0 and v.max() < n


def test_config4_through_both_paths(R):
    """Config 4 (1000 points, threshold 0.15: 1.2 % of the edges) at full size through the sparse path (what
    RIPS_MODE_AUTO picks for it) and through the dense path: every array of every dimension against the oracle."""
    w = inputs.config(4)
    o = oracle.barcodes(w.dist, w.n, w.dim_max, w.threshold)
    for mode in ("sparse", "dense"):
        with R.Rips(w.dist, w.n, w.dim_max, w.threshold) as g:
            g.set_mode(mode)
            g.compute()
            for d in range(0, w.dim_max + 1):
                _compare_dimension(g, o, d, f"{w.name} {mode} d={d}")
            st = g.stats(2)
            assert st["n_candidates"] == comb(w.n, 3) and st["n_slots"] == (o[2]["counts"]["kept"] + o[2]["counts"]["cleared"] if mode == "sparse" else st["n_columns"])


def test_config7_sparse_only(R):
    """1700 points under a threshold that admits ~2.4 % of the edges, dimensions 1..3: C(1700,4) = 3.5e11 candidate
    tetrahedra, which the oracle's Algorithm 7 cannot enumerate in a test's time (the dense path needs seconds and a
    43 GB bitmap).  Dimension 1 against the
    oracle; above it what can be checked independently: the number of simplices the sparse path lists against clique
    counts of the threshold graph (numpy), the orders of the arrays, zero persistence of sampled apparent pairs, and
    the sparse path of a 500-point version of the same cloud against the oracle in full (same code path, sizes the
    oracle reaches)."""
    import torch
    w = inputs.config(7)
    n = w.n
    sq = inputs.square_from_lower(w.dist, n)
    A = ((sq <= np.float32(w.threshold)) & ~np.eye(n, dtype=bool))
    Af = A.astype(np.float32)
    n_edges = int(A.sum()) // 2
    n_tri = int(round(float(np.trace(Af @ Af @ Af)) / 6.0))
    iu, ju = np.nonzero(np.triu(A, 1))
    n_tet = 0
    for a, b in zip(iu, ju):                      # 4-cliques: edges inside the common neighbourhood of every edge, / 6
        cn = np.nonzero(A[a] & A[b])[0]
        if cn.size >= 2:
            n_tet += int(A[np.ix_(cn, cn)].sum()) // 2
    n_tet //= 6
    o1 = oracle.barcodes(w.dist, n, 1, w.threshold)
    with R.Rips(w.dist, n, 3, w.threshold) as g:
        g.compute()                               # RIPS_MODE_AUTO: sparse
        _compare_dimension(g, o1, 0, "cfg7 d=0")
        _compare_dimension(g, o1, 1, "cfg7 d=1")
        for d, cliques in ((1, n_edges), (2, n_tri), (3, n_tet)):
            st = g.stats(d)
            assert st["n_slots"] == cliques == st["n_columns"] + st["n_cleared"], (d, st, cliques)
            assert st["n_candidates"] == comb(n, d + 1) and st["n_removed_by_diameter"] == comb(n, d + 1) - cliques
            assert st["n_apparent"] + st["n_nonapparent"] == st["n_columns"]
            assert st["n_cleared"] == g.pivots(d - 1)[0].numel()   # every pivot row of dimension d-1 is a simplex of the complex
            fd, fc = g.filtration(d)
            dd = fd[1:] - fd[:-1]
            assert bool((dd <= 0).all()) and bool((fc[1:][dd == 0] > fc[:-1][dd == 0]).all())
            assert float(fd.max()) <= w.threshold
            at, as_ = g.apparent_pairs(d)
            assert bool((at[1:] > at[:-1]).all())
            idx = torch.linspace(0, at.numel() - 1, 60).long()
            for t, s_ in zip(at[idx].tolist(), as_[idx].tolist()):
                assert oracle.diameter(w.dist, t, d + 2, n) == oracle.diameter(w.dist, s_, d + 1, n)
            pt, ps = g.pivots(d)
            assert pt.numel() + st["n_essential"] == st["n_columns"] and torch.unique(ps).numel() == ps.numel()
    ws = inputs.config(7, 500)
    o = oracle.barcodes(ws.dist, ws.n, 3, ws.threshold)
    with R.Rips(ws.dist, ws.n, 3, ws.threshold) as g:
        g.set_mode("sparse")
        g.compute()
        for d in range(0, 4):
            _compare_dimension(g, o, d, f"{ws.name} d={d}")


@pytest.mark.parametrize("k", [2, 4, 5])
def test_full_size_barcodes(R, k):
    """BASELINE.json configs 2, 4, 5 at full size through rips_compute: EVERY array of EVERY dimension -- filtration,
    apparent pairs, non-apparent columns, pivots (apparent united with the device reduction's), bars -- element by
    element against the oracle's whole pipeline (oracle.barcodes: Algorithms 7-8, 3, and the reduction).  Config 2's
    dimension 3 costs the oracle about a minute (54.9 million candidates, 142,819 columns to reduce)."""
    w = inputs.config(k)
    o = oracle.barcodes(w.dist, w.n, w.dim_max, w.threshold)
    with R.Rips(w.dist, w.n, w.dim_max, w.threshold) as g:
        g.compute()
        for d in range(0, w.dim_max + 1):
            _compare_dimension(g, o, d, f"{w.name} d={d}")
        if w.threshold == inf:   # P9: every column of a full complex gets a pivot, no essential class above dimension 0
            for d in range(1, w.dim_max + 1):
                assert g.stats(d)["n_essential"] == 0 and g.pivots(d)[0].numel() == comb(w.n - 1, d + 1)


def test_config3_dimension1_barcodes_and_dimension2_columns(R):
    """Config 3 (400-point random matrix).  Dimension 1 completely: the device reduction (3,118 columns, ~1.5e5
    additions, reduced columns of up to 10^6 entries) against the oracle's explicit reduction.  Dimension 2: stage 1
    and stage 2 with the TRUE clearing set (the pivots of dimension 1), checked by test_full_size_sampled on slices
    and here by the properties that hold at any size; its reduction is out of reach of any sparse Z/2 reduction at
    n = 400 (~10^13 entries to add), so it has no barcodes to compare."""
    import torch
    w = inputs.config(3)
    o = oracle.barcodes(w.dist, w.n, 1, w.threshold, explicit=True)
    with R.Rips(w.dist, w.n, 2, w.threshold) as g:
        g.dim0()
        g.stage1(1); g.stage2(1); g.reduce(1)
        for d in (0, 1):
            _compare_dimension(g, o, d, f"{w.name} d={d}")
        assert g.pivots(1)[0].numel() == comb(w.n - 1, 2) and g.stats(1)["n_essential"] == 0
        g.stage1(2); g.stage2(2)
        st = g.stats(2)
        assert st["n_cleared"] == comb(w.n - 1, 2) and st["n_columns"] == comb(w.n - 1, 3)      # P9
        assert st["n_apparent"] + st["n_nonapparent"] == st["n_columns"]
        at, as_ = g.apparent_pairs(2)
        assert bool((at[1:] > at[:-1]).all()) and torch.unique(as_).numel() == as_.numel()     # all t, all s distinct
        idx = torch.linspace(0, at.numel() - 1, 200).long()
        for t, s_ in zip(at[idx].tolist(), as_[idx].tolist()):                                  # zero persistence
            assert oracle.diameter(w.dist, t, 4, w.n) == oracle.diameter(w.dist, s_, 3, w.n)


def test_config2_lower_dimensions_complete(R):
    """Dimensions 1 and 2 of config 2 are small enough for the oracle to produce every array."""
    w = inputs.config(2)
    o = oracle.barcodes(w.dist, w.n, 2, w.threshold)
    with R.Rips(w.dist, w.n, 3, w.threshold) as g:
        g.dim0()
        for d in (1, 2):
            g.stage1(d); g.stage2(d); g.reduce(d)
            fd, fc = g.filtration(d)
            assert np.array_equal(fc.cpu().numpy().astype(np.uint64), o[d]["filt_cidx"])
            assert np.array_equal(fd.cpu().numpy().view(np.uint32), o[d]["filt_diam"].view(np.uint32))
            pt, ps = g.pivots(d)
            assert np.array_equal(pt.cpu().numpy().astype(np.uint64), o[d]["pivot_t"])
            assert np.array_equal(ps.cpu().numpy().astype(np.uint64), o[d]["pivot_s"])
            assert np.array_equal(g.barcodes(d).view(np.uint32), o[d]["bars"].reshape(-1, 2).view(np.uint32))


@pytest.mark.parametrize("n", [1000, 3000, 5792, 10000])
def test_second_workload_dim1_random_matrix(R, n):
    """SURVEY.md 8(f) item 4, the experiment of PAPER.md:719-729 as a sweep: dimension-1 apparent pairs of a random
    matrix without triangle inequality (a random permutation of 1..C(n,2) up to n = 5792, i.i.d. uniform fp32 above).
    (a) the apparent fraction against the closed form behind the paper's printed means (pin P11; the paper reports a
    very low variance); (b) on slices of the edges, the exact arrays against the oracle."""
    import math
    import torch
    w = inputs.second_workload(n)
    low = w.dist
    E = n * (n - 1) // 2
    with R.Rips(torch.from_numpy(low).cuda(), n, 1) as g:
        g.dim0()
        g.stage1(1)
        g.stage2(1)
        st = g.stats(1)
        assert st["n_candidates"] == E and st["n_cleared"] == n - 1 and st["n_columns"] == E - (n - 1)
        closed = 1 - (math.sqrt(math.pi) / 2) * math.exp(math.lgamma(n - 1) - math.lgamma(n - 0.5))
        assert abs(st["n_apparent"] / E - closed) < (3e-3 if n <= 1000 else 1e-3)
        z = oracle.dim0(low, n)
        pt, ps = g.pivots(0)
        assert np.array_equal(pt.cpu().numpy().astype(np.uint64), z["t"])
        at, as_ = g.apparent_pairs(1)
        nd, nc = g.nonapparent(1)
        assert bool((at[1:] > at[:-1]).all())
        for lo in (0, E // 2, E - 20000):
            hi = lo + 20000
            od, oc, _ = oracle.stage1(low, n, 1, inf, z["t"], lo, hi, sort=False)
            s2 = oracle.stage2(low, n, 1, od, oc)
            m = (as_ >= lo) & (as_ < hi)
            gs, order = torch.sort(as_[m])
            o_order = np.argsort(s2["app_s"], kind="stable")
            assert np.array_equal(gs.cpu().numpy().astype(np.uint64), s2["app_s"][o_order])
            assert np.array_equal(at[m][order].cpu().numpy().astype(np.uint64), s2["app_t"][o_order])
            m = (nc >= lo) & (nc < hi)
            assert np.array_equal(torch.sort(nc[m])[0].cpu().numpy().astype(np.uint64), np.sort(s2["non_cidx"]))


def test_compact_mode_with_dense_runs(R):
    """Thresholded input whose survivors come in long dense runs of the index space (two tight clusters far
    apart, threshold between the two scales): the estimate of the surviving share is low, so compact mode picks
    long chunks, the chunks inside a cluster overflow the staging, and the launch is repeated with short ones.
    The result must not depend on any of that."""
    import torch
    n = 400
    rng = np.random.default_rng(5)
    pts = rng.random((n, 3), dtype=np.float32) * 0.05
    pts[n // 2:] += 10.0
    low = inputs.euclidean_lower(pts)
    thr = 1.0
    z = oracle.dim0(low, n, thr)
    fd1, fc1, _ = oracle.stage1(low, n, 1, thr, z["t"])
    s21 = oracle.stage2(low, n, 1, fd1, fc1)
    red = oracle.reduce_columns(low, n, 1, thr, s21["non_cidx"], s21["app_t"], s21["app_s"])
    cleared2 = np.sort(np.concatenate([s21["app_t"], red["t"]]))
    od, oc, counts = oracle.stage1(low, n, 2, thr, cleared2)
    s2 = oracle.stage2(low, n, 2, od, oc)
    with R.Rips(low, n, 2, thr) as g:
        g.dim0()
        g.stage1(1); g.stage2(1); g.reduce(1)
        g.stage1(2); g.stage2(2)
        st = g.stats(2)
        assert st["n_slots"] == st["n_columns"]          # compact mode
        assert (st["n_columns"], st["n_removed_by_diameter"], st["n_cleared"]) == \
               (counts["kept"], counts["removed_by_diameter"], counts["cleared"])
        fd, fc = g.filtration(2)
        assert np.array_equal(fc.cpu().numpy().astype(np.uint64), oc)
        assert np.array_equal(fd.cpu().numpy().view(np.uint32), od.view(np.uint32))
        at, as_ = g.apparent_pairs(2)
        assert np.array_equal(at.cpu().numpy().astype(np.uint64), s2["app_t"])
        assert np.array_equal(as_.cpu().numpy().astype(np.uint64), s2["app_s"])
        nd, nc = g.nonapparent(2)
        assert np.array_equal(nc.cpu().numpy().astype(np.uint64), s2["non_cidx"])
