"""GPU parity: the CUDA path, called through the C ABI (paper_2003_07989_b200.rips), against the CPU
oracle (oracle/), element by element and bit-exact, on the same seeded inputs.  Every output is
integer / index data or a selected fp32 input value, so the tolerance is zero."""
from math import comb, inf

import numpy as np
import pytest

from oracle import oracle
from paper_2003_07989_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def R():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2003_07989_b200 import rips
    rips.lib()
    return rips


def _np(t):
    return t.cpu().numpy()


def check_against_oracle(R, low, n, dim_max, thr=inf, what="", mode=None):
    o = oracle.barcodes(low, n, dim_max, thr)
    with R.Rips(low, n, dim_max, thr) as g:
        if mode is not None:
            g.set_mode(mode)
        g.compute()
        # dimension 0
        pt, ps = g.pivots(0)
        assert np.array_equal(_np(pt).astype(np.uint64), o[0]["pivot_t"]), what
        assert np.array_equal(_np(ps).astype(np.uint64), o[0]["pivot_s"]), what
        assert np.array_equal(g.barcodes(0), o[0]["bars"].reshape(-1, 2)), what
        for d in range(1, dim_max + 1):
            tag = f"{what} d={d}"
            fd, fc = g.filtration(d)
            assert np.array_equal(_np(fc).astype(np.uint64), o[d]["filt_cidx"]), tag
            assert np.array_equal(_np(fd).view(np.uint32), o[d]["filt_diam"].view(np.uint32)), tag
            at, as_ = g.apparent_pairs(d)
            assert np.array_equal(_np(at).astype(np.uint64), o[d]["app_t"]), tag
            assert np.array_equal(_np(as_).astype(np.uint64), o[d]["app_s"]), tag
            nd, nc = g.nonapparent(d)
            assert np.array_equal(_np(nc).astype(np.uint64), o[d]["non_cidx"]), tag
            assert np.array_equal(_np(nd).view(np.uint32), o[d]["non_diam"].view(np.uint32)), tag
            pt, ps = g.pivots(d)
            assert np.array_equal(_np(pt).astype(np.uint64), o[d]["pivot_t"]), tag
            assert np.array_equal(_np(ps).astype(np.uint64), o[d]["pivot_s"]), tag
            assert np.array_equal(g.barcodes(d).view(np.uint32), o[d]["bars"].reshape(-1, 2).view(np.uint32)), tag
            st = g.stats(d)
            c = o[d]["counts"]
            assert st["n_candidates"] == comb(n, d + 1)
            assert (st["n_columns"], st["n_removed_by_diameter"], st["n_cleared"]) == \
                   (c["kept"], c["removed_by_diameter"], c["cleared"]), tag
            assert st["n_apparent"] == o[d]["app_t"].size and st["n_nonapparent"] == o[d]["non_cidx"].size
            assert st["n_essential"] == o[d]["essential"].size
            # a10: lookup of every pivot row, and of rows that are not pivots
            if o[d]["pivot_t"].size:
                q = o[d]["pivot_t"][:: max(1, o[d]["pivot_t"].size // 500)]
                got = _np(g.pivot_lookup(d, q.astype(np.int64)))
                want = o[d]["pivot_s"][:: max(1, o[d]["pivot_t"].size // 500)].astype(np.int64)
                assert np.array_equal(got, want), tag
            allrows = np.arange(min(comb(n, d + 2), 2000), dtype=np.int64)
            isp = np.isin(allrows.astype(np.uint64), o[d]["pivot_t"])
            got = _np(g.pivot_lookup(d, allrows))
            assert np.array_equal(got >= 0, isp), tag


@pytest.mark.parametrize("k,n", [(1, 12), (2, 14), (3, 16), (4, 40), (5, 18), (1, 50), (2, 40), (3, 60), (5, 48)])
def test_shadow_configs(R, k, n):
    w = inputs.config(k, n)
    thr = w.threshold if k != 5 else inputs.enclosing_radius(w.dist, n)
    if k == 4:
        thr = float(np.float32(np.quantile(w.dist, 0.25)))
    check_against_oracle(R, w.dist, n, w.dim_max, thr, w.name)


@pytest.mark.parametrize("k,n,q", [(1, 40, 0.1), (2, 30, 0.3), (3, 50, 0.05), (4, 120, 0.04), (5, 48, 0.5), (1, 70, 1.0), (4, 300, 0.02)])
def test_sparse_path_shadow_configs(R, k, n, q):
    """The sparse path (RIPS_MODE_SPARSE: neighbour lists, simplices of dimension d from those of dimension d-1,
    cofacets from common neighbours) on the five distributions under thresholds that admit a share q
    of the edges (q = 1: the full complex through the sparse path): every array against the oracle, and the dense path
    on the same input gives the same counts."""
    w = inputs.config(k, n)
    thr = inf if q == 1.0 else float(np.float32(np.quantile(w.dist, q)))
    dm = w.dim_max if n <= 120 else 2
    check_against_oracle(R, w.dist, n, dm, thr, f"sparse {w.name} q={q}", mode="sparse")
    check_against_oracle(R, w.dist, n, dm, thr, f"dense {w.name} q={q}", mode="dense")


@pytest.mark.parametrize("seed", range(12))
def test_sparse_path_randomized(R, seed):
    rng = np.random.default_rng(3000 + seed)
    n = int(rng.integers(5, 90))
    dim_max = int(rng.integers(1, 4)) if n <= 40 else int(rng.integers(1, 3))
    regime = seed % 3
    if regime == 0:
        low = inputs.random_matrix_lower(n, 150 + seed)
    elif regime == 1:
        low = inputs.small_integer_lower(n, 160 + seed, hi=int(rng.integers(2, 9)))
    else:
        low = inputs.euclidean_lower(inputs.cube_points(n, int(rng.integers(1, 4)), 170 + seed))
    q = float(rng.choice([1.0, 0.6, 0.3, 0.1, 0.03, 0.0]))
    thr = inf if q == 1.0 else float(np.float32(np.quantile(low, q)))
    check_against_oracle(R, low, n, dim_max, thr, f"sparse seed {seed}: n={n} dim_max={dim_max} regime={regime} q={q}", mode="sparse")


def test_stress_build(R):
    """The chained scans (decoupled look-back of the sort, of compact mode, of the sparse path's scan, of the edge
    ranking) and the lock-free reduction under shuffled schedules: the library built with -DRIPS_STRESS (sort tiles of
    512 records instead of 5120, short chunks, pseudo-random delays in front of every publication) must produce the
    same arrays.  compute-sanitizer is not available on this pool; this is the litmus test in its place."""
    import torch
    from paper_2003_07989_b200 import build
    try:
        R.use_library(build.build_stress())
        rng = np.random.default_rng(5)
        for n, lo, hi in [(513, 0, 8), (70001, 3, 19), (300007, 0, 24), (1 << 18, 40, 64)]:
            a = rng.integers(0, 1 << 62, n, dtype=np.int64)
            t = torch.from_numpy(a).cuda()
            R.rips_sort_u64(t, lo, hi)
            u = a.view(np.uint64)
            key = (u >> np.uint64(lo)) & np.uint64((1 << (hi - lo)) - 1)
            assert np.array_equal(t.cpu().numpy().view(np.uint64), u[np.argsort(key, kind="stable")]), (n, lo, hi)
        for rep in range(3):
            w = inputs.config(4, 200)
            thr = float(np.float32(np.quantile(w.dist, 0.12)))
            check_against_oracle(R, w.dist, w.n, 2, thr, "stress compact", mode="dense")
            check_against_oracle(R, w.dist, w.n, 2, thr, "stress sparse", mode="sparse")
            w = inputs.config(3, 70)
            check_against_oracle(R, w.dist, w.n, 2, inf, "stress reduction")
            w = inputs.config(2, 40)
            check_against_oracle(R, w.dist, w.n, 3, inf, "stress slot")
        # the stress build sends the triangles of more than ~130 points to the general kernel in slot mode, and builds
        # the block maxima for every input: that kernel's scan guided by them (in the product build: n >= 2048 with
        # tables that do not fit shared memory)
        w = inputs.config(2, 140)
        check_against_oracle(R, w.dist, w.n, 2, inf, "stress general kernel, slot mode, block maxima")
    finally:
        R.use_library(None)


def test_mode_is_fixed_by_the_first_stage1(R):
    w = inputs.config(1, 20)
    with R.Rips(w.dist, w.n, 1) as g:
        g.dim0()
        g.stage1(1)
        with pytest.raises(R.RipsError) as e:
            g.set_mode("sparse")
        assert e.value.code == R.RIPS_EINVAL


@pytest.mark.parametrize("name", ["constant", "cyclic", "cross", "descending", "smallint", "zeros"])
def test_degenerate_value_patterns(R, name):
    n = 13
    low = {"constant": inputs.constant_lower(n), "cyclic": inputs.cyclic_lower(n),
           "cross": inputs.cross_polytope_lower(6), "descending": inputs.descending_lower(n),
           "smallint": inputs.small_integer_lower(n, 7),
           "zeros": inputs.euclidean_lower(np.repeat(inputs.cube_points(5, 2, 1), 3, axis=0)[:n])}[name]
    nn = 12 if name == "cross" else n
    check_against_oracle(R, low, nn, 3 if name != "zeros" else 2, inf, name)


@pytest.mark.parametrize("n", [1, 2, 3, 4])
def test_tiny_n(R, n):
    low = inputs.random_matrix_lower(n, 3)
    check_against_oracle(R, low, n, 2, inf, f"n={n}")
    check_against_oracle(R, low + 1.0, n, 2, 0.5, f"n={n} below every distance")


@pytest.mark.parametrize("n", [5, 8, 15, 16, 17, 20, 33, 47])
def test_queue_of_open_scans_boundaries(R, n):
    """The slot kernel's queue of open cofacet scans around its boundaries: fewer vertices than
    a drained lane tests on its own (n < 16: no warp-cooperative scan at all), exactly as many, a few more (one partial
    group of 32 behind them).  Random matrices: their scans are long, so most lanes are queued, the
    queue fills and is drained in the middle of a slab, and many lanes are still open after the twelve vertices; the
    matrix with heavy ties makes columns without any cofacet of equal diameter rare and irregular pairs common."""
    check_against_oracle(R, inputs.random_matrix_lower(n, 400 + n), n, 3, inf, f"queue n={n} random matrix")
    check_against_oracle(R, inputs.small_integer_lower(n, 500 + n, hi=3), n, 3, inf, f"queue n={n} ties")


def test_threshold_sweep(R):
    w = inputs.config(1, 30)
    for q in (0.0, 0.1, 0.5, 0.9, 1.0):
        thr = float(np.float32(np.quantile(w.dist, q)))
        check_against_oracle(R, w.dist, 30, 2, thr, f"q={q}")


def test_config1_full(R):
    w = inputs.config(1)
    check_against_oracle(R, w.dist, w.n, w.dim_max, w.threshold, w.name)


def test_sort_primitive(R):
    import torch
    rng = np.random.default_rng(11)
    for n, lo, hi in [(1, 0, 8), (2, 3, 20), (1000, 0, 64), (8192, 5, 22), (8193, 0, 9), (100003, 13, 30),
                      (1 << 20, 40, 57), (300007, 0, 1),
                      # around the tile of 256 x 20 records and the look-back batch of 8 tiles
                      (5119, 0, 8), (5120, 2, 10), (5121, 0, 16), (5120 * 9, 7, 15), (5120 * 10 + 1, 0, 15),
                      (5120 * 17 - 1, 20, 27), (3000017, 3, 19)]:
        a = rng.integers(0, 1 << 63, n, dtype=np.int64) * 2 + rng.integers(0, 2, n, dtype=np.int64)
        if n == 100003:
            a[:] = a[0]                       # all keys equal: must come back untouched (stability)
            a += np.arange(n) << 32
        t = torch.from_numpy(a).cuda()
        R.rips_sort_u64(t, lo, hi)
        u = a.view(np.uint64)
        key = (u >> np.uint64(lo)) & np.uint64((1 << (hi - lo)) - 1)
        want = u[np.argsort(key, kind="stable")]
        assert np.array_equal(t.cpu().numpy().view(np.uint64), want), (n, lo, hi)


def test_invalid_inputs(R):
    bad = np.array([1.0, np.nan, 2.0], dtype=np.float32)
    for arr in (bad, np.array([1.0, -2.0, 2.0], dtype=np.float32), np.array([1.0, np.inf, 2.0], dtype=np.float32)):
        with pytest.raises(R.RipsError) as e:
            R.Rips(arr, 3, 1)
        assert e.value.code == R.RIPS_EINVAL
    with pytest.raises(R.RipsError):
        R.Rips(np.ones(3, dtype=np.float32), 3, 7)
    with pytest.raises(R.RipsError):
        R.Rips(np.ones(3, dtype=np.float32), 3, 1, float("nan"))
    g = R.Rips(np.ones(3, dtype=np.float32), 3, 1)
    with pytest.raises(R.RipsError):
        g.stage2(1)                           # stage 1 has not run
    neg0 = np.array([-0.0, 1.0, 1.0], dtype=np.float32)
    check_against_oracle(R, np.abs(neg0), 3, 1)
    with R.Rips(neg0, 3, 1) as h:
        h.compute()
        assert np.array_equal(h.barcodes(0), oracle.barcodes(np.abs(neg0), 3, 1)[0]["bars"].reshape(-1, 2))


def test_scale_row_entry_points(R):
    """rips_stage1 / rips_stage2 at d = dim_max + 1 (the scale row): the same
    arrays the oracle produces for that dimension."""
    w = inputs.config(2, 36)
    o = oracle.barcodes(w.dist, w.n, 3, w.threshold)
    with R.Rips(w.dist, w.n, 2, w.threshold) as g:
        g.compute()
        g.stage1(3)
        g.stage2(3)
        fd, fc = g.filtration(3)
        assert np.array_equal(_np(fc).astype(np.uint64), o[3]["filt_cidx"])
        assert np.array_equal(_np(fd).view(np.uint32), o[3]["filt_diam"].view(np.uint32))
        at, as_ = g.apparent_pairs(3)
        assert np.array_equal(_np(at).astype(np.uint64), o[3]["app_t"])
        assert np.array_equal(_np(as_).astype(np.uint64), o[3]["app_s"])
        nd, nc = g.nonapparent(3)
        assert np.array_equal(_np(nc).astype(np.uint64), o[3]["non_cidx"])
        st = g.stats(3)
        assert st["n_cleared"] == o[2]["pivot_t"].size
        # re-running the stages gives the same arrays (bench.py's step)
        g.stage1(3); g.stage2(3)
        at2, _ = g.apparent_pairs(3)
        assert bool((at2 == at).all())


def test_dim_max_4(R):
    """The widest instantiations (columns of 5 vertices, cofacets of 6), every array against the oracle."""
    w = inputs.config(2, 13)
    check_against_oracle(R, w.dist, w.n, 4, inf, "dim_max 4")
    w = inputs.config(1, 12)
    thr = float(np.float32(np.quantile(w.dist, 0.6)))
    check_against_oracle(R, w.dist, w.n, 4, thr, "dim_max 4 with a threshold")


def test_more_than_256_vertices(R):
    """n > 256: vertex fields of 9 bits and a pair partition of two radix passes."""
    w = inputs.config(1, 300)
    check_against_oracle(R, w.dist, w.n, 1, inf, "n = 300, dimension 1")
    thr = float(np.float32(np.quantile(w.dist, 0.05)))
    check_against_oracle(R, w.dist, w.n, 2, thr, "n = 300, dimension 2, 5 % of the edges")


def _everything(g, D):
    out = [g.barcodes(0)]
    for d in range(1, D + 1):
        out += [g.filtration(d), g.apparent_pairs(d), g.nonapparent(d), g.pivots(d), g.barcodes(d)]
    return out


def test_caller_workspace(R):
    """rips_init with a caller's workspace of rips_workspace_bytes: rips_compute and every accessor fit, the
    context's device bytes are that workspace and never change, the results are the library-owned ones."""
    import torch
    for k, n in [(1, 50), (2, 60), (5, 120), (4, 200)]:
        w = inputs.config(k, n)
        thr = w.threshold if k != 5 else inputs.enclosing_radius(w.dist, n)
        size = R.rips_workspace_bytes(n, w.dim_max)
        ws = torch.empty(size, dtype=torch.uint8, device="cuda")
        with R.Rips(w.dist, n, w.dim_max, thr, workspace=ws) as g, R.Rips(w.dist, n, w.dim_max, thr) as h:
            assert g.device_bytes() == size // 256 * 256
            g.compute(); h.compute()
            a, b = _everything(g, w.dim_max), _everything(h, w.dim_max)
            assert g.device_bytes() == size // 256 * 256
            used, peak = g.workspace_in_use()
            assert 0 < used <= peak <= size
            for x, y in zip(a, b):
                if isinstance(x, tuple):
                    assert all(bool((p == q).all()) for p, q in zip(x, y))
                else:
                    assert np.array_equal(x, y)
            # the hot path again on the same context: no growth
            for d in range(1, w.dim_max + 1):
                g.stage1(d); g.stage2(d)
            assert g.workspace_in_use()[1] <= size


def test_workspace_too_small(R):
    """A workspace that cannot hold the computation: RIPS_ENOMEM with the size that would have fitted, nothing
    crashes, and a workspace of the reported size gets further."""
    import torch
    w = inputs.config(2, 60)
    with pytest.raises(R.RipsError) as e:
        R.Rips(w.dist, w.n, w.dim_max, w.threshold, workspace=8192)          # not even the set-up
    assert e.value.code == R.RIPS_ENOMEM and R.rips_last_required_bytes() > 8192
    with pytest.raises(R.RipsError) as e:
        R.Rips(w.dist, w.n, w.dim_max, w.threshold, workspace=torch.empty(5000, dtype=torch.uint8, device="cuda")[1:])
    assert e.value.code == R.RIPS_EINVAL                                    # misaligned
    size = 2 << 20                                                          # the set-up fits, dimension 3 does not
    for _ in range(40):
        g = R.Rips(w.dist, w.n, w.dim_max, w.threshold, workspace=size)
        try:
            g.compute()
            _everything(g, w.dim_max)
            break
        except R.RipsError as err:
            assert err.code == R.RIPS_ENOMEM
            need = R.rips_last_required_bytes()
            assert need > size
            size = max(need, size + size // 2)   # the report covers the request that failed, not the ones after it
        finally:
            g.free()
    else:
        raise AssertionError("the reported sizes never sufficed")
    assert size <= 2 * R.rips_workspace_bytes(w.n, w.dim_max)     # (the loop grows geometrically)
    o = oracle.barcodes(w.dist, w.n, w.dim_max, w.threshold)
    with R.Rips(w.dist, w.n, w.dim_max, w.threshold, workspace=size) as g:
        g.compute()
        for d in range(1, w.dim_max + 1):
            assert np.array_equal(g.barcodes(d).view(np.uint32), o[d]["bars"].reshape(-1, 2).view(np.uint32))


def test_two_contexts_interleaved_and_repeated_stages(R):
    """Contexts are independent (own streams, own buffers); stages may be repeated in any valid order."""
    wa, wb = inputs.config(1, 30), inputs.config(3, 28)
    oa = oracle.barcodes(wa.dist, wa.n, 2, wa.threshold)
    ob = oracle.barcodes(wb.dist, wb.n, 2, wb.threshold)
    a = R.Rips(wa.dist, wa.n, 2, wa.threshold)
    b = R.Rips(wb.dist, wb.n, 2, wb.threshold)
    a.dim0(); b.dim0()
    for d in (1, 2):
        a.stage1(d); b.stage1(d); b.stage2(d); a.stage2(d)
        a.stage2(d)                       # nothing new to partition: a no-op
        b.stage1(d); b.stage2(d)          # recomputed from scratch
        a.reduce(d); b.reduce(d)
    for g, o in ((a, oa), (b, ob)):
        for d in (1, 2):
            pt, ps = g.pivots(d)
            assert np.array_equal(_np(pt).astype(np.uint64), o[d]["pivot_t"])
            assert np.array_equal(_np(ps).astype(np.uint64), o[d]["pivot_s"])
            assert np.array_equal(g.barcodes(d).view(np.uint32), o[d]["bars"].reshape(-1, 2).view(np.uint32))
    a.free(); b.free()


def test_import_pivots(R):
    """rips_import_pivots installs a reduction done elsewhere (here: the oracle's) and rejects unsorted rows."""
    w = inputs.config(2, 20)
    o = oracle.barcodes(w.dist, w.n, 2, w.threshold)
    with R.Rips(w.dist, w.n, 2, w.threshold) as g:
        g.dim0(); g.stage1(1); g.stage2(1)
        order = np.argsort(o[1]["red_t"])
        with pytest.raises(R.RipsError) as e:
            g.import_pivots(1, o[1]["red_t"][order][::-1], o[1]["red_s"][order][::-1])
        if o[1]["red_t"].size > 1:
            assert e.value.code == R.RIPS_EINVAL
        g.import_pivots(1, o[1]["red_t"][order], o[1]["red_s"][order])
        pt, ps = g.pivots(1)
        assert np.array_equal(_np(pt).astype(np.uint64), o[1]["pivot_t"])
        g.stage1(2); g.stage2(2)
        fd, fc = g.filtration(2)
        assert np.array_equal(_np(fc).astype(np.uint64), o[2]["filt_cidx"])


@pytest.mark.parametrize("seed", range(24))
def test_randomized_shapes(R, seed):
    """Seeded random shapes: n, dimension, value regime (distinct reals, heavy ties, clustered points) and
    threshold all vary; every array against the oracle."""
    rng = np.random.default_rng(1000 + seed)
    n = int(rng.integers(5, 70))
    dim_max = int(rng.integers(1, 4)) if n <= 40 else int(rng.integers(1, 3))
    regime = seed % 4
    if regime == 0:
        low = inputs.random_matrix_lower(n, 50 + seed)
    elif regime == 1:
        low = inputs.small_integer_lower(n, 60 + seed, hi=int(rng.integers(2, 9)))
    elif regime == 2:
        pts = rng.random((n, 3), dtype=np.float32) * 0.1
        pts[rng.random(n) < 0.5] += 5.0
        low = inputs.euclidean_lower(pts)
    else:
        low = inputs.euclidean_lower(inputs.cube_points(n, int(rng.integers(1, 5)), 70 + seed))
    q = float(rng.choice([1.0, 1.0, 0.9, 0.5, 0.2, 0.05]))
    thr = inf if q == 1.0 else float(np.float32(np.quantile(low, q)))
    check_against_oracle(R, low, n, dim_max, thr, f"seed {seed}: n={n} dim_max={dim_max} regime={regime} q={q}")
