"""ORACLE tier O1 -- brute force, straight from the definitions.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import anything under oracle/.  Nothing here is shared with, or imported by, the CUDA path.

What it does (tiny inputs only, n <~ 14; pure Python loops):
  * every simplex of dimension <= dim_max+1 as a sorted vertex tuple
  * cidx by Eq. 2 literally
  * diameter = max pairwise distance, Eq. 1
  * the simplex-wise filtration order: diameter up, dimension up, cidx DOWN
  * the explicit boundary matrix over Z/2 and Algorithm 1 (standard reduction) PAPER.md:99-121
  * apparent pairs by Definition 5 literally (oldest cofacet / youngest facet) PAPER.md:256-258

It never uses the Apparent Pairs Lemma (Lemma 7), clearing, cohomology or implicit matrices, so
that the C oracle (oracle/rips_oracle.c), which does, can be checked against it.

Distances are handled as Python floats converted from float32 (exact), so comparisons are the
float32 comparisons.
"""
from __future__ import annotations

from itertools import combinations
from math import comb, inf


def dist_lookup(low, n):
    """low: strict lower triangle, (i>j) at i*(i-1)/2+j.  Returns d(i,j)."""
    vals = [float(x) for x in low]
    assert len(vals) == n * (n - 1) // 2

    def d(i, j):
        if i == j:
            return 0.0
        if i < j:
            i, j = j, i
        return vals[i * (i - 1) // 2 + j]
    return d


def cidx(verts):
    """Eq. 2: (v_d > ... > v_0) -> C(v_d, d+1) + ... + C(v_0, 1)."""
    vs = sorted(verts)                       # v_0 < v_1 < ... < v_d
    return sum(comb(v, k + 1) for k, v in enumerate(vs))


def diameter(verts, d):
    """Eq. 1: max pairwise distance; a vertex has diameter 0."""
    return max((d(a, b) for a, b in combinations(verts, 2)), default=0.0)


def filtration(low, n, top_dim, threshold=inf):
    """All simplices of dimension <= top_dim with diam <= threshold, in the order of PAPER.md:77-79.

    Returns a list of (diam, dim, cidx, verts) sorted by (diam asc, dim asc, cidx desc)."""
    d = dist_lookup(low, n)
    simplices = []
    for k in range(1, top_dim + 2):          # k vertices, dimension k-1
        for verts in combinations(range(n), k):
            dm = diameter(verts, d)
            if dm <= threshold:              # inclusive: PAPER.md:65
                simplices.append((dm, k - 1, cidx(verts), verts))
    simplices.sort(key=lambda s: (s[0], s[1], -s[2]))
    return simplices


def standard_reduction(simplices):
    """Algorithm 1 on the explicit boundary matrix.  Returns (pairs, zero_columns).

    pairs: list of (row_position, col_position), positions in the filtration order."""
    pos = {(s[1], s[2]): p for p, s in enumerate(simplices)}
    columns = []
    for (_, dim, _, verts) in simplices:
        if dim == 0:
            columns.append(set())
        else:
            columns.append({pos[(dim - 1, cidx(f))] for f in combinations(verts, dim)})
    low_to_col = {}
    pairs = []
    zero = []
    for j, col in enumerate(columns):
        col = set(col)
        while col and max(col) in low_to_col:
            col ^= columns[low_to_col[max(col)]]          # column k + column j over Z/2
        columns[j] = col
        if col:
            low_to_col[max(col)] = j
            pairs.append((max(col), j))
        else:
            zero.append(j)
    return pairs, zero


def persistence(low, n, dim_max, threshold=inf):
    """Persistence pairs and bars of H_0..H_dim_max of the Rips filtration, by Algorithm 1.

    Returns dict d -> {"pairs": sorted [(cidx_birth, cidx_death)], "essential": sorted [cidx_birth],
                       "bars": sorted [(birth, death)] with zero-length bars dropped, death=inf for essential}."""
    sx = filtration(low, n, dim_max + 1, threshold)
    pairs, zero = standard_reduction(sx)
    out = {d: {"pairs": [], "essential": [], "bars": []} for d in range(dim_max + 1)}
    paired_rows = set()
    for (r, c) in pairs:
        paired_rows.add(r)
        d = sx[r][1]
        if d <= dim_max:
            out[d]["pairs"].append((sx[r][2], sx[c][2]))
            if sx[r][0] != sx[c][0]:
                out[d]["bars"].append((sx[r][0], sx[c][0]))
    for j in zero:                            # zero column and never a pivot row: essential class
        d = sx[j][1]
        if j not in paired_rows and d <= dim_max:
            out[d]["essential"].append(sx[j][2])
            out[d]["bars"].append((sx[j][0], inf))
    for d in out:
        out[d]["pairs"].sort()
        out[d]["essential"].sort()
        out[d]["bars"].sort()
    return out


def apparent_pairs(low, n, d, threshold=inf):
    """Definition 5 literally, on the complex of all simplices with diam <= threshold.

    For each d-simplex s that has a cofacet: t = the cofacet of s that comes first in the
    filtration order ("oldest"); (s,t) is apparent iff s is the facet of t that comes last
    ("youngest").  Returns sorted [(cidx_t, cidx_s)]."""
    dist = dist_lookup(low, n)

    def key(verts):                           # position in the order of PAPER.md:77-79
        return (diameter(verts, dist), len(verts) - 1, -cidx(verts))

    out = []
    for s in combinations(range(n), d + 1):
        if diameter(s, dist) > threshold:
            continue
        cof = [tuple(sorted(s + (v,))) for v in range(n) if v not in s]
        cof = [t for t in cof if diameter(t, dist) <= threshold]
        if not cof:
            continue
        t = min(cof, key=key)                 # oldest cofacet
        facets = list(combinations(t, d + 1))
        youngest = max(facets, key=key)       # youngest facet
        if tuple(sorted(youngest)) == tuple(sorted(s)):
            out.append((cidx(t), cidx(s)))
    out.sort()
    return out


def coboundary_columns(low, n, d, threshold=inf, cleared=()):
    """The columns of the dimension-d coboundary matrix after filtering (Algorithms 7-8), as the
    definition states them: all d-simplices with diam <= threshold that are not in `cleared`,
    sorted by decreasing diameter, then increasing cidx.
    Returns [(diam, cidx)]."""
    dist = dist_lookup(low, n)
    cleared = set(cleared)
    cols = []
    for s in combinations(range(n), d + 1):
        dm = diameter(s, dist)
        c = cidx(s)
        if dm <= threshold and c not in cleared:
            cols.append((dm, c))
    cols.sort(key=lambda x: (-x[0], x[1]))
    return cols


def connected_components(low, n, threshold):
    """Independent check for Betti_0 of the threshold graph: plain BFS."""
    dist = dist_lookup(low, n)
    seen = [False] * n
    comps = 0
    for s in range(n):
        if seen[s]:
            continue
        comps += 1
        stack = [s]
        seen[s] = True
        while stack:
            a = stack.pop()
            for b in range(n):
                if not seen[b] and dist(a, b) <= threshold:
                    seen[b] = True
                    stack.append(b)
    return comps
