"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic (no simplex indexing, no diameters of
simplices, no sorting into filtration order, no pairing).  It only produces distance
matrices: the strict lower triangle, row-major, element (i > j) at position i*(i-1)/2 + j,
as float32 -- the layout `include/rips.h` documents for `rips_init`.

The five configurations are the ones BASELINE.json names; they stand in for the paper's
datasets, which are not available here.  Recipe: SURVEY.md section 8(d) and
DESIGN.md "Input recipe".  numpy.random.default_rng(seed) (PCG64) everywhere.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np

INF = float("inf")


@dataclass(frozen=True)
class Workload:
    name: str
    n: int
    dim_max: int
    threshold: float          # +inf = full complex
    dist: np.ndarray          # float32[n*(n-1)/2], strict lower triangle, row-major
    note: str = ""


def lower_from_square(sq: np.ndarray) -> np.ndarray:
    """Strict lower triangle of a square matrix, row-major: (1,0),(2,0),(2,1),(3,0),..."""
    n = sq.shape[0]
    i, j = np.tril_indices(n, k=-1)
    return np.ascontiguousarray(sq[i, j])


def square_from_lower(low: np.ndarray, n: int) -> np.ndarray:
    sq = np.zeros((n, n), dtype=low.dtype)
    i, j = np.tril_indices(n, k=-1)
    sq[i, j] = low
    sq[j, i] = low
    return sq


def euclidean_lower(points: np.ndarray) -> np.ndarray:
    """D[i][j] = fp32( sqrt( sum_k (double(x_ik) - double(x_jk))^2 ) ), lower triangle."""
    x = np.asarray(points, dtype=np.float64)
    n = x.shape[0]
    i, j = np.tril_indices(n, k=-1)
    diff = x[i] - x[j]
    d = np.sqrt(np.einsum("ij,ij->i", diff, diff))
    return d.astype(np.float32)


def enclosing_radius(low: np.ndarray, n: int) -> float:
    """min_i max_j D[i][j] over the fp32 matrix; an input value of cfg 5."""
    sq = square_from_lower(np.asarray(low, dtype=np.float32), n)
    return float(np.float32(sq.max(axis=1).min()))


# ---------------------------------------------------------------- point clouds / matrices

def cube_points(n: int, dim: int, seed: int) -> np.ndarray:
    return np.random.default_rng(seed).random((n, dim), dtype=np.float32)


def sphere_points(n: int, dim: int, seed: int) -> np.ndarray:
    g = np.random.default_rng(seed).standard_normal((n, dim))
    return (g / np.linalg.norm(g, axis=1, keepdims=True)).astype(np.float32)


def gaussian_points(n: int, dim: int, seed: int) -> np.ndarray:
    return np.random.default_rng(seed).standard_normal((n, dim)).astype(np.float32)


def random_matrix_lower(n: int, seed: int) -> np.ndarray:
    """i.i.d. Uniform(0,1) fp32 entries written directly in lower-triangle order."""
    return np.random.default_rng(seed).random(n * (n - 1) // 2, dtype=np.float32)


def permutation_matrix_lower(n: int, seed: int) -> np.ndarray:
    """A uniformly random permutation of 1..n(n-1)/2, exact in fp32 for n <= 5792."""
    e = n * (n - 1) // 2
    return (np.random.default_rng(seed).permutation(e) + 1).astype(np.float32)


def small_integer_lower(n: int, seed: int, hi: int = 4) -> np.ndarray:
    """Heavy-tie regime: entries i.i.d. in {1..hi}."""
    return np.random.default_rng(seed).integers(1, hi + 1, n * (n - 1) // 2).astype(np.float32)


def constant_lower(n: int, value: float = 1.0) -> np.ndarray:
    return np.full(n * (n - 1) // 2, value, dtype=np.float32)


def cyclic_lower(n: int) -> np.ndarray:
    """Integer cyclic metric D[i][j] = min(|i-j|, n-|i-j|): the regular n-gon up to a monotone rescaling."""
    i, j = np.tril_indices(n, k=-1)
    d = np.abs(i - j)
    return np.minimum(d, n - d).astype(np.float32)


def cross_polytope_lower(m: int) -> np.ndarray:
    """2m points, antipodal pairs (2k, 2k+1) at distance 2, every other pair at distance 1."""
    n = 2 * m
    i, j = np.tril_indices(n, k=-1)
    anti = (i // 2 == j // 2)
    return np.where(anti, 2.0, 1.0).astype(np.float32)


def descending_lower(n: int) -> np.ndarray:
    """PAPER.md:511-523 (Fig. 6): the edge with combinatorial index k gets the value C(n,2) - k."""
    e = n * (n - 1) // 2
    return (e - np.arange(e)).astype(np.float32)


# ---------------------------------------------------------------- the five configurations

def config(k: int, n: int | None = None) -> Workload:
    """BASELINE.json configs[k-1]; `n` overrides the point count (shadow configs, same distribution)."""
    if k == 1:
        n = n or 50
        return Workload(f"cfg1_cube3_n{n}", n, 2, INF, euclidean_lower(cube_points(n, 3, 0)),
                        "uniform in unit cube R^3, seed 0, full complex")
    if k == 2:
        n = n or 192
        return Workload(f"cfg2_sphere3_n{n}", n, 3, INF, euclidean_lower(sphere_points(n, 4, 1)),
                        "uniform on S^3 in R^4, seed 1, full complex")
    if k == 3:
        n = n or 400
        return Workload(f"cfg3_randmat_n{n}", n, 2, INF, random_matrix_lower(n, 2),
                        "i.i.d. U(0,1) distance matrix (no triangle inequality), seed 2, full complex")
    if k == 4:
        n = n or 1000
        return Workload(f"cfg4_cube3_thr_n{n}", n, 2, float(np.float32(0.15)),
                        euclidean_lower(cube_points(n, 3, 3)),
                        "uniform in unit cube R^3, seed 3, threshold 0.15")
    if k == 5:
        n = n or 512
        low = euclidean_lower(gaussian_points(n, 8, 4))
        return Workload(f"cfg5_gauss8_encl_n{n}", n, 2, enclosing_radius(low, n), low,
                        "standard Gaussian in R^8, seed 4, threshold = enclosing radius")
    if k == 6:
        return second_workload(n or 5000)
    if k == 7:
        # the regime of the paper's sparse option (o3 with a threshold that keeps 0.00038 % of the
        # possible simplices, Table 5): a point cloud under a threshold far below the enclosing radius.
        # C(1700, 4) = 3.5e11 candidate tetrahedra (a 43 GB clearing bitmap, seconds of enumeration for the dense path,
        # hours for the oracle's Algorithm 7); the complex itself has ~3.4e4 edges.  1700 is about the largest n whose
        # reduction entries of dimension 3 (key + row index) still fit 64 bits.
        n = n or 1700
        return Workload(f"cfg7_sparse_cube3_n{n}", n, 3, float(np.float32(0.1777 * (1700.0 / n) ** (1.0 / 3.0))),
                        euclidean_lower(cube_points(n, 3, 5)),
                        "uniform in unit cube R^3, seed 5, threshold for a mean degree of ~40: sparse path only")
    raise ValueError(f"no config {k}")


def second_workload(n: int, seed: int = 7) -> Workload:
    """The experiment of PAPER.md:719-729 (section 6.6, Fig. 13): dimension-1 apparent pairs of a random distance
    matrix with no triangle inequality.  n <= 5792: a uniformly random permutation of 1..n(n-1)/2 (exact in fp32);
    above that the integers are no longer exact in fp32, so i.i.d. Uniform(0,1) fp32 entries are used (a few tied
    values among 10^8: the closed form of the apparent fraction assumes none and is off by far less than its own
    sampling noise)."""
    if n <= 5792:
        low = permutation_matrix_lower(n, seed)
        note = "uniformly random permutation matrix (PAPER.md:719)"
    else:
        low = random_matrix_lower(n, seed)
        note = "i.i.d. U(0,1) fp32 distance matrix (permutation values are not exact in fp32 beyond n = 5792)"
    return Workload(f"sec66_randmat_n{n}", n, 1, INF, low, note + ", dimension 1 only, full complex")


def n_choose_k(n: int, k: int) -> int:
    """Only for sizing buffers and reporting counts in the harness."""
    return math.comb(n, k) if 0 <= k <= n else 0
