"""CPU oracle for the Mantel test (Pearson and Spearman) -- TEST INFRASTRUCTURE ONLY.

Only tests/ and bench.py's cpu_baseline leg may import this module; it imports nothing from the CUDA package.

What it follows.  PAPER.md:41 (section III): "The Mantel test is often used to check for correlations between two
distance matrices ... Correlation can be computed using either Pearson's product-moment correlation coefficient or
Spearman's rank correlation coefficient."  The paper gives no formula (it cites scikit-bio); this is the plain textbook
definition of the test, written out in fp64 with no shortcut (readings M1-M4):

  * the data are the N(N-1)/2 entries above the diagonal of the two symmetric hollow matrices X and Y (each unordered
    pair of objects once, diagonal excluded);
  * r = Pearson's product-moment correlation of those two vectors (two-pass: subtract the means, then the ratio of the
    cross product to the product of the norms);
  * for each permutation pi_k of the objects, rows AND columns of X are permuted together, X^pi[i][j] = X[pi(i)][pi(j)],
    and r_k = Pearson(upper(X^pi_k), upper(Y)); the permutations are inputs (no random numbers are drawn here);
  * p = (count + 1) / (K + 1) with count = #{k: |r_k| >= |r|} (two-sided), #{r_k >= r} (greater), #{r_k <= r} (less);
  * a matrix with zero variance gives r = 0 (reading M4; Pearson is undefined there).
"""
from __future__ import annotations

import numpy as np


def square_from_condensed(c: np.ndarray, n: int) -> np.ndarray:
    """Symmetric hollow n x n matrix from the row-major upper triangle (scipy squareform order)."""
    c = np.asarray(c, dtype=np.float64)
    assert c.shape == (n * (n - 1) // 2,)
    m = np.zeros((n, n), dtype=np.float64)
    iu = np.triu_indices(n, k=1)
    m[iu] = c
    m[(iu[1], iu[0])] = c
    return m


def upper(m: np.ndarray) -> np.ndarray:
    return m[np.triu_indices(m.shape[0], k=1)]


def pearson(a: np.ndarray, b: np.ndarray) -> float:
    """Two-pass product-moment correlation of two equally long vectors; 0 if either has zero variance (M4)."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    da = a - a.mean()
    db = b - b.mean()
    den = np.sqrt(np.sum(da * da) * np.sum(db * db))
    return float(np.sum(da * db) / den) if den > 0.0 else 0.0


def mantel_pearson(x_condensed, y_condensed, n: int, perms):
    """Returns (r, p_two_sided, p_greater, p_less, r_perm[K]).  perms: [K, n] integer array of permutations."""
    X = square_from_condensed(x_condensed, n)
    y = np.asarray(y_condensed, dtype=np.float64)
    r = pearson(upper(X), y)
    perms = np.asarray(perms, dtype=np.int64).reshape(-1, n)
    rk = np.empty(len(perms), dtype=np.float64)
    for k, pi in enumerate(perms):
        Xp = X[pi][:, pi]                       # X^pi[i][j] = X[pi(i)][pi(j)]
        rk[k] = pearson(upper(Xp), y)
    K = len(perms)
    p_two = (np.sum(np.abs(rk) >= abs(r)) + 1.0) / (K + 1.0)
    p_gr = (np.sum(rk >= r) + 1.0) / (K + 1.0)
    p_le = (np.sum(rk <= r) + 1.0) / (K + 1.0)
    return r, float(p_two), float(p_gr), float(p_le), rk


# ---------------------------------------------------------------------------------------------------------------------
# Spearman variant.  PAPER.md:41 (section III): "... or Spearman's rank correlation coefficient"; "the
# Spearman variety requires about 18 minutes".  Textbook definition (readings M5-M6): Spearman's rho of two
# vectors is Pearson's correlation of their RANKS, ties receiving the average of the ranks they span (1-based,
# "fractional ranking").  The Mantel test is otherwise unchanged: for every permutation the upper triangle of the
# permuted X is ranked again and correlated with the ranks of y.
def average_ranks(a: np.ndarray) -> np.ndarray:
    """1-based ranks of a vector; a run of equal values gets the mean of the positions it occupies.  Plain loop over
    the sorted order (no scipy): obviously correct, O(n log n)."""
    a = np.asarray(a, dtype=np.float64)
    order = np.argsort(a, kind="stable")
    ranks = np.empty(a.shape[0], dtype=np.float64)
    s = 0
    n = a.shape[0]
    while s < n:
        e = s
        while e + 1 < n and a[order[e + 1]] == a[order[s]]:
            e += 1
        ranks[order[s:e + 1]] = 0.5 * (s + e) + 1.0            # positions s..e (0-based) -> ranks s+1..e+1, averaged
        s = e + 1
    return ranks


def spearman(a: np.ndarray, b: np.ndarray) -> float:
    return pearson(average_ranks(a), average_ranks(b))


def mantel_spearman(x_condensed, y_condensed, n: int, perms):
    """Returns (rho, p_two_sided, p_greater, p_less, rho_perm[K]); same conventions as mantel_pearson."""
    X = square_from_condensed(x_condensed, n)
    y = np.asarray(y_condensed, dtype=np.float64)
    r = spearman(upper(X), y)
    perms = np.asarray(perms, dtype=np.int64).reshape(-1, n)
    rk = np.empty(len(perms), dtype=np.float64)
    for k, pi in enumerate(perms):
        rk[k] = spearman(upper(X[pi][:, pi]), y)
    K = len(perms)
    p_two = (np.sum(np.abs(rk) >= abs(r)) + 1.0) / (K + 1.0)
    p_gr = (np.sum(rk >= r) + 1.0) / (K + 1.0)
    p_le = (np.sum(rk <= r) + 1.0) / (K + 1.0)
    return r, float(p_two), float(p_gr), float(p_le), rk
