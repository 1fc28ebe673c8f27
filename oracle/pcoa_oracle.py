"""CPU oracle for principal coordinates analysis (PCoA) of a distance matrix -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it imports nothing from the
CUDA package.

What it follows.  PAPER.md:13 (section I): "researchers often apply principal coordinates analysis (PCoA)" to the
distance matrix; PAPER.md:33 (section II): "PCoA can also be computed as part of the Hybrid UniFrac compute itself";
PAPER.md:59 (section IV).  The paper gives no formula; this is classical (Torgerson / Gower) metric scaling written out in
fp64 with a full symmetric eigendecomposition -- no randomisation, no truncation (readings P1-P5):

  P1  A = -1/2 D o D            (element-wise square of the symmetric hollow distance matrix)
  P2  B = A - rowmean(A) 1' - 1 colmean(A)' + mean(A)         (Gower double centring; rows and columns of B sum to 0)
  P3  B = V diag(lambda) V',  lambda_1 >= lambda_2 >= ...;   coordinates of axis i:  V[:, i] * sqrt(lambda_i)
  P4  proportion explained by axis i = lambda_i / trace(B)    (the convention of the randomised "fsvd" PCoA, where only the
      leading eigenvalues are known; trace(B) = sum of ALL eigenvalues = (1/n) sum_{i<j} d_ij^2)
  P5  an eigenvector's sign is arbitrary: callers compare coordinates up to a sign per axis (and, for repeated eigenvalues,
      up to a rotation inside the eigenspace -- the tests use the Gram matrix of the coordinates there).
"""
from __future__ import annotations

import numpy as np


def square_from_condensed(c: np.ndarray, n: int) -> np.ndarray:
    c = np.asarray(c, dtype=np.float64)
    assert c.shape == (n * (n - 1) // 2,)
    m = np.zeros((n, n), dtype=np.float64)
    iu = np.triu_indices(n, k=1)
    m[iu] = c
    m[(iu[1], iu[0])] = c
    return m


def gower_center(D: np.ndarray) -> np.ndarray:
    """P1 + P2."""
    A = -0.5 * D * D
    rm = A.mean(axis=1, keepdims=True)
    cm = A.mean(axis=0, keepdims=True)
    return A - rm - cm + A.mean()


def pcoa(d_condensed, n: int, k: int):
    """Returns (eigenvalues[k] descending, coordinates[n, k], proportion_explained[k]).  Axes whose eigenvalue is not
    positive get zero coordinates."""
    B = gower_center(square_from_condensed(d_condensed, n))
    lam, V = np.linalg.eigh(B)                   # ascending
    lam, V = lam[::-1], V[:, ::-1]
    lam_k, V_k = lam[:k], V[:, :k]
    coords = V_k * np.sqrt(np.maximum(lam_k, 0.0))[None, :]
    tr = np.trace(B)
    prop = lam_k / tr if tr > 0 else np.zeros(k)
    return lam_k.copy(), coords, prop
