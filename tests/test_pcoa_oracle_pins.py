"""Pins of oracle/pcoa_oracle.py against things other than itself: a hand-worked 3-point example in exact rationals
(tests/golden/pcoa_3points.txt), points with known Euclidean coordinates (classical scaling recovers their centred Gram matrix,
the eigenvalues are those of the small d x d scatter matrix -- a different matrix through a different routine), the trace
identity trace(B) = (1/n) sum_{i<j} d_ij^2, zero row sums, and scale / relabelling behaviour."""
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import pcoa_oracle as O

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden():
    g = {}
    for line in open(os.path.join(HERE, "golden", "pcoa_3points.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        g[k] = v
    return g


def _condensed_from_points(X):
    n = X.shape[0]
    iu = np.triu_indices(n, 1)
    return np.sqrt(((X[iu[0]] - X[iu[1]]) ** 2).sum(1))


def test_handworked_three_points():
    g = _golden()
    n = int(g["n"][0])
    d = np.array([float(t) for t in g["d"]])
    B = O.gower_center(O.square_from_condensed(d, n))
    assert B.ravel() == pytest.approx([float(Fraction(t)) for t in g["B"]], abs=1e-15)
    lam, coords, prop = O.pcoa(d, n, 3)
    assert lam == pytest.approx([float(Fraction(t)) for t in g["eigenvalues"]], abs=1e-14)
    want = np.array([float(Fraction(t)) for t in g["coords_axis1"]])
    c = coords[:, 0] * np.sign(coords[2, 0])
    assert c == pytest.approx(want, abs=1e-14)
    assert prop[0] == pytest.approx(float(Fraction(g["proportion"][0])), abs=1e-14)
    assert np.abs(coords[:, 1:]).max() <= 1e-7          # sqrt of eigenvalues that are 0 up to rounding


@pytest.mark.parametrize("seed,n,dim", [(0, 12, 2), (1, 40, 3), (2, 25, 5)])
def test_points_with_known_coordinates(seed, n, dim):
    rng = np.random.default_rng(seed)
    X = rng.normal(size=(n, dim)) * np.arange(1, dim + 1)[None, :]       # distinct spreads -> distinct eigenvalues
    d = _condensed_from_points(X)
    lam, coords, prop = O.pcoa(d, n, dim + 2)
    Xc = X - X.mean(0)
    # eigenvalues of the n x n matrix B = the eigenvalues of the dim x dim scatter matrix Xc' Xc, then zeros
    want = np.sort(np.linalg.eigvalsh(Xc.T @ Xc))[::-1]
    assert lam[:dim] == pytest.approx(want, rel=1e-10)
    assert np.abs(lam[dim:]).max() <= 1e-9 * want[0]
    # the coordinates reproduce the centred Gram matrix and therefore every distance
    assert coords[:, :dim] @ coords[:, :dim].T == pytest.approx(Xc @ Xc.T, abs=1e-9 * want[0])
    assert _condensed_from_points(coords[:, :dim]) == pytest.approx(d, rel=1e-9)
    # axis i = projection of the centred points on the i-th principal direction (up to sign)
    w, U = np.linalg.eigh(Xc.T @ Xc)
    U = U[:, ::-1]
    for i in range(dim):
        proj = Xc @ U[:, i]
        s = np.sign(proj @ coords[:, i])
        assert coords[:, i] == pytest.approx(s * proj, abs=1e-8 * np.sqrt(want[0]))
    assert prop[:dim].sum() == pytest.approx(1.0, abs=1e-10)


def test_trace_identity_row_sums_scale_and_relabelling():
    rng = np.random.default_rng(4)
    n = 30
    d = rng.random(n * (n - 1) // 2) + 0.2                  # an arbitrary (non-Euclidean) dissimilarity
    B = O.gower_center(O.square_from_condensed(d, n))
    assert np.abs(B.sum(0)).max() <= 1e-12 and np.abs(B.sum(1)).max() <= 1e-12
    assert np.trace(B) == pytest.approx(np.sum(d * d) / n, rel=1e-13)
    assert B == pytest.approx(B.T, abs=1e-14)
    lam, coords, prop = O.pcoa(d, n, 4)
    lam2, coords2, prop2 = O.pcoa(3.0 * d, n, 4)
    assert lam2 == pytest.approx(9.0 * lam, rel=1e-12) and prop2 == pytest.approx(prop, rel=1e-12)
    assert np.abs(coords2) == pytest.approx(3.0 * np.abs(coords), rel=1e-9)
    # relabelling the objects permutes the coordinates' rows
    pi = rng.permutation(n)
    D = O.square_from_condensed(d, n)[np.ix_(pi, pi)]
    lam3, coords3, _ = O.pcoa(D[np.triu_indices(n, 1)], n, 4)
    assert lam3 == pytest.approx(lam, rel=1e-12)
    assert np.abs(coords3) == pytest.approx(np.abs(coords[pi]), abs=1e-9)
    # eigen-equation on the full matrix
    for i in range(4):
        v = coords[:, i]
        assert B @ v == pytest.approx(lam[i] * v, abs=1e-10)
