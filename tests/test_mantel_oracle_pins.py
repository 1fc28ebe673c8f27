"""Pins of the Mantel / Pearson oracle (oracle/mantel_oracle.py) against things other than itself: a hand-worked example in
exact rationals (tests/golden/mantel_4objects.txt), scipy's pearsonr, closed forms, invariances, and a second formulation
(pure-Python loops over the condensed index, no square matrices) on tiny inputs."""
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy import stats

from oracle import mantel_oracle as M

HERE = os.path.dirname(os.path.abspath(__file__))


def _rand_condensed(rng, n):
    return rng.random(n * (n - 1) // 2)


def _golden():
    g = {"perm": []}
    for line in open(os.path.join(HERE, "golden", "mantel_4objects.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        if k == "perm":
            g["perm"].append([int(t) for t in v])
        else:
            g[k] = v
    return g


def test_handworked_four_objects_exact_rationals():
    g = _golden()
    n = int(g["n"][0])
    x = np.array([float(t) for t in g["x"]])
    y = np.array([float(t) for t in g["y"]])
    r, p2, pg, pl, rk = M.mantel_pearson(x, y, n, np.array(g["perm"]))
    assert r == pytest.approx(float(Fraction(g["r"][0])), abs=1e-15)
    assert rk == pytest.approx([float(Fraction(t)) for t in g["r_perm"]], abs=1e-15)
    assert p2 == pytest.approx(float(Fraction(g["p_two_sided"][0])))
    assert pg == pytest.approx(float(Fraction(g["p_greater"][0])))
    assert pl == pytest.approx(float(Fraction(g["p_less"][0])))


def _loops(x, y, n, pi):
    """second formulation: explicit loops over i < j with condensed index arithmetic, means subtracted term by term"""
    idx = lambda i, j: i * (2 * n - i - 1) // 2 + (j - i - 1)
    xs, ys = [], []
    for i in range(n):
        for j in range(i + 1, n):
            a, b = pi[i], pi[j]
            xs.append(x[idx(min(a, b), max(a, b))])
            ys.append(y[idx(i, j)])
    mx, my = sum(xs) / len(xs), sum(ys) / len(ys)
    sxy = sum((a - mx) * (b - my) for a, b in zip(xs, ys))
    sxx = sum((a - mx) ** 2 for a in xs)
    syy = sum((b - my) ** 2 for b in ys)
    return sxy / (sxx * syy) ** 0.5


@pytest.mark.parametrize("n", [3, 5, 9])
def test_against_scipy_pearsonr_and_loop_formulation(n):
    rng = np.random.default_rng(n)
    x, y = _rand_condensed(rng, n), _rand_condensed(rng, n)
    perms = np.array([rng.permutation(n) for _ in range(6)])
    r, _, _, _, rk = M.mantel_pearson(x, y, n, perms)
    assert r == pytest.approx(stats.pearsonr(x, y)[0], abs=1e-13)
    assert r == pytest.approx(_loops(x, y, n, list(range(n))), abs=1e-13)
    for k, pi in enumerate(perms):
        assert rk[k] == pytest.approx(_loops(x, y, n, list(pi)), abs=1e-13)
        Xp = M.square_from_condensed(x, n)[np.ix_(pi, pi)]
        assert rk[k] == pytest.approx(stats.pearsonr(Xp[np.triu_indices(n, 1)], y)[0], abs=1e-13)


def test_closed_forms_and_invariances():
    rng = np.random.default_rng(0)
    n = 12
    x, y = _rand_condensed(rng, n), _rand_condensed(rng, n)
    ident = np.arange(n)[None, :]
    assert M.mantel_pearson(x, 3.0 * x + 2.0, n, ident)[0] == pytest.approx(1.0, abs=1e-14)       # Y = aX + b, a > 0
    assert M.mantel_pearson(x, -0.5 * x + 1.0, n, ident)[0] == pytest.approx(-1.0, abs=1e-14)     # a < 0
    r, p2, pg, pl, rk = M.mantel_pearson(x, y, n, ident)
    assert rk[0] == pytest.approx(r, abs=1e-15) and p2 == 1.0 and pg == 1.0 and pl == 1.0       # identity permutation
    assert M.mantel_pearson(y, x, n, ident)[0] == pytest.approx(r, abs=1e-15)                     # symmetric in X, Y
    assert M.mantel_pearson(5.0 * x + 1.0, 0.1 * y, n, ident)[0] == pytest.approx(r, abs=1e-13)    # affine invariance
    pi = rng.permutation(n)
    inv = np.argsort(pi)
    X, Y = M.square_from_condensed(x, n), M.square_from_condensed(y, n)
    # relabelling the objects of BOTH matrices does not change r;  r(X^pi, Y) = r(X, Y^(pi^-1))
    assert M.pearson(M.upper(X[np.ix_(pi, pi)]), M.upper(Y[np.ix_(pi, pi)])) == pytest.approx(r, abs=1e-14)
    r_pi = M.mantel_pearson(x, y, n, pi[None, :])[4][0]
    assert M.pearson(M.upper(X), M.upper(Y[np.ix_(inv, inv)])) == pytest.approx(r_pi, abs=1e-14)
    assert -1.0 <= r_pi <= 1.0


def test_zero_variance_gives_zero_and_p_value_counts():
    n = 6
    rng = np.random.default_rng(1)
    y = _rand_condensed(rng, n)
    assert M.mantel_pearson(np.full(15, 0.25), y, n, np.arange(n)[None, :])[0] == 0.0
    # X = Y: r = 1 is the maximum, so no random permutation beats it: p_greater = (ties + 1) / (K + 1)
    perms = np.array([rng.permutation(n) for _ in range(19)])
    r, p2, pg, pl, rk = M.mantel_pearson(y, y, n, perms)
    ties = int(np.sum(rk >= 1.0 - 1e-15))
    assert r == pytest.approx(1.0) and pg == pytest.approx((ties + 1) / 20) and pl == 1.0
