"""Pins of the Spearman half of oracle/mantel_oracle.py against things other than itself: a hand-worked example with ties in
exact rationals (tests/golden/mantel_spearman_4objects.txt), scipy's rankdata / spearmanr, the no-ties closed form
1 - 6 sum d^2 / (m (m^2 - 1)), invariance under strictly monotone transforms, and brute-force ranks on tiny inputs."""
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy import stats

from oracle import mantel_oracle as M

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden():
    g = {"perm": []}
    for line in open(os.path.join(HERE, "golden", "mantel_spearman_4objects.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        if k == "perm":
            g["perm"].append([int(t) for t in v])
        else:
            g[k] = v
    return g


def test_handworked_four_objects_with_ties():
    g = _golden()
    n = int(g["n"][0])
    x = np.array([float(t) for t in g["x"]])
    y = np.array([float(t) for t in g["y"]])
    assert M.average_ranks(x).tolist() == [float(Fraction(t)) for t in g["ranks_x"]]
    assert M.average_ranks(y).tolist() == [float(Fraction(t)) for t in g["ranks_y"]]
    r, p2, pg, pl, rk = M.mantel_spearman(x, y, n, np.array(g["perm"]))
    assert r == pytest.approx(float(Fraction(g["r"][0])), abs=1e-15)
    assert rk == pytest.approx([float(Fraction(t)) for t in g["r_perm"]], abs=1e-15)
    assert (p2, pg, pl) == pytest.approx((float(Fraction(g["p_two_sided"][0])), float(Fraction(g["p_greater"][0])),
                                          float(Fraction(g["p_less"][0]))))


@pytest.mark.parametrize("seed", [0, 1, 2])
def test_ranks_and_rho_match_scipy_with_and_without_ties(seed):
    rng = np.random.default_rng(seed)
    a = rng.integers(0, 12, size=300).astype(np.float64)       # many ties
    b = rng.random(300)                                        # none
    assert np.array_equal(M.average_ranks(a), stats.rankdata(a, method="average"))
    assert np.array_equal(M.average_ranks(b), stats.rankdata(b, method="average"))
    assert M.spearman(a, b) == pytest.approx(stats.spearmanr(a, b)[0], abs=1e-14)
    assert M.spearman(a, a[::-1].copy()) == pytest.approx(stats.spearmanr(a, a[::-1])[0], abs=1e-14)


def test_brute_force_ranks_tiny():
    rng = np.random.default_rng(5)
    a = rng.integers(0, 4, size=9).astype(np.float64)
    brute = [sum(1 for v in a if v < t) + (sum(1 for v in a if v == t) + 1) / 2 for t in a]   # (#smaller) + (ties + 1) / 2
    assert M.average_ranks(a).tolist() == brute


def test_no_ties_closed_form_and_monotone_invariance():
    rng = np.random.default_rng(7)
    m = 200
    a, b = rng.random(m), rng.random(m)
    d = M.average_ranks(a) - M.average_ranks(b)
    assert M.spearman(a, b) == pytest.approx(1.0 - 6.0 * np.sum(d * d) / (m * (m * m - 1.0)), abs=1e-13)
    assert M.spearman(np.exp(3 * a), b ** 3) == pytest.approx(M.spearman(a, b), abs=1e-15)     # strictly increasing maps
    assert M.spearman(a, -b) == pytest.approx(-M.spearman(a, b), abs=1e-15)
    assert M.spearman(a, 2 * a + 1) == pytest.approx(1.0, abs=1e-15)
    assert M.spearman(np.full(m, 0.3), b) == 0.0                                               # zero variance (M4)


def test_mantel_spearman_properties():
    rng = np.random.default_rng(11)
    n = 9
    P = n * (n - 1) // 2
    x = np.round(rng.random(P), 1)                       # ties
    y = rng.random(P)
    perms = np.stack([rng.permutation(n) for _ in range(6)])
    r, p2, pg, pl, rk = M.mantel_spearman(x, y, n, perms)
    # the statistic equals Mantel/Pearson of the rank-transformed matrices (ranks do not depend on the order of the entries)
    r2, _, _, _, rk2 = M.mantel_pearson(M.average_ranks(x), M.average_ranks(y), n, perms)
    assert r == pytest.approx(r2, abs=1e-15) and rk == pytest.approx(rk2, abs=1e-14)
    ident = np.arange(n)[None, :]
    assert M.mantel_spearman(x, y, n, ident)[4][0] == pytest.approx(r, abs=1e-15)
    assert p2 == (np.sum(np.abs(rk) >= abs(r)) + 1) / 7 and pg == (np.sum(rk >= r) + 1) / 7 and pl == (np.sum(rk <= r) + 1) / 7
