"""Pins for the CPU oracle (oracle/unifrac_oracle.c) against things other than itself:
a hand-worked example with exact rationals, closed forms, scipy's Jaccard / Bray-Curtis on star
trees, a second numpy formulation with the I1 closed-form denominator, brute force over all
pairs for N <= 16, the invariants BASELINE.json:5 lists, and metamorphic relations.
None of this needs a GPU."""
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy.spatial.distance import pdist, squareform

from oracle import oracle
from paper_2107_05397_b200 import synth
import refmath

GOLD = os.path.join(os.path.dirname(__file__), "golden", "handworked_7node.txt")
U, W = oracle.UNWEIGHTED, oracle.WEIGHTED_NORMALIZED


def _all(p, variant):
    return oracle.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant)


def _read_gold():
    parent = bl = None
    rows, exp = [], {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        k, *rest = line.split()
        if k == "parent":
            parent = [int(x) for x in rest]
        elif k == "branch_len":
            bl = [float(x) for x in rest]
        elif k == "sample":
            rows.append({int(a.split(":")[0]): int(a.split(":")[1]) for a in rest})
        else:
            exp[k] = [Fraction(x) for x in rest]
    return synth.problem_from_parent(parent, bl, rows), exp


def test_handworked_example_exact():
    p, exp = _read_gold()
    assert oracle.validate(p.parent, p.branch_len, p.postorder, p.indptr, p.indices, p.counts) == 0
    for variant, key in ((U, "unweighted"), (W, "weighted_normalized")):
        d = _all(p, variant)
        want = np.array([float(f) for f in exp[key]])
        np.testing.assert_allclose(d, want, rtol=1e-15, atol=0)
        # the same values through exact rational arithmetic of the second formulation
        k = 0
        for a in range(5):
            for b in range(a + 1, 5):
                assert refmath.unifrac_pair_exact(p, variant, a, b) == exp[key][k]
                k += 1
        assert d[2] == 0.0            # D is proportional to A -> exactly 0


def test_two_tip_closed_forms():
    l0, l1 = 0.7, 1.9
    parent = [2, 2, -1]
    p = synth.problem_from_parent(parent, [l0, l1, 0.0], [{0: 4}, {1: 9}, {0: 1, 1: 1}, {0: 1}])
    du, dw = _all(p, U), _all(p, W)
    # a on t0 only, b on t1 only -> 1 (both variants)
    assert du[0] == 1.0 and dw[0] == 1.0
    # a = {t0:1,t1:1}, b = {t0:1}:  d_U = l1/(l0+l1) ; d_W = (l0/2 + l1/2)/(3/2 l0 + l1/2)
    n = 4
    k = int(synth.condensed_index(n, 2, 3))
    assert du[k] == pytest.approx(l1 / (l0 + l1), rel=1e-15)
    assert dw[k] == pytest.approx((0.5 * l0 + 0.5 * l1) / (1.5 * l0 + 0.5 * l1), rel=1e-15)


@pytest.mark.parametrize("seed", [0, 1])
def test_star_tree_reduces_to_jaccard_and_braycurtis(seed):
    rng = np.random.default_rng(seed)
    n_tips, n = 40, 12
    parent, bl = synth.star_tree(n_tips, np.ones(n_tips))
    rows = synth.random_table(np.arange(n_tips), n, rng, density=0.3)
    p = synth.problem_from_parent(parent, bl, rows)
    X = refmath.dense_counts(p, np.arange(n_tips)).astype(float)
    np.testing.assert_allclose(_all(p, U), pdist(X > 0, "jaccard"), rtol=1e-14)
    P = X / X.sum(1, keepdims=True)
    np.testing.assert_allclose(_all(p, W), pdist(P, "braycurtis"), rtol=1e-13)
    np.testing.assert_allclose(_all(p, W), 0.5 * pdist(P, "cityblock"), rtol=1e-13)


def test_star_tree_arbitrary_lengths_weighted_jaccard():
    rng = np.random.default_rng(3)
    n_tips, n = 30, 10
    ell = rng.exponential(1.0, n_tips)
    parent, bl = synth.star_tree(n_tips, ell)
    p = synth.problem_from_parent(parent, bl, synth.random_table(np.arange(n_tips), n, rng))
    X = refmath.dense_counts(p, np.arange(n_tips)).astype(float)
    B = X > 0
    P = X / X.sum(1, keepdims=True)
    du, dw, k = _all(p, U), _all(p, W), 0
    for a in range(n):
        for b in range(a + 1, n):
            assert du[k] == pytest.approx((ell * (B[a] ^ B[b])).sum() / (ell * (B[a] | B[b])).sum(), rel=1e-14)
            assert dw[k] == pytest.approx((ell * np.abs(P[a] - P[b])).sum() / (ell * (P[a] + P[b])).sum(), rel=1e-13)
            k += 1


@pytest.mark.parametrize("seed", range(6))
def test_bruteforce_second_formulation_random_trees(seed):
    """General trees (multifurcations, unary nodes, zero lengths, shuffled ids), N <= 16:
    every pair against E = X A^T with the I1 closed-form weighted denominator."""
    rng = np.random.default_rng(100 + seed)
    parent, bl = synth.random_tree(int(rng.integers(8, 60)), rng)
    tips = synth.tip_ids(parent)
    p = synth.problem_from_parent(parent, bl, synth.random_table(tips, int(rng.integers(2, 17)), rng))
    assert oracle.validate(p.parent, p.branch_len, p.postorder, p.indptr, p.indices, p.counts) == 0
    for variant in (U, W):
        D = refmath.unifrac_matrix_np(p, variant)
        np.testing.assert_allclose(_all(p, variant), squareform(D, checks=False), rtol=1e-12, atol=1e-15)


def test_tiny_config_against_second_formulation():
    p = synth.make_config("tiny", seed=0)
    for variant in (U, W):
        D = refmath.unifrac_matrix_np(p, variant)
        np.testing.assert_allclose(_all(p, variant), squareform(D, checks=False), rtol=1e-12)


def test_invariants_tiny():
    p = synth.make_config("tiny", seed=0)
    n = p.n_samples
    for variant in (U, W):
        d = _all(p, variant)
        assert np.all(d >= 0) and np.all(d <= 1)
        for a in (0, 5, n - 1):
            assert oracle.pair(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant, a, a) == 0.0
        for a, b in ((0, 1), (3, 40), (62, 63)):
            dab = oracle.pair(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant, a, b)
            dba = oracle.pair(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant, b, a)
            assert dab == pytest.approx(dba, rel=1e-15)
            assert dab == pytest.approx(d[int(synth.condensed_index(n, a, b))], rel=1e-15)
    # triangle inequality: unweighted only (weighted-normalized is Bray-Curtis-like, not a metric)
    D = squareform(_all(p, U))
    viol = D[:, :, None] - (D[:, None, :] + D.T[None, :, :])       # d(a,b) - d(a,c) - d(c,b)
    assert viol.max() <= 1e-12


def test_disjoint_branch_sets_give_one_unweighted_and_weighted():
    # tips under different children of the root share no branch
    parent = [4, 4, 5, 5, 6, 6, -1]
    p = synth.problem_from_parent(parent, [1, 2, 3, 4, 5, 6, 0], [{0: 2, 1: 1}, {2: 7}, {3: 1, 2: 1}])
    du, dw = _all(p, U), _all(p, W)
    assert du[0] == 1.0 and du[1] == 1.0 and dw[0] == 1.0 and dw[1] == 1.0
    assert du[2] < 1.0


def _rand_problem(seed, n=9):
    rng = np.random.default_rng(seed)
    parent, bl = synth.random_tree(40, rng)
    tips = synth.tip_ids(parent)
    return parent, bl, synth.random_table(tips, n, rng), rng


def test_metamorphic_scale_lengths_and_counts():
    parent, bl, rows, rng = _rand_problem(7)
    base = synth.problem_from_parent(parent, bl, rows)
    scaled = synth.problem_from_parent(parent, bl * 3.0, rows)      # exact in binary? x3 is not; use rtol
    rows2 = [dict(r) for r in rows]
    rows2[2] = {t: 5 * c for t, c in rows2[2].items()}              # one sample's counts x5
    mult = synth.problem_from_parent(parent, bl, rows2)
    dup = synth.problem_from_parent(parent, bl, rows + [rows2[2]])
    for variant in (U, W):
        d0 = _all(base, variant)
        np.testing.assert_allclose(_all(scaled, variant), d0, rtol=1e-13, atol=1e-16)
        np.testing.assert_allclose(_all(mult, variant), d0, rtol=1e-13, atol=1e-16)
        n = dup.n_samples
        dd = _all(dup, variant)
        assert dd[int(synth.condensed_index(n, 2, n - 1))] == 0.0   # proportional copy -> exactly 0


def test_metamorphic_permute_samples_relabel_nodes_split_branch_add_unobserved():
    parent, bl, rows, rng = _rand_problem(11)
    base = synth.problem_from_parent(parent, bl, rows)
    n = base.n_samples
    perm = rng.permutation(n)
    permuted = synth.problem_from_parent(parent, bl, [rows[i] for i in perm])
    # relabel nodes
    m = len(parent)
    rel = rng.permutation(m)
    parent2 = np.full(m, -1, dtype=np.int32)
    bl2 = np.zeros(m)
    for v in range(m):
        bl2[rel[v]] = bl[v]
        if parent[v] >= 0:
            parent2[rel[v]] = rel[parent[v]]
    relabeled = synth.problem_from_parent(parent2, bl2, [{int(rel[t]): c for t, c in r.items()} for r in rows])
    # split the branch above some observed tip into two unary pieces of the same total length,
    # and hang an unobserved 3-node subtree under the root
    t = next(iter(rows[0]))
    root = int(np.nonzero(np.asarray(parent) < 0)[0][0])
    parent3 = list(parent) + [parent[t], root, m + 1, m + 1]
    bl3 = list(bl) + [bl[t] * 0.25, 0.3, 0.5, 0.7]
    parent3[t] = m
    bl3[t] = bl[t] * 0.75
    extended = synth.problem_from_parent(parent3, bl3, rows)
    for variant in (U, W):
        D0 = squareform(_all(base, variant))
        Dp = squareform(_all(permuted, variant))
        np.testing.assert_allclose(Dp, D0[np.ix_(perm, perm)], rtol=1e-13, atol=1e-16)
        np.testing.assert_allclose(_all(relabeled, variant), _all(base, variant), rtol=1e-13, atol=1e-16)
        np.testing.assert_allclose(_all(extended, variant), _all(base, variant), rtol=1e-13, atol=1e-16)


def test_identities_I3_I4_I5_hold_for_oracle_values():
    """The algebraic shortcuts the CUDA path uses (I2-I5), checked against the oracle's
    definitional values with sums computed here from the second formulation's embeddings."""
    p = synth.make_config("tiny", seed=1)
    A, tips = refmath.ancestor_matrix(p.parent)
    X = refmath.dense_counts(p, tips)
    ell = np.where(p.parent >= 0, p.branch_len, 0.0)
    Cn = X @ A.T
    Pm = (Cn > 0).astype(float)
    Um = Cn / X.sum(1, keepdims=True)
    S = Pm @ ell
    R = Um @ ell
    G = (Pm * ell) @ Pm.T
    n = p.n_samples
    du, dw = squareform(_all(p, U)), squareform(_all(p, W))
    for a, b in ((0, 1), (2, 9), (10, 63), (31, 32)):
        num_u = S[a] + S[b] - 2 * G[a, b]                                   # I5
        assert du[a, b] == pytest.approx(num_u / (S[a] + S[b] - G[a, b]), rel=1e-12)
        assert du[a, b] == pytest.approx(2 * num_u / (S[a] + S[b] + num_u), rel=1e-12)   # I4
        M = (ell * np.minimum(Um[a], Um[b])).sum()
        assert dw[a, b] == pytest.approx((R[a] + R[b] - 2 * M) / (R[a] + R[b]), rel=1e-12)  # I2, I3


def test_pair_list_driver_matches_all_pairs_driver():
    p = synth.make_problem(1500, 96, 0.1, 1.1, synth.CONFIGS["small"][4], synth.CONFIGS["small"][5], seed=5)
    pairs = synth.sample_pairs(p.n_samples, 3000, seed=1)
    idx = synth.condensed_index(p.n_samples, pairs[:, 0], pairs[:, 1])
    for variant in (U, W):
        full = _all(p, variant)
        lst = oracle.pair_list(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant, pairs)
        np.testing.assert_allclose(lst, full[idx], rtol=1e-15, atol=0)


def test_zero_denominator_gives_zero():
    parent, bl = synth.star_tree(3, [0.0, 0.0, 1.0])
    p = synth.problem_from_parent(parent, bl, [{0: 1}, {1: 2}, {2: 1}])
    for variant in (U, W):
        d = _all(p, variant)
        assert d[0] == 0.0 and not np.isnan(d).any()         # reading Q3
        assert d[1] == 1.0


def test_validation_codes():
    p, _ = _read_gold()
    v = lambda **kw: oracle.validate(kw.get("parent", p.parent), kw.get("bl", p.branch_len),
                                     kw.get("post", p.postorder), kw.get("indptr", p.indptr),
                                     kw.get("indices", p.indices), kw.get("counts", p.counts))
    assert v() == oracle.OK
    assert v(parent=np.array([4, 4, 5, 5, 6, -1, -1], np.int32)) == oracle.ERR_TREE      # two roots
    assert v(post=np.array([4, 0, 1, 2, 3, 5, 6], np.int32)) == oracle.ERR_TREE          # parent before child
    assert v(post=np.array([0, 1, 4, 2, 3, 6, 5], np.int32)) == oracle.ERR_TREE          # root not last
    assert v(bl=np.array([1, -2, 3, 4, 5, 6, 0], float)) == oracle.ERR_TREE
    assert v(bl=np.array([1, np.nan, 3, 4, 5, 6, 0], float)) == oracle.ERR_TREE
    assert v(indices=np.array([0, 1, 1, 2, 2, 3, 0, 1, 4], np.int32)) == oracle.ERR_TABLE  # internal node as column
    assert v(indices=np.array([1, 0, 1, 2, 2, 3, 0, 1, 0], np.int32)) == oracle.ERR_TABLE  # not increasing
    assert v(counts=np.array([1, 1, 2, 2, 1, 3, 3, 3, -5], np.int32)) == oracle.ERR_TABLE
    assert v(counts=np.array([1, 1, 2, 2, 1, 3, 3, 3, 0], np.int32)) == oracle.ERR_EMPTY_SAMPLE


def test_hypothesis_random_small_problems():
    hyp = pytest.importorskip("hypothesis")
    from hypothesis import given, settings, strategies as st

    @settings(max_examples=40, deadline=None)
    @given(st.integers(0, 2**31 - 1), st.integers(3, 30), st.integers(2, 8))
    def run(seed, n_nodes, n):
        rng = np.random.default_rng(seed)
        parent, bl = synth.random_tree(n_nodes, rng, p_unary=0.3, p_zero_len=0.3)
        tips = synth.tip_ids(parent)
        p = synth.problem_from_parent(parent, bl, synth.random_table(tips, n, rng, density=0.5))
        for variant in (U, W):
            D = refmath.unifrac_matrix_np(p, variant)
            d = _all(p, variant)
            np.testing.assert_allclose(d, squareform(D, checks=False), rtol=1e-11, atol=1e-15)
            assert np.all((d >= 0) & (d <= 1 + 1e-15))
    run()
