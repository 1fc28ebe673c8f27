"""The grouped join of the mid branches (midg.cuh): branches whose presence sets nest are joined with one
shared-memory atomic per pair of the group's root.  All sums are exact integer sums of the same fixed-point values the ungrouped
join (k_mid) adds, into the same accumulators, so with the head / mid / tail classes held fixed the two paths must agree BIT FOR
BIT, for any grouping threshold; against the oracle the usual tolerance applies.  Trees where nesting is extreme (a caterpillar:
every internal node has one tip and one internal child; unary chains: equal presence sets) are the degenerate cases."""
import numpy as np
import pytest

from paper_2107_05397_b200 import synth

pytestmark = pytest.mark.gpu

U, W = 0, 1
FP32 = 0


@pytest.fixture(scope="module")
def B():
    from paper_2107_05397_b200 import binding
    binding.load()
    return binding


@pytest.fixture(scope="module")
def O():
    from oracle import oracle
    return oracle


def run(B, p, variant, flags=0):
    import torch
    out = B.unifrac_dm(*B.to_device(p), p.n_samples, variant, FP32, flags=flags)
    torch.cuda.synchronize()
    return out.cpu().numpy(), B.unifrac_last_stats()


def fix_classes(monkeypatch):
    # the cost model moves the head / mid boundary when the grouped join is expected: pin its rates so that both runs classify alike
    monkeypatch.setenv("UNIFRAC_B200_R_MID", "1.6e12")
    monkeypatch.setenv("UNIFRAC_B200_R_MID_SPARSE", "5.5e11")
    # and no tail class (every row with a pair goes to the join): the tail's fp32 REDs reach a cell in arbitrary order, which
    # may move the last bit from run to run; without them the whole path is order-independent
    monkeypatch.setenv("UNIFRAC_B200_R_TAIL", "1e3")


def check_oracle(got, want):
    err = np.abs(got.astype(np.float64) - want)
    assert np.all(err <= 1e-5 * np.abs(want) + 1e-7), float(np.max(err / np.maximum(np.abs(want), 1e-300)))


@pytest.mark.parametrize("variant", [U, W])
def test_grouped_join_equals_ungrouped_join_bit_for_bit(B, O, variant, monkeypatch):
    """Small config shape at 700 samples (6 tiles, ragged tail), forced through the mid class (NO_TENSOR keeps the unweighted head on
    the CUDA cores; the default split leaves hundreds of mid rows at this size)."""
    fix_classes(monkeypatch)
    p = synth.make_problem(12000, 700, 0.05, 1.05, synth.CONFIGS["small"][4], synth.CONFIGS["small"][5], seed=5)
    monkeypatch.setenv("UNIFRAC_B200_MID_GROUPS", "0")
    ref, s_ref = run(B, p, variant)
    assert s_ref["mid_groups"] == 0 and s_ref["mid_rows"] > 50 and s_ref["mid_atomics"] == s_ref["mid_updates"] and s_ref["tail_updates"] == 0
    for theta in ("0.35", "0.05", "0.9"):
        monkeypatch.setenv("UNIFRAC_B200_MID_GROUPS", "1")
        monkeypatch.setenv("UNIFRAC_B200_MID_GROUP_THETA", theta)
        got, s = run(B, p, variant)
        assert s["mid_rows"] == s_ref["mid_rows"] and s["head_rows"] == s_ref["head_rows"]
        assert s["mid_groups"] > 0 and 2 * s["mid_groups"] <= s["mid_group_rows"] <= 4 * s["mid_groups"]
        assert s["mid_atomics"] < s["mid_updates"]
        # bit for bit -- except that the fp64 side sums are accumulated with atomics in arbitrary order, which can move an fp32
        # result by one ulp when its fp64 value sits on a rounding boundary (probability ~1e-9 per element): allow 3 such elements
        differ = got != ref
        assert int(differ.sum()) <= 3 and float(np.max(np.abs(got - ref))) <= 1.2e-7, (variant, theta, int(differ.sum()))
    want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant)
    check_oracle(ref, want)


def caterpillar(n_tips, rng):
    """node ids: tips 0..n_tips-1, internal n_tips..2 n_tips - 2; internal k has tip k and internal k+1 (the last one two tips)."""
    n = 2 * n_tips - 1
    parent = np.full(n, -1, np.int32)
    for k in range(n_tips - 1):
        node = n_tips + k
        parent[k] = node
        if k + 1 < n_tips - 1:
            parent[node + 1] = node
    parent[n_tips - 1] = n - 1
    return parent, rng.exponential(0.05, n)


@pytest.mark.parametrize("variant", [U, W])
def test_caterpillar_and_unary_chains_against_the_oracle(B, O, variant, monkeypatch):
    """Every internal branch of a caterpillar contains the next one: long chains of nested presence sets, n_child / n_parent close
    to 1.  ALL_TAIL off, mid forced wide by a high head rate; then the same through a tree with unary internal nodes (equal sets)."""
    monkeypatch.setenv("UNIFRAC_B200_R_HEAD", "1e11")              # a slow dense kernel: (almost) every row below the root goes to mid / tail
    rng = np.random.default_rng(21)
    parent, bl = caterpillar(400, rng)
    tips = np.arange(400)
    rows = []
    for s in range(300):
        k = int(rng.integers(5, 120))
        lo = int(rng.integers(0, 400 - k))                        # a window of neighbouring tips plus a few far ones
        ids = set(range(lo, lo + k)) | set(int(t) for t in rng.choice(tips, 3))
        rows.append({t: int(rng.integers(1, 50)) for t in ids})
    p = synth.problem_from_parent(parent, bl, rows)
    got, s = run(B, p, variant, flags=B.FLAG_NO_TENSOR)
    assert s["mid_groups"] > 0
    check_oracle(got, O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant))
    parent, bl = synth.random_tree(900, rng, p_unary=0.4)
    rows = synth.random_table(synth.tip_ids(parent), 260, rng, density=0.2)
    p = synth.problem_from_parent(parent, bl, rows)
    got, s = run(B, p, variant, flags=B.FLAG_NO_TENSOR)
    assert s["mid_groups"] > 0
    check_oracle(got, O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant))
