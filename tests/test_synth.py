"""Host-side checks of the seeded input generators (shapes, determinism, structure)."""
import numpy as np

from paper_2107_05397_b200 import synth
from oracle import oracle


def test_tiny_shapes_and_determinism():
    p = synth.make_config("tiny", seed=0)
    q = synth.make_config("tiny", seed=0)
    r = synth.make_config("tiny", seed=1)
    assert p.n_nodes == 511 and p.n_samples == 64
    for f in ("parent", "branch_len", "postorder", "indptr", "indices", "counts"):
        assert np.array_equal(getattr(p, f), getattr(q, f))
    assert not np.array_equal(p.indices, r.indices)
    assert p.counts.min() >= 1 and p.branch_len[0] == 0.0
    assert np.all(p.parent[1:] < np.arange(1, p.n_nodes))          # Yule: parent id < child id
    assert oracle.validate(p.parent, p.branch_len, p.postorder, p.indptr, p.indices, p.counts) == 0


def test_yule_is_binary_and_postorder_is_dfs():
    p = synth.make_config("tiny", seed=3)
    deg = np.bincount(p.parent[p.parent >= 0], minlength=p.n_nodes)
    assert set(np.unique(deg)) == {0, 2}
    pos = np.empty(p.n_nodes, dtype=np.int64)
    pos[p.postorder] = np.arange(p.n_nodes)
    nonroot = p.parent >= 0
    assert np.all(pos[nonroot] < pos[p.parent[nonroot]])
    assert p.parent[p.postorder[-1]] == -1


def test_rows_sorted_distinct_tips():
    p = synth.make_config("tiny", seed=2)
    tips = set(synth.tip_ids(p.parent).tolist())
    for s in range(p.n_samples):
        row = p.indices[p.indptr[s]:p.indptr[s + 1]]
        assert row.size >= 1 and np.all(np.diff(row) > 0) and set(row.tolist()) <= tips


def test_small_density_matches_survey_estimate():
    p = synth.make_config("small", seed=0, n_samples=256)
    per = np.diff(p.indptr)
    assert 150 < per.mean() < 320            # ~229 features/sample


def test_sample_pairs_and_condensed_index():
    pr = synth.sample_pairs(100, 1000, seed=0)
    assert np.all(pr[:, 0] < pr[:, 1]) and pr.min() >= 0 and pr.max() < 100
    assert synth.condensed_index(5, 0, 1) == 0 and synth.condensed_index(5, 3, 4) == 9
    assert synth.condensed_index(50000, 49998, 49999) == 50000 * 49999 // 2 - 1
