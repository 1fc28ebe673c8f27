"""Near-duplicate samples (d -> 0) on the DEFAULT path: the separable forms lose relative accuracy there, so the finalize
epilogues list every pair with d < 1/16 and k_guard recomputes it from the definition (PAPER.md:11 --
placing new samples into the context of existing data is where replicate / proportional samples occur).
Duplicates and integer multiples must come out EXACTLY 0; copies with one count changed by 1 and one feature dropped
(d ~ 1e-4 .. 1e-2) must match the
oracle to the RELATIVE tolerance alone (the absolute clause must not be what passes them)."""
import numpy as np
import pytest

from paper_2107_05397_b200 import synth

pytestmark = pytest.mark.gpu

U, W = 0, 1
RTOL = {0: 1e-5, 1: 1e-10}
ATOL = {0: 1e-7, 1: 1e-12}


@pytest.fixture(scope="module")
def B():
    from paper_2107_05397_b200 import binding
    binding.load()
    return binding


@pytest.fixture(scope="module")
def O():
    from oracle import oracle
    return oracle


def gpu_dm(B, p, variant, precision, flags=0):
    import torch
    out = B.unifrac_dm(*B.to_device(p), p.n_samples, variant, precision, flags=flags)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


def test_duplicate_and_proportional_samples_give_exactly_zero(B, O):
    parent, bl = synth.random_tree(60, np.random.default_rng(9), p_zero_len=0.0)
    tips = synth.tip_ids(parent)
    rows = synth.random_table(tips, 6, np.random.default_rng(10))
    rows.append(dict(rows[1]))
    rows.append({t: 7 * c for t, c in rows[2].items()})
    p = synth.problem_from_parent(parent, bl, rows)
    n = p.n_samples
    k16, k27 = int(synth.condensed_index(n, 1, 6)), int(synth.condensed_index(n, 2, 7))
    for variant in (U, W):
        want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant)
        assert want[k16] == 0.0 and want[k27] == 0.0
        for precision in (1, 0):
            for flags in (0, B.FLAG_NO_MID, B.FLAG_NO_TENSOR, B.FLAG_ALL_TAIL):
                d = gpu_dm(B, p, variant, precision, flags)
                assert d[k16] == 0.0 and d[k27] == 0.0, (variant, precision, flags, d[k16], d[k27])
                assert B.unifrac_last_stats()["guard_pairs"] >= 2
                err = np.abs(d - want)
                assert ((err <= RTOL[precision] * np.abs(want)) | (err <= ATOL[precision])).all()
                assert np.all(d >= 0) and np.all(d <= 1 + 1e-6) and not np.isnan(d).any()
        d = gpu_dm(B, p, variant, 1, flags=B.FLAG_ABSDIFF)          # direct form: exactly 0 without the guard
        assert d[k16] == 0.0 and d[k27] == 0.0


@pytest.mark.parametrize("variant", [U, W])
def test_planted_near_duplicates_across_tiles_all_pairs(B, O, variant):
    """>= 3 tiles (330 samples = 2 full tiles + a ragged one), 3,000 tips: head, mid and tail classes all non-empty in
    fp32 (and the tensor-core Gram kernel for unweighted); 20 duplicates, 20 integer multiples and 20 slightly changed
    copies whose source / copy sit in different tiles or on tile boundaries.  All 54,285 pairs against the oracle."""
    cfg = synth.CONFIGS["small"]
    base = synth.make_problem(3000, 330, 0.1, 1.1, cfg[4], cfg[5], seed=11)
    p, pairs, kinds = synth.plant_near_duplicates(base, 20, seed=1)
    n = p.n_samples
    assert len({(int(a) // 128, int(b) // 128) for a, b in pairs}) >= 4          # several different tile pairs
    assert any(int(a) // 128 != int(b) // 128 for a, b in pairs)
    idx = synth.condensed_index(n, pairs[:, 0], pairs[:, 1])
    want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant)
    assert np.all(want[idx[kinds < 2]] == 0.0)
    near = want[idx[kinds == 2]]
    assert np.all(near > 0.0) and near.max() < 0.0625                           # d ~ 1e-4 .. 1e-2: all below the guard threshold
    for precision in (0, 1):
        for flags in ((0, B.FLAG_NO_TENSOR) if (variant == U and precision == 0) else
                      (0, B.FLAG_RICHNESS_ZONES) if (variant == W and precision == 0) else (0,)):
            got = gpu_dm(B, p, variant, precision, flags)
            st = B.unifrac_last_stats()
            assert st["skip"] == (1 if flags == B.FLAG_RICHNESS_ZONES else 0)
            if precision == 0:
                assert st["head_rows"] > 0 and st["mid_rows"] > 0 and st["tail_rows"] > 0, st
                assert st["gram"] == (1 if (variant == U and flags == 0) else 0)
            assert st["guard_pairs"] >= 60 and st["quant_fallback"] == 0
            assert np.all(got[idx[kinds < 2]] == 0.0), "duplicates / integer multiples must be exactly 0"
            rel_near = np.abs(got[idx[kinds == 2]] - near) / near
            assert rel_near.max() <= RTOL[precision], f"near-duplicates: max rel err {rel_near.max():.3e} (relative clause only)"
            err = np.abs(got - want)
            ok = (err <= RTOL[precision] * np.abs(want)) | (err <= ATOL[precision])
            assert ok.all(), f"max rel err {(err / np.maximum(want, 1e-300))[~ok].max():.3e}"
            # every pair the guard recomputed (d < 1/16) meets the relative clause alone
            small = (want > 0) & (want < 0.0625)
            if small.any():
                assert (err[small] / want[small]).max() <= RTOL[precision]


def test_guard_in_shard_mode(B, O):
    """Each shard guards the pairs of its own blocks: planted duplicates stay exactly 0 in the merged matrix."""
    import torch
    cfg = synth.CONFIGS["small"]
    base = synth.make_problem(2000, 1700, 0.1, 1.1, cfg[4], cfg[5], seed=13)     # 14 tiles = 2 shard-block rows
    p, pairs, kinds = synth.plant_near_duplicates(base, 8, seed=2)
    n = p.n_samples
    idx = synth.condensed_index(n, pairs[:, 0], pairs[:, 1])
    want = O.pair_list(p.parent, p.branch_len, p.indptr, p.indices, p.counts, W, pairs)
    args = B.to_device(p)
    total = None
    for s in range(2):
        part = B.unifrac_dm(*args, n, W, B.FP32, shard=(s, 2))
        total = part if total is None else total + part
    torch.cuda.synchronize()
    got = total[torch.from_numpy(idx).cuda()].cpu().numpy().astype(np.float64)
    assert np.all(got[kinds < 2] == 0.0)
    assert (np.abs(got[kinds == 2] - want[kinds == 2]) / want[kinds == 2]).max() <= 1e-5


def test_guard_with_segmented_finalize_in_host_multi(B, O):
    """unifrac_dm_host_multi finalizes the last variant in segments of block rows (guard + result copy after each one): planted
    duplicates stay exactly 0 and the host result equals the device entry point's (to the last bits).  1,700 samples = 105 tile pairs,
    enough for the segmentation to kick in."""
    cfg = synth.CONFIGS["small"]
    base = synth.make_problem(2000, 1700, 0.1, 1.1, cfg[4], cfg[5], seed=17)
    p, pairs, kinds = synth.plant_near_duplicates(base, 8, seed=3)
    n = p.n_samples
    idx = synth.condensed_index(n, pairs[:, 0], pairs[:, 1])
    for order in ([U, W], [W, U]):                       # either variant last
        outs = B.unifrac_dm_host_multi(p.parent, p.branch_len, p.postorder, p.indptr, p.indices, p.counts, n, order, B.FP32)
        for v, got in zip(order, outs):
            assert np.all(got[idx[kinds < 2]] == 0.0)
            # (not bit for bit: the tail's fp32 REDs reach a cell in arbitrary order, so the last bit may differ between two runs)
            assert np.allclose(got.astype(np.float64), gpu_dm(B, p, v, 0), rtol=2e-6, atol=1e-7)
    B.unifrac_release_host_pool()
