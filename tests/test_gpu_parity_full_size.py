"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (device
entry point, fp32, default flags): sampled outputs the oracle computes one by one (pair-list
driver): 200,000 seeded pairs, ALL 32,640 pairs among 256 seeded samples (a clique: it puts
many pairs into the same tile pairs, which is what catches a wrong cell inside one tile pair),
structured pairs (first/last rows, tile-boundary neighbours, last condensed element) -- SURVEY
8(c) "Large configs" -- and properties that hold at any size (range, no NaN)."""
import numpy as np
import pytest

from paper_2107_05397_b200 import synth

pytestmark = pytest.mark.gpu


def _structured_pairs(n):
    e = [[0, 1], [0, n - 1], [n - 2, n - 1], [127, 128], [0, 128], [127, 255], [128, 129], [0, 127],
         [n - 129, n - 1], [n // 2, n // 2 + 1], [(n // 128) * 128 - 1, (n // 128) * 128], [1, n - 2]]
    return np.array([p for p in e if 0 <= p[0] < p[1] < n], dtype=np.int32)


def _clique_pairs(n, k=256, seed=17):
    members = np.sort(np.random.default_rng(seed).choice(n, size=min(k, n), replace=False))
    i, j = np.triu_indices(len(members), 1)
    return np.stack([members[i], members[j]], 1).astype(np.int32)


@pytest.mark.parametrize("name,n_pairs", [("medium", 200000), ("emp", 200000), ("large", 200000)])
def test_full_size_sampled_pairs(name, n_pairs):
    import torch
    from paper_2107_05397_b200 import binding as B
    from oracle import oracle as O
    free, _ = torch.cuda.mem_get_info()
    if name == "large" and free < 90 * 2**30:
        pytest.skip("needs ~80 GB of free HBM")
    p = synth.make_config(name, seed=0)
    n = p.n_samples
    pairs = np.concatenate([synth.sample_pairs(n, n_pairs, seed=1), _clique_pairs(n), _structured_pairs(n)])
    idx = torch.from_numpy(synth.condensed_index(n, pairs[:, 0], pairs[:, 1])).cuda()
    args = B.to_device(p)
    variants = (0,) if name == "medium" else (0, 1)
    for variant in variants:
        want = O.pair_list(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant, pairs)
        out = B.unifrac_dm(*args, n, variant, B.FP32)
        torch.cuda.synchronize()
        got = out[idx].cpu().numpy().astype(np.float64)
        lo, hi = float(out.min()), float(out.max())
        assert 0.0 <= lo and hi <= 1.0 and not bool(torch.isnan(out).any())
        del out
        err = np.abs(got - want)
        rel = err / np.maximum(np.abs(want), 1e-30)
        ok = (err <= 1e-5 * np.abs(want)) | (err <= 1e-7)
        assert ok.all(), f"{name} variant {variant}: max rel err {rel.max():.3e}"
        print(f"{name} variant {variant}: max rel err {rel.max():.3e}, p99.99 {np.quantile(rel, 0.9999):.3e}, "
              f"min d {want.min():.4f}, pairs {len(want)}")


def _permute_samples(p, perm):
    """Problem with sample k of the result = sample perm[k] of p (CSR rows reordered; nothing else changes)."""
    import copy
    lens = np.diff(p.indptr)[perm]
    indptr = np.concatenate([[0], np.cumsum(lens)]).astype(p.indptr.dtype)
    take = np.concatenate([np.arange(p.indptr[s], p.indptr[s + 1]) for s in perm]) if len(perm) else np.zeros(0, np.int64)
    q = copy.copy(p)
    q.indptr, q.indices, q.counts = indptr, p.indices[take], p.counts[take]
    return q


@pytest.mark.parametrize("name", ["medium", "emp"])
def test_full_size_sample_permutation_property(name):
    """A property that holds at any size (no oracle needed): permuting the samples permutes the matrix.  The permuted run
    puts every pair into a different tile pair / shared-memory cell / TMEM lane and sums in a different order, so agreement
    on 5e6 random pairs per variant checks the tiling, the condensed indexing and the head / mid / tail split against
    themselves at BASELINE.json's sizes (tolerance: twice the fp32 parity tolerance, both runs carry rounding)."""
    import torch
    from paper_2107_05397_b200 import binding as B
    p = synth.make_config(name, seed=0)
    n = p.n_samples
    rng = np.random.default_rng(11)
    perm = rng.permutation(n)
    q = _permute_samples(p, perm)
    inv = np.empty(n, dtype=np.int64)
    inv[perm] = np.arange(n)                                  # sample s of p is sample inv[s] of q
    pairs = synth.sample_pairs(n, 5_000_000, seed=5).astype(np.int64)
    a, b = inv[pairs[:, 0]], inv[pairs[:, 1]]
    idx_p = torch.from_numpy(synth.condensed_index(n, pairs[:, 0], pairs[:, 1])).cuda()
    idx_q = torch.from_numpy(synth.condensed_index(n, np.minimum(a, b), np.maximum(a, b))).cuda()
    args_p, args_q = B.to_device(p), B.to_device(q)
    for variant in ((0,) if name == "medium" else (0, 1)):
        dp = B.unifrac_dm(*args_p, n, variant, B.FP32)[idx_p].double()
        dq = B.unifrac_dm(*args_q, n, variant, B.FP32)[idx_q].double()
        torch.cuda.synchronize()
        err = (dp - dq).abs()
        ok = (err <= 2e-5 * dp.abs()) | (err <= 2e-7)
        assert bool(ok.all()), f"{name} variant {variant}: max rel diff {float((err / dp.abs().clamp_min(1e-30)).max()):.3e}"
        print(f"{name} variant {variant}: permuted run max rel diff {float((err / dp.abs().clamp_min(1e-30)).max()):.3e}")


def test_full_size_richness_zones_flag_emp_weighted():
    """UNIFRAC_FLAG_RICHNESS_ZONES at the EMP-shaped size (196 tiles: permuted samples, 120k+ rows with a dense zone, k_zone +
    join + tail + un-permute): 20,000 sampled + clique + structured pairs against the oracle, and agreement with the default
    path on 5e6 pairs."""
    import torch
    from paper_2107_05397_b200 import binding as B
    from oracle import oracle as O
    p = synth.make_config("emp", seed=0)
    n = p.n_samples
    pairs = np.concatenate([synth.sample_pairs(n, 20000, seed=2), _clique_pairs(n, 128, seed=3), _structured_pairs(n)])
    idx = torch.from_numpy(synth.condensed_index(n, pairs[:, 0], pairs[:, 1])).cuda()
    want = O.pair_list(p.parent, p.branch_len, p.indptr, p.indices, p.counts, 1, pairs)
    args = B.to_device(p)
    out = B.unifrac_dm(*args, n, 1, B.FP32, flags=B.FLAG_RICHNESS_ZONES)
    torch.cuda.synchronize()
    st = B.unifrac_last_stats()
    assert st["skip"] == 1 and st["skip_row_pair_visits"] > 0 and st["mid_updates"] > 0
    got = out[idx].cpu().numpy().astype(np.float64)
    err = np.abs(got - want)
    assert ((err <= 1e-5 * np.abs(want)) | (err <= 1e-7)).all(), f"max rel err {(err / np.maximum(want, 1e-30)).max():.3e}"
    ref = B.unifrac_dm(*args, n, 1, B.FP32)
    big = torch.from_numpy(synth.condensed_index(n, *synth.sample_pairs(n, 5_000_000, seed=6).T)).cuda()
    d = (out[big].double() - ref[big].double()).abs()
    assert bool(((d <= 2e-5 * ref[big].double()) | (d <= 2e-7)).all())
    print(f"zones vs oracle max rel err {(err / np.maximum(want, 1e-30)).max():.3e}; vs default path max abs diff {float(d.max()):.3e}")


def test_full_size_other_seed_emp():
    """DESIGN.md reading Q16: another seed at the EMP-shaped size (a different tree, table and split), both variants and the
    RICHNESS_ZONES flag, 20,000 sampled pairs each against the oracle."""
    import torch
    from paper_2107_05397_b200 import binding as B
    from oracle import oracle as O
    p = synth.make_config("emp", seed=1)
    n = p.n_samples
    pairs = np.concatenate([synth.sample_pairs(n, 20000, seed=9), _structured_pairs(n)])
    idx = torch.from_numpy(synth.condensed_index(n, pairs[:, 0], pairs[:, 1])).cuda()
    args = B.to_device(p)
    for variant, flags in ((0, 0), (1, 0), (1, B.FLAG_RICHNESS_ZONES)):
        want = O.pair_list(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant, pairs)
        out = B.unifrac_dm(*args, n, variant, B.FP32, flags=flags)
        torch.cuda.synchronize()
        got = out[idx].cpu().numpy().astype(np.float64)
        del out
        err = np.abs(got - want)
        assert ((err <= 1e-5 * np.abs(want)) | (err <= 1e-7)).all(), (variant, flags, (err / np.maximum(want, 1e-30)).max())
        assert B.unifrac_last_stats()["quant_fallback"] == 0
