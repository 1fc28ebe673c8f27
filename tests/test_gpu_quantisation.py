"""Inputs chosen against the fixed-point representations of the fp32 path (tensor-core Gram: per-row-shifted 24-bit
lengths; shared-memory mid kernel: 32-bit fixed-point accumulators): branch lengths spread over six decades, many
identical lengths plus one very long branch, one sample whose side sum is ~100x the others.  The library tracks the
exact per-sample sum of |fixed-point value - value| and reruns without the fixed-point kernels when its ratio to
the side sum is over budget (unifrac_last_stats: quant_err_ratio, quant_fallback); either way the result must meet
BASELINE.json:5's 1e-5 relative tolerance against the oracle."""
import numpy as np
import pytest

from paper_2107_05397_b200 import synth

pytestmark = pytest.mark.gpu

U, W = 0, 1


@pytest.fixture(scope="module")
def B():
    from paper_2107_05397_b200 import binding
    binding.load()
    return binding


@pytest.fixture(scope="module")
def O():
    from oracle import oracle
    return oracle


def run_and_check(B, O, p, variant, label):
    import torch
    want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant)
    out = B.unifrac_dm(*B.to_device(p), p.n_samples, variant, B.FP32)
    torch.cuda.synchronize()
    got = out.cpu().numpy().astype(np.float64)
    st = B.unifrac_last_stats()
    err = np.abs(got - want)
    ok = (err <= 1e-5 * np.abs(want)) | (err <= 1e-7)
    rel = err / np.maximum(np.abs(want), 1e-300)
    print(f"{label} variant {variant}: max rel err {rel[want > 1e-6].max():.3e} quant_err_ratio {st['quant_err_ratio']:.3e} "
          f"fallback {st['quant_fallback']} gram {st['gram']} mid_rows {st['mid_rows']} mid_F {st['mid_F']}")
    assert ok.all(), f"{label}: max rel err {rel[~ok].max():.3e}"
    return st


def _base(seed):
    cfg = synth.CONFIGS["small"]
    return synth.make_problem(4000, 400, 0.1, 1.1, cfg[4], cfg[5], seed=seed)


@pytest.mark.parametrize("variant", [U, W])
def test_log_uniform_branch_lengths_over_six_decades(B, O, variant):
    p = _base(21)
    rng = np.random.default_rng(5)
    bl = 10.0 ** rng.uniform(-4.0, 2.0, size=p.n_nodes)
    bl[p.parent < 0] = 0.0
    run_and_check(B, O, synth.with_rows(p, synth.rows_of(p), branch_len=bl), variant, "log-uniform lengths")


@pytest.mark.parametrize("ratio", [100.0, 1e4, 1e7])
@pytest.mark.parametrize("variant", [U, W])
def test_identical_lengths_plus_one_long_branch(B, O, variant, ratio):
    """Every branch 0.1 (its fixed-point error has ONE sign for all of them) except one branch near the root that is
    `ratio` times longer and sets the fixed-point scale."""
    p = _base(22)
    bl = np.full(p.n_nodes, 0.1)
    bl[p.parent < 0] = 0.0
    kids = np.nonzero(p.parent == int(np.nonzero(p.parent < 0)[0][0]))[0]
    bl[kids[0]] = 0.1 * ratio
    run_and_check(B, O, synth.with_rows(p, synth.rows_of(p), branch_len=bl), variant, f"identical + one x{ratio:g}")


@pytest.mark.parametrize("variant", [U, W])
def test_fallback_path_when_the_error_ratio_is_over_budget(B, O, variant, monkeypatch):
    """Budget forced to ~0 through the tuning environment variable: the call must rerun without the fixed-point kernels
    (no tensor-core Gram, no shared-memory mid), report it, and still meet the tolerance."""
    monkeypatch.setenv("UNIFRAC_B200_QUANT_BUDGET", "1e-30")
    st = run_and_check(B, O, _base(24), variant, "forced fallback")
    assert st["quant_fallback"] == 1 and st["gram"] == 0 and st["mid_rows"] == 0
    monkeypatch.delenv("UNIFRAC_B200_QUANT_BUDGET")
    st = run_and_check(B, O, _base(24), variant, "default budget")
    assert st["quant_fallback"] == 0 and st["mid_rows"] > 0 and st["gram"] == (1 if variant == U else 0)


@pytest.mark.parametrize("variant", [U, W])
def test_one_sample_with_a_hundred_times_the_side_sum(B, O, variant):
    """One sample observes (nearly) every tip while the others observe a handful, so its side sum S_s is ~100x theirs
    (unweighted); the fixed-point scale of the mid kernel is set by the largest per-sample sum."""
    p = _base(23)
    rows = synth.rows_of(p)
    tips = synth.tip_ids(p.parent)
    rng = np.random.default_rng(6)
    for s in range(len(rows)):
        keep = sorted(rows[s])[:max(2, len(rows[s]) // 20)]
        rows[s] = {t: rows[s][t] for t in keep}
    rows[7] = {int(t): int(rng.integers(1, 50)) for t in tips}
    rows[200] = {int(t): int(rng.integers(1, 50)) for t in tips[::2]}
    run_and_check(B, O, synth.with_rows(p, rows), variant, "one rich sample")
