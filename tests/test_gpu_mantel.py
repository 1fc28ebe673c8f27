"""Parity of unifrac_mantel_pearson (CUDA, through the C ABI) with oracle/mantel_oracle.py on the same seeded inputs:
statistic, every permuted statistic and the three p-values.  Tolerance: 1e-10 absolute on correlations for fp64 inputs;
for fp32 inputs the oracle is given the same fp32-rounded data, so the tolerance stays 1e-10 (all sums are fp64 on both
sides)."""
import numpy as np
import pytest

from paper_2107_05397_b200 import synth

pytestmark = pytest.mark.gpu


def _case(n, K, seed, dtype):
    rng = np.random.default_rng(seed)
    P = n * (n - 1) // 2
    x = rng.random(P)
    y = 0.3 * x + 0.7 * rng.random(P)            # correlated matrices, r ~ 0.4
    perms = np.stack([rng.permutation(n) for _ in range(K)]).astype(np.int32) if K else np.zeros((0, n), np.int32)
    return x.astype(dtype), y.astype(dtype), perms


def _run(B, x, y, n, perms):
    import torch
    out = B.unifrac_mantel_pearson(torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda(), n,
                                   torch.from_numpy(np.ascontiguousarray(perms)).cuda())
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("n,K", [(3, 4), (33, 7), (257, 25), (700, 12)])
def test_mantel_matches_oracle(n, K, dtype):
    from paper_2107_05397_b200 import binding as B
    from oracle import mantel_oracle as M
    x, y, perms = _case(n, K, seed=n + K, dtype=dtype)
    got = _run(B, x, y, n, perms)
    r, p2, pg, pl, rk = M.mantel_pearson(x.astype(np.float64), y.astype(np.float64), n, perms)
    assert abs(got[0] - r) <= 1e-10
    assert np.max(np.abs(got[4:] - rk)) <= 1e-10
    if min(np.min(np.abs(rk - r)), np.min(np.abs(np.abs(rk) - abs(r)))) > 1e-9:     # counts are well defined unless a permuted value ties r
        assert got[1] == pytest.approx(p2, abs=1e-12) and got[2] == pytest.approx(pg, abs=1e-12) and got[3] == pytest.approx(pl, abs=1e-12)


def test_mantel_edge_cases():
    from paper_2107_05397_b200 import binding as B
    import torch
    n = 40
    x, y, perms = _case(n, 5, seed=1, dtype=np.float64)
    ident = np.arange(n, dtype=np.int32)[None, :]
    got = _run(B, x, y, n, ident)
    assert abs(got[4] - got[0]) <= 1e-13 and got[1] == 1.0                      # identity permutation reproduces r
    assert abs(_run(B, x, 2.0 * x + 1.0, n, ident)[0] - 1.0) <= 1e-12          # Y = aX + b
    assert _run(B, np.full_like(x, 0.5), y, n, ident)[0] == 0.0               # zero variance -> 0 (reading M4)
    assert _run(B, np.full_like(x, 0.3), y, n, ident)[0] == 0.0               # ... also when the constant does not sum exactly
    assert _run(B, x, np.full_like(y, 0.1), n, ident)[0] == 0.0
    assert _run(B, np.full_like(x, 0.3, dtype=np.float32), y.astype(np.float32), n, ident)[0] == 0.0
    got0 = _run(B, x, y, n, np.zeros((0, n), np.int32))                        # no permutations: p = 1 / 1
    assert got0.shape == (4,) and got0[1] == 1.0
    with pytest.raises(B.UnifracError):
        B.unifrac_mantel_pearson(torch.zeros(1, device="cuda"), torch.zeros(1, device="cuda"), 2,
                                 torch.zeros(0, dtype=torch.int32, device="cuda"))


def test_mantel_on_unifrac_matrices_and_sampled_property_at_scale():
    """The use the paper describes: correlate two distance matrices of the same samples (here unweighted vs
    weighted-normalized UniFrac of the Small config, fp32, straight from unifrac_dm) -- r against the oracle on the same
    data; and at N = 6000 (18 M pairs, beyond what the oracle does per permutation in seconds) properties that hold at any
    size: identity permutation = r, permuting both matrices' objects consistently leaves r unchanged."""
    import torch
    from paper_2107_05397_b200 import binding as B
    from oracle import mantel_oracle as M
    p = synth.make_config("small", seed=0)
    args = B.to_device(p)
    du = B.unifrac_dm(*args, p.n_samples, 0, B.FP32)
    dw = B.unifrac_dm(*args, p.n_samples, 1, B.FP32)
    rng = np.random.default_rng(3)
    perms = np.stack([rng.permutation(p.n_samples) for _ in range(3)]).astype(np.int32)
    got = B.unifrac_mantel_pearson(du, dw, p.n_samples, torch.from_numpy(perms).cuda()).cpu().numpy()
    r, p2, pg, pl, rk = M.mantel_pearson(du.cpu().numpy().astype(np.float64), dw.cpu().numpy().astype(np.float64), p.n_samples, perms)
    assert abs(got[0] - r) <= 1e-10 and np.max(np.abs(got[4:] - rk)) <= 1e-10 and got[0] > 0.2
    n = 6000
    x, y, _ = _case(n, 0, seed=9, dtype=np.float32)
    pi = rng.permutation(n).astype(np.int32)
    base = _run(B, x, y, n, np.stack([np.arange(n, dtype=np.int32), pi]))
    assert abs(base[4] - base[0]) <= 1e-12
    # relabel the objects of y by pi as well: r(X^pi, Y^pi) = r(X, Y)
    iu = np.triu_indices(n, 1)
    Y = np.zeros((n, n), np.float32); Y[iu] = y; Y = Y + Y.T
    y_pi = np.ascontiguousarray(Y[np.ix_(pi, pi)][iu])
    both = _run(B, x, y_pi, n, pi[None, :])
    assert abs(both[4] - base[0]) <= 1e-10


@pytest.mark.parametrize("bufs", ["", "2"])
def test_mantel_row_longer_than_one_ring_buffer(bufs, monkeypatch):
    """fp64, N = 14,000: a row of the square copy is 112 KB, so two whole rows do not fit in shared memory.  Default: ONE
    whole-row buffer (the path N = 50,000 takes in fp32); UNIFRAC_B200_MANTEL_BUFS=2: two buffers of half a row, every row
    staged in two column segments (the path of rows beyond 208 KB).  One permutation against the oracle, identity against r."""
    from paper_2107_05397_b200 import binding as B
    from oracle import mantel_oracle as M
    if bufs:
        monkeypatch.setenv("UNIFRAC_B200_MANTEL_BUFS", bufs)
    else:
        monkeypatch.delenv("UNIFRAC_B200_MANTEL_BUFS", raising=False)
    n = 14000
    x, y, perms = _case(n, 1, seed=4, dtype=np.float64)
    perms = np.concatenate([perms, np.arange(n, dtype=np.int32)[None, :]])
    got = _run(B, x, y, n, perms)
    r, _, _, _, rk = M.mantel_pearson(x, y, n, perms[:1])
    assert abs(got[0] - r) <= 1e-10 and abs(got[4] - rk[0]) <= 1e-10 and got[5] == got[0]


# ------------------------------------------------------------------------------------------------ Spearman
def _run_s(B, x, y, n, perms):
    import torch
    out = B.unifrac_mantel_spearman(torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda(), n,
                                    torch.from_numpy(np.ascontiguousarray(perms)).cuda())
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("n,K,ties", [(3, 4, False), (33, 7, True), (257, 9, True), (700, 5, False), (700, 4, True)])
def test_mantel_spearman_matches_oracle(n, K, ties, dtype):
    """rho, every permuted rho and the p-values against oracle/mantel_oracle.py::mantel_spearman (which ranks the permuted
    triangle again for every permutation).  With `ties` the values are rounded to 2 decimals, so runs of equal values span
    radix-sort tiles and blocks; signs and zeros (+0 / -0) are mixed in as well."""
    from paper_2107_05397_b200 import binding as B
    from oracle import mantel_oracle as M
    x, y, perms = _case(n, K, seed=3 * n + K, dtype=np.float64)
    x = x - 0.5                                                   # negative keys exercise the sign flip of the key map
    if ties:
        x, y = np.round(x, 2), np.round(y, 1)
        x[x == 0.0] = -0.0                                        # -0 and +0 are the same value: one run
        x[::7] = 0.0
    x, y = x.astype(dtype), y.astype(dtype)
    got = _run_s(B, x, y, n, perms)
    r, p2, pg, pl, rk = M.mantel_spearman(x.astype(np.float64), y.astype(np.float64), n, perms)
    assert abs(got[0] - r) <= 1e-10
    assert np.max(np.abs(got[4:] - rk)) <= 1e-10
    if min(np.min(np.abs(rk - r)), np.min(np.abs(np.abs(rk) - abs(r)))) > 1e-9:
        assert got[1] == pytest.approx(p2, abs=1e-12) and got[2] == pytest.approx(pg, abs=1e-12) and got[3] == pytest.approx(pl, abs=1e-12)


def test_mantel_spearman_properties_at_scale():
    """N = 6000 (18 M pairs: 4,400 radix tiles over 1,184 block ranges): rho is invariant under strictly increasing maps of
    either matrix, equals Pearson of the oracle-free closed form for a monotone pair (1), and a constant matrix gives 0."""
    from paper_2107_05397_b200 import binding as B
    n = 6000
    x, y, _ = _case(n, 0, seed=21, dtype=np.float32)
    ident = np.arange(n, dtype=np.int32)[None, :]
    a = _run_s(B, x, y, n, ident)
    b = _run_s(B, np.exp(3.0 * x).astype(np.float32), (y.astype(np.float64) ** 3).astype(np.float32), n, ident)
    assert abs(a[0] - b[0]) <= 1e-9 and abs(a[4] - a[0]) <= 1e-12
    assert abs(_run_s(B, x, np.sqrt(x), n, ident)[0] - 1.0) <= 1e-12
    assert _run_s(B, np.full_like(x, 0.3), y, n, ident)[0] == 0.0
    # fp64 keys (8 digit passes), two-segment rows: N = 14,000 against the Pearson entry point on host-made ranks
    from scipy import stats
    n = 14000
    x, y, perms = _case(n, 1, seed=5, dtype=np.float64)
    x = np.round(x, 3)
    got = _run_s(B, x, y, n, perms)
    want = _run(B, stats.rankdata(x), stats.rankdata(y), n, perms)
    assert abs(got[0] - want[0]) <= 1e-10 and abs(got[4] - want[4]) <= 1e-10
