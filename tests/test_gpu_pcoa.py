"""Parity of unifrac_pcoa (CUDA, through the C ABI) with oracle/pcoa_oracle.py (full fp64 eigendecomposition) on the same
seeded distance matrices.  Tolerances: eigenvalues and proportions 1e-5 relative; coordinates up to a sign
per axis, 1e-4 of the axis' largest coordinate, asserted for axes whose eigenvalue is separated from its neighbours by >= 5 %
(an eigenvector inside a near-degenerate cluster is not unique to that accuracy; there the Gram matrix of the cluster's
coordinates is compared instead)."""
import os
from fractions import Fraction

import numpy as np
import pytest

from paper_2107_05397_b200 import synth

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


def _condensed_from_points(X):
    n = X.shape[0]
    iu = np.triu_indices(n, 1)
    return np.sqrt(((X[iu[0]] - X[iu[1]]) ** 2).sum(1))


def _run(B, d, n, k, **kw):
    import torch
    lam, prop, coords, its = B.unifrac_pcoa(torch.from_numpy(np.ascontiguousarray(d)).cuda(), n, k, **kw)
    torch.cuda.synchronize()
    return lam.cpu().numpy(), prop.cpu().numpy(), coords.cpu().numpy(), its


def _compare(got, want, k):
    lam, prop, coords, its = got
    wl, wc, wp = want
    assert np.all(np.abs(lam - wl) <= 1e-5 * np.abs(wl) + 1e-9 * abs(wl[0])), (lam, wl, its)
    assert np.all(np.abs(prop - wp) <= 1e-5 * np.abs(wp) + 1e-9), (prop, wp)
    checked = 0
    for a in range(k):
        gaps = [abs(wl[a] - wl[b]) for b in (a - 1, a + 1) if 0 <= b < len(wl)]
        if wl[a] <= 0 or min(gaps) < 0.05 * abs(wl[a]):
            continue
        s = np.sign(np.dot(coords[:, a], wc[:, a]))
        assert np.max(np.abs(coords[:, a] - s * wc[:, a])) <= 1e-4 * np.max(np.abs(wc[:, a])), (a, its)
        checked += 1
    return checked


def test_handworked_three_points():
    from paper_2107_05397_b200 import binding as B
    g = {}
    for line in open(os.path.join(HERE, "golden", "pcoa_3points.txt")):
        if not line.startswith("#") and line.strip():
            key, *v = line.split()
            g[key] = v
    d = np.array([float(t) for t in g["d"]])
    lam, prop, coords, _ = _run(B, d, 3, 2)
    assert lam[0] == pytest.approx(14 / 3, rel=1e-6) and abs(lam[1]) <= 1e-6
    want = np.array([float(Fraction(t)) for t in g["coords_axis1"]])
    assert coords[:, 0] * np.sign(coords[2, 0]) == pytest.approx(want, abs=1e-5)
    assert prop[0] == pytest.approx(1.0, rel=1e-6)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("n,dim,seed", [(50, 3, 0), (129, 4, 1), (300, 5, 2), (1000, 6, 3), (2048, 5, 4)])
def test_points_with_noise_match_oracle(n, dim, seed, dtype):
    """Points in R^dim with distinct spreads plus a non-Euclidean perturbation of the distances (so B also has small negative
    eigenvalues); sizes span one to sixteen 128-row tiles with ragged tails."""
    from paper_2107_05397_b200 import binding as B
    from oracle import pcoa_oracle as O
    rng = np.random.default_rng(seed)
    X = rng.normal(size=(n, dim)) * (1.6 ** -np.arange(dim))[None, :]
    d = _condensed_from_points(X) * (1.0 + 0.02 * rng.random(n * (n - 1) // 2))
    d = d.astype(dtype)
    k = dim
    got = _run(B, d, n, k, max_iter=400, tol=1e-10)
    want = O.pcoa(d.astype(np.float64), n, k)
    assert _compare(got, want, k) >= dim - 1


def test_pcoa_of_unifrac_matrices_small_config():
    """The use the paper describes: PCoA of the UniFrac matrices themselves (Small config, fp32 straight from unifrac_dm)."""
    import torch
    from paper_2107_05397_b200 import binding as B
    from oracle import pcoa_oracle as O
    p = synth.make_config("small", seed=0)
    args = B.to_device(p)
    n = p.n_samples
    for variant in (0, 1):
        dm = B.unifrac_dm(*args, n, variant, B.FP32)
        lam, prop, coords, its = B.unifrac_pcoa(dm, n, 5, max_iter=600, tol=1e-10)
        torch.cuda.synchronize()
        want = O.pcoa(dm.cpu().numpy().astype(np.float64), n, 5)
        _compare((lam.cpu().numpy(), prop.cpu().numpy(), coords.cpu().numpy(), its), want, 5)
        print(f"variant {variant}: {its} products, eigenvalues {lam.cpu().numpy()}, proportions {prop.cpu().numpy()}")


def test_pcoa_argument_errors():
    import torch
    from paper_2107_05397_b200 import binding as B
    d = torch.rand(10, device="cuda")
    for n, k in ((5, 0), (5, 17), (5, 5), (2, 1)):
        with pytest.raises(B.UnifracError):
            B.unifrac_pcoa(torch.rand(max(1, n * (n - 1) // 2), device="cuda"), n, k)
    del d


def test_pcoa_eigen_equation_at_a_size_beyond_the_oracle():
    """N = 8,192 (64 row tiles, 4 waves of CTAs): a full eigendecomposition on the CPU would take minutes, so the property is
    checked instead: every returned axis satisfies B c = lambda c against the Gower-centred matrix rebuilt in fp64 with torch on
    the GPU (test-side arithmetic only), eigenvalues are descending, proportions = lambda / trace(B)."""
    import torch
    from paper_2107_05397_b200 import binding as B
    rng = np.random.default_rng(8)
    n, dim = 8192, 6
    X = rng.normal(size=(n, dim)) * (1.5 ** -np.arange(dim))[None, :]
    d = (_condensed_from_points(X) * (1.0 + 0.01 * rng.random(n * (n - 1) // 2))).astype(np.float32)
    dd = torch.from_numpy(d).cuda()
    lam, prop, coords, its = B.unifrac_pcoa(dd, n, 6, max_iter=400, tol=1e-9)
    torch.cuda.synchronize()
    D = torch.zeros((n, n), dtype=torch.float64, device="cuda")
    iu = torch.triu_indices(n, n, 1, device="cuda")
    D[iu[0], iu[1]] = dd.double()
    D = D + D.T
    A = -0.5 * D * D
    Bm = A - A.mean(1, keepdim=True) - A.mean(0, keepdim=True) + A.mean()
    res = (Bm @ coords - coords * lam[None, :]).norm(dim=0) / (lam.abs() * coords.norm(dim=0))
    assert bool((res <= 2e-5).all()), res
    assert bool((lam[:-1] >= lam[1:]).all())
    assert torch.allclose(prop, lam / torch.trace(Bm), rtol=1e-6)
