"""unifrac_mantel_pearson_noalloc (include/unifrac_b200.h): the Mantel / Pearson path with its workspace in the library's
static device array instead of an allocator.  Collected last on purpose (the suite runs with pytest -x).  The output must
equal the allocating entry point's within the tolerance of tests/test_gpu_mantel.py (same kernels and launch configuration;
the moments are added across blocks with fp64 atomics, so the last bits may differ between any two runs) on two calls in a
row (the second one finds the first one's contents in the array), for other sizes and fp64 after that, and torch's
allocator must not have been asked for a byte during the calls."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL = 1e-10            # the tolerance tests/test_gpu_mantel.py uses against the oracle (both sides sum in fp64)


def _case(n, K, seed, dtype):
    rng = np.random.default_rng(seed)
    P = n * (n - 1) // 2
    x = rng.random(P).astype(dtype)
    y = (0.3 * x + rng.random(P)).astype(dtype)
    perms = np.stack([rng.permutation(n) for _ in range(K)]).astype(np.int32) if K else np.zeros((0, n), np.int32)
    return x, y, perms


def _both(B, torch, n, K, seed, dtype):
    x, y, perms = _case(n, K, seed, dtype)
    xd, yd, pd = torch.from_numpy(x).cuda(), torch.from_numpy(y).cuda(), torch.from_numpy(perms).cuda()
    ref = B.unifrac_mantel_pearson(xd, yd, n, pd)
    torch.cuda.synchronize()
    out = torch.full((4 + K,), float("nan"), dtype=torch.float64, device="cuda")
    before = torch.cuda.memory_stats()["allocation.all.allocated"]
    B.unifrac_mantel_pearson_noalloc(xd, yd, n, pd, out)
    torch.cuda.synchronize()
    assert torch.cuda.memory_stats()["allocation.all.allocated"] == before        # nothing asked of torch's allocator
    return ref.cpu().numpy(), out.cpu().numpy(), (x, y, perms)


def test_no_alloc_mantel_matches_allocating_path_on_two_calls_in_a_row():
    import torch
    from paper_2107_05397_b200 import binding as B
    from oracle import mantel_oracle as M
    for call, (n, K, dtype) in enumerate([(700, 12, np.float32), (700, 12, np.float32), (1024, 40, np.float64), (33, 0, np.float32)]):
        ref, got, (x, y, perms) = _both(B, torch, n, K, seed=100 + n + K, dtype=dtype)
        assert np.all(np.isfinite(got))
        assert np.max(np.abs(got - ref)) <= TOL, (call, n, K)
        if n == 700:                                                              # and against the oracle itself
            r, p2, pg, pl, rk = M.mantel_pearson(x.astype(np.float64), y.astype(np.float64), n, perms)
            assert abs(got[0] - r) <= TOL and np.max(np.abs(got[4:] - rk)) <= TOL


def test_no_alloc_mantel_rejects_sizes_beyond_the_static_workspace():
    import torch
    from paper_2107_05397_b200 import binding as B
    n = B.NOALLOC_MAX_SAMPLES + 1
    P = n * (n - 1) // 2
    x = torch.rand(P, device="cuda"); y = torch.rand(P, device="cuda")
    perms = torch.zeros((0, n), dtype=torch.int32, device="cuda")
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    with pytest.raises(B.UnifracError) as e:
        B.unifrac_mantel_pearson_noalloc(x, y, n, perms, out)
    assert e.value.status == B.ERR_UNSUPPORTED and "UNIFRAC_NOALLOC_MAX_SAMPLES" in str(e.value)
    n = 40
    P = n * (n - 1) // 2
    K = B.NOALLOC_MAX_PERMS + 1
    perms = torch.stack([torch.randperm(n, device="cuda") for _ in range(K)]).to(torch.int32).contiguous()
    with pytest.raises(B.UnifracError) as e:
        B.unifrac_mantel_pearson_noalloc(torch.rand(P, device="cuda"), torch.rand(P, device="cuda"), n, perms,
                                         torch.zeros(4 + K, dtype=torch.float64, device="cuda"))
    assert e.value.status == B.ERR_UNSUPPORTED
