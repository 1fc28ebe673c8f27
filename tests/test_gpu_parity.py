"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json:5's: 1e-10 relative (fp64), 1e-5 relative
(fp32); the absolute clause (1e-12 / 1e-7, reading Q12) only matters for d ~ 0."""
import numpy as np
import pytest

from paper_2107_05397_b200 import synth

pytestmark = pytest.mark.gpu

U, W = 0, 1
RTOL = {0: 1e-5, 1: 1e-10}       # precision enum -> rtol
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
    args = B.to_device(p)
    out = B.unifrac_dm(*args, p.n_samples, variant, precision, flags=flags)
    torch.cuda.synchronize()
    return out.cpu().numpy().astype(np.float64)


def check(got, want, precision):
    err = np.abs(got - want)
    ok = (err <= RTOL[precision] * np.abs(want)) | (err <= ATOL[precision])
    rel = err / np.maximum(np.abs(want), 1e-300)
    assert ok.all(), f"max rel err {rel[~ok].max():.3e} at {np.argmax(~ok)} (got {got[np.argmax(~ok)]}, want {want[np.argmax(~ok)]})"
    return float(rel[np.abs(want) > 1e-6].max()) if (np.abs(want) > 1e-6).any() else 0.0


@pytest.mark.parametrize("variant", [U, W])
@pytest.mark.parametrize("precision", [1, 0])
@pytest.mark.parametrize("flags", [0, 128, 16, 32, 8, 1])   # head/mid/tail split (default), no mid, all head, all tail, direct |u-v| form, literal
def test_tiny_all_pairs(B, O, variant, precision, flags):
    p = synth.make_config("tiny", seed=0)
    want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant)
    check(gpu_dm(B, p, variant, precision, flags), want, precision)


@pytest.mark.parametrize("variant", [U, W])
@pytest.mark.parametrize("precision", [1, 0])
@pytest.mark.parametrize("flags", [0, 128, 64, 16, 32, 8, 512, 256, 4])
def test_three_tiles_ragged_tail_all_pairs(B, O, variant, precision, flags):
    """300 samples = 2 full 128-tiles + a 44-sample tail; 3000 tips -> 5998 branches (several stages)."""
    p = synth.make_problem(3000, 300, 0.1, 1.1, synth.CONFIGS["small"][4], synth.CONFIGS["small"][5], seed=3)
    want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant)
    check(gpu_dm(B, p, variant, precision, flags), want, precision)


@pytest.mark.parametrize("name", ["tiny", "three_tiles", "deep"])
def test_tensor_core_gram_path_unweighted_fp32(B, O, name):
    """UNIFRAC_FLAG_TENSOR_GRAM: head branches through the tcgen05 int8 Gram kernel (24-bit fixed-point
    lengths, exact int32 accumulation), tail branches through the scatter; same 1e-5 tolerance."""
    if name == "tiny":
        p = synth.make_config("tiny", seed=0)
    elif name == "three_tiles":
        p = synth.make_problem(3000, 300, 0.1, 1.1, synth.CONFIGS["small"][4], synth.CONFIGS["small"][5], seed=3)
    else:
        p = synth.make_problem(12000, 700, 0.05, 1.05, synth.CONFIGS["small"][4], synth.CONFIGS["small"][5], seed=5)
    want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, U)
    for flags in (0, B.FLAG_NO_TAIL):                 # default head/tail split; dense GEMM over every branch
        got = gpu_dm(B, p, U, 0, flags=flags)
        st = B.unifrac_last_stats()
        assert st["gram"] == 1 and st["gram_k"] >= st["head_rows"] > 0
        rel = check(got, want, 0)
        print(f"gram {name} flags {flags}: head {st['head_rows']} tail {st['tail_rows']} q {st['gram_q']} max rel err {rel:.3e}")
    got = gpu_dm(B, p, U, 0, flags=B.FLAG_NO_TENSOR)
    assert B.unifrac_last_stats()["gram"] == 0
    check(got, want, 0)


@pytest.mark.parametrize("n_samples", [2, 3, 127, 128, 129, 257])
def test_tile_boundary_sample_counts(B, O, n_samples):
    p = synth.make_problem(400, n_samples, 0.1, 1.1, synth._k_poisson40, synth._c_geometric, seed=n_samples)
    for variant in (U, W):
        want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant)
        check(gpu_dm(B, p, variant, 1), want, 1)
        check(gpu_dm(B, p, variant, 0), want, 0)


@pytest.mark.parametrize("seed", range(5))
def test_general_trees_multifurcation_unary_zero_length(B, O, seed):
    rng = np.random.default_rng(500 + seed)
    parent, bl = synth.random_tree(int(rng.integers(5, 400)), rng, p_unary=0.25, p_zero_len=0.25)
    tips = synth.tip_ids(parent)
    p = synth.problem_from_parent(parent, bl, synth.random_table(tips, int(rng.integers(2, 150)), rng, density=0.2))
    for variant in (U, W):
        want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant)
        for flags in (0, 16, 32, 8, 1):
            check(gpu_dm(B, p, variant, 1, flags), want, 1)
        for flags in (0, 16, 32, 64, 64 + 16, 128, 64 + 128):
            check(gpu_dm(B, p, variant, 0, flags), want, 0)


def test_zero_denominator_gives_zero(B):
    parent, bl = synth.star_tree(3, [0.0, 0.0, 1.0])
    p = synth.problem_from_parent(parent, bl, [{0: 1}, {1: 2}, {2: 1}])
    for variant in (U, W):
        for flags in (0, 16, 32, 8, 1):
            d = gpu_dm(B, p, variant, 1, flags)
            assert d[0] == 0.0 and d[1] == 1.0 and d[2] == 1.0


def test_small_config_sampled_pairs(B, O):
    """BASELINE.json config 'Small' (20k tips, 2048 samples, fp64, both variants): 20k seeded pairs +
    tile-boundary neighbours + first/last condensed elements via the oracle's pair-list driver."""
    p = synth.make_config("small", seed=0)
    n = p.n_samples
    pairs = synth.sample_pairs(n, 20000, seed=0)
    extra = np.array([[0, 1], [0, n - 1], [n - 2, n - 1], [127, 128], [0, 128], [127, 255], [128, 129],
                      [1919, 1920], [2047 - 128, 2047]], dtype=np.int32)
    pairs = np.concatenate([pairs, extra])
    idx = synth.condensed_index(n, pairs[:, 0], pairs[:, 1])
    for variant in (U, W):
        want = O.pair_list(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant, pairs)
        got = gpu_dm(B, p, variant, 1)
        check(got[idx], want, 1)
        got32 = gpu_dm(B, p, variant, 0)
        check(got32[idx], want, 0)
        assert np.all(got >= 0) and np.all(got <= 1)
        st = B.unifrac_last_stats()
        assert st["head_rows"] > 0 and st["tail_rows"] > 0 and st["mid_rows"] > 0     # the default split uses all three paths here
        check(gpu_dm(B, p, variant, 0, flags=128)[idx], want, 0)    # head + tail only
        check(gpu_dm(B, p, variant, 0, flags=16)[idx], want, 0)     # all head
        check(gpu_dm(B, p, variant, 0, flags=64)[idx], want, 0)     # CUDA-core head for unweighted too


def test_host_entry_point_matches_device_entry_point(B, O):
    p = synth.make_config("tiny", seed=2)
    for variant in (U, W):
        want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant)
        got = B.unifrac_dm_host(p.parent, p.branch_len, p.postorder, p.indptr, p.indices, p.counts,
                                p.n_samples, variant, B.FP64)
        check(got, want, 1)
        got32 = B.unifrac_dm_host(p.parent, p.branch_len, p.postorder, p.indptr, p.indices, p.counts,
                                  p.n_samples, variant, B.FP32).astype(np.float64)
        check(got32, want, 0)


def test_error_codes(B):
    import torch
    p = synth.make_config("tiny", seed=0)

    def rc_of(**kw):
        q = synth.Problem(kw.get("parent", p.parent), kw.get("bl", p.branch_len), kw.get("post", p.postorder),
                          kw.get("indptr", p.indptr), kw.get("indices", p.indices), kw.get("counts", p.counts))
        try:
            B.unifrac_dm(*B.to_device(q), q.n_samples, U, B.FP64)
            torch.cuda.synchronize()
            return 0
        except B.UnifracError as e:
            return e.status

    assert rc_of() == 0
    bad = p.parent.copy(); bad[5] = -1
    assert rc_of(parent=bad) == B.ERR_INVALID_TREE                       # two roots
    bad = p.parent.copy(); bad[5] = p.n_nodes + 3
    assert rc_of(parent=bad) == B.ERR_INVALID_TREE
    post = p.postorder.copy(); post[[0, -1]] = post[[-1, 0]]
    assert rc_of(post=post) == B.ERR_INVALID_TREE                        # root not last
    post = p.postorder.copy(); post[3] = post[4]
    assert rc_of(post=post) == B.ERR_INVALID_TREE                        # not a permutation
    bl = p.branch_len.copy(); bl[7] = -1.0
    assert rc_of(bl=bl) == B.ERR_INVALID_TREE
    bl = p.branch_len.copy(); bl[7] = np.nan
    assert rc_of(bl=bl) == B.ERR_INVALID_TREE
    idx = p.indices.copy(); idx[0] = 0                                   # node 0 is the root (internal)
    assert rc_of(indices=idx) == B.ERR_INVALID_TABLE
    idx = p.indices.copy(); idx[[0, 1]] = idx[[1, 0]]
    assert rc_of(indices=idx) == B.ERR_INVALID_TABLE                     # not increasing
    cnt = p.counts.copy(); cnt[3] = -2
    assert rc_of(counts=cnt) == B.ERR_INVALID_TABLE
    cnt = p.counts.copy(); cnt[p.indptr[4]:p.indptr[5]] = 0
    assert rc_of(counts=cnt) == B.ERR_EMPTY_SAMPLE


def test_stats_work_counters_match_definitions(B):
    """W_dense / W_union / W_inter against their closed forms computed from presence."""
    import torch
    import refmath
    p = synth.make_config("tiny", seed=4)
    B.unifrac_dm(*B.to_device(p), p.n_samples, U, B.FP64)
    torch.cuda.synchronize()
    st = B.unifrac_last_stats()
    A, tips = refmath.ancestor_matrix(p.parent)
    X = refmath.dense_counts(p, tips)
    pres = (X @ A.T) > 0
    keep = (p.parent >= 0) & (p.branch_len > 0)
    nv = pres[:, keep].sum(0)
    N = p.n_samples
    assert st["branches_embedded"] == int((nv > 0).sum())
    assert st["updates_dense"] == int((nv > 0).sum()) * N * (N - 1) // 2
    assert st["updates_inter"] == int((nv * (nv - 1) // 2).sum())
    assert st["updates_union"] == int((N * (N - 1) // 2 - (N - nv) * (N - nv - 1) // 2)[nv > 0].sum())
    assert st["updates_executed"] > 0 and st["kernel_launches"] > 0 and st["stripe_launches"] == 1
    assert st["head_rows"] + st["tail_rows"] + st["mid_rows"] == st["branches_embedded"]
    tail = nv[(nv > 0)]
    B.unifrac_dm(*B.to_device(p), p.n_samples, U, B.FP64, flags=B.FLAG_ALL_TAIL)
    torch.cuda.synchronize()
    st = B.unifrac_last_stats()
    assert st["head_rows"] == 0 and st["tail_updates"] == int((tail * (tail - 1) // 2).sum())
    assert st["tail_entries"] == int(tail.sum()) and st["updates_executed"] == st["tail_updates"]


@pytest.mark.parametrize("variant,precision", [(U, 0), (W, 0), (W, 1)])
def test_shards_partition_the_matrix(B, O, variant, precision):
    """unifrac_dm_shard: the shards' buffers are disjoint (a pair is non-zero only in the shard
    unifrac_shard_of_pair names) and their sum is the matrix -- checked against the oracle on sampled pairs and
    against the unsharded call.  26 tiles = 3 block rows of 12 tiles, ragged last tile."""
    import torch
    cfg = synth.CONFIGS["small"]
    p = synth.make_problem(3000, 3300, 0.1, 1.1, cfg[4], cfg[5], seed=3)
    n, S = p.n_samples, 4
    pairs = np.concatenate([synth.sample_pairs(n, 6000, seed=1),
                            np.array([[0, 1], [0, n - 1], [n - 2, n - 1], [1535, 1536], [0, 1536], [1536, 3072],
                                      [3071, 3072], [1535, 3299]], dtype=np.int32)])
    idx = synth.condensed_index(n, pairs[:, 0], pairs[:, 1])
    want = O.pair_list(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant, pairs)
    args = B.to_device(p)
    full = B.unifrac_dm(*args, n, variant, precision)
    total = torch.zeros_like(full)
    owners = np.array([B.unifrac_shard_of_pair(int(i), int(j), S) for i, j in pairs])
    assert set(owners.tolist()) == set(range(S))
    for s in range(S):
        part = B.unifrac_dm(*args, n, variant, precision, shard=(s, S))
        torch.cuda.synchronize()
        got = part[torch.from_numpy(idx).cuda()].cpu().numpy().astype(np.float64)
        assert np.all(got[owners != s] == 0.0)
        check(got[owners == s], want[owners == s], precision)
        assert int(torch.count_nonzero(part)) <= int(torch.count_nonzero(full))
        total += part
    torch.cuda.synchronize()
    a, b = total.cpu().numpy().astype(np.float64), full.cpu().numpy().astype(np.float64)
    assert np.allclose(a, b, rtol=2e-6 if precision == 0 else 1e-12, atol=1e-7 if precision == 0 else 1e-13)
    with pytest.raises(B.UnifracError):
        B.unifrac_dm(*args, n, variant, precision, shard=(4, 4))


@pytest.mark.parametrize("seed", [1, 2])
@pytest.mark.parametrize("variant", [U, W])
def test_other_seeds_six_tiles_all_pairs_fp32_and_fp64(B, O, variant, seed):
    """DESIGN.md reading Q16: seeds 1 and 2 as extra parity runs.  700 samples = 6 tiles (ragged last one), 8,000 tips:
    all 244,650 pairs against the oracle's all-pairs driver, default split (head + mid + tail all non-empty in fp32)."""
    cfg = synth.CONFIGS["small"]
    p = synth.make_problem(8000, 700, 0.05, 1.05, cfg[4], cfg[5], seed=seed)
    want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant)
    check(gpu_dm(B, p, variant, 1), want, 1)
    check(gpu_dm(B, p, variant, 0), want, 0)
    st = B.unifrac_last_stats()
    assert st["head_rows"] > 0 and st["tail_rows"] > 0


@pytest.mark.parametrize("seed", [1, 2])
def test_richness_zones_flag_weighted_fp32(B, O, seed):
    """UNIFRAC_FLAG_RICHNESS_ZONES: samples sorted by richness inside the call, k_zone for the tile pairs inside a branch's dense
    zone, the join for the rest, result un-permuted -- all 244,650 pairs of a 6-tile problem against the oracle, and the stats
    say that both kernels had work.  A table whose poorest and richest samples differ by 30x makes the zones non-trivial."""
    cfg = synth.CONFIGS["small"]
    p = synth.make_problem(8000, 700, 0.05, 1.05, cfg[4], cfg[5], seed=seed)
    rows = synth.rows_of(p)
    for s in range(0, 700, 3):                                  # thin every third sample down to ~1/10 of its features
        keys = sorted(rows[s])
        rows[s] = {t: rows[s][t] for t in keys[::10]} or {keys[0]: 1}
    p = synth.with_rows(p, rows)
    want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, W)
    check(gpu_dm(B, p, W, 0, flags=B.FLAG_RICHNESS_ZONES), want, 0)
    st = B.unifrac_last_stats()
    assert st["skip"] == 1 and st["skip_row_pair_visits"] > 0 and st["mid_updates"] > 0 and st["tail_rows"] > 0
    assert 0 < st["skip_rows"] <= st["list_rows"]
    check(gpu_dm(B, p, U, 0, flags=B.FLAG_RICHNESS_ZONES), O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, U), 0)   # ignored for unweighted


def test_measure_rates_probe(B):
    """unifrac_measure_rates (the peaks of the k_mid / k_tail_scatter rooflines): positive, plausible, repeatable to 10 %."""
    a, b = B.unifrac_measure_rates(), B.unifrac_measure_rates()
    for k in ("smem_atomic_conflict_free_per_s", "smem_atomic_random_per_s", "l2_red_random_per_s"):
        assert a[k] > 1e10 and abs(a[k] - b[k]) <= 0.1 * a[k]
    assert a["sm_count"] > 0 and a["sm_clock_khz"] > 0
    assert a["smem_atomic_random_per_s"] <= a["sm_count"] * a["sm_clock_khz"] * 1e3 * 32     # at most one full wavefront per clock


@pytest.mark.parametrize("case", range(8))
def test_randomized_shapes_all_pairs(B, O, case):
    """Seeded random shapes (tips 50..6000, samples 2..900, the count / richness recipes, branch-length scale and Zipf
    exponent varied): all pairs, both variants, fp32 and fp64, default split and head + tail only."""
    rng = np.random.default_rng(1000 + case)
    n_tips = int(rng.integers(50, 6000))
    n = int(rng.integers(2, 900))
    # the richer recipes need enough tips (the generator draws features until k of them are distinct)
    names = ["tiny"] if n_tips < 500 else ["tiny", "small"] if n_tips < 3000 else ["tiny", "small", "medium"]
    cfg = synth.CONFIGS[names[int(rng.integers(0, len(names)))]]
    p = synth.make_problem(n_tips, n, float(rng.choice([0.05, 0.1, 1.0])), float(rng.choice([1.05, 1.1, 1.3])), cfg[4], cfg[5],
                           seed=int(rng.integers(0, 10**6)))
    for variant in (U, W):
        want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant)
        for precision in (0, 1):
            for flags in (0, 128):
                check(gpu_dm(B, p, variant, precision, flags), want, precision)


@pytest.mark.parametrize("variant", [U, W])
def test_two_shards_on_two_streams_merge_to_the_oracle_matrix(B, O, variant):
    """The N > 1 path of bench.py on one GPU: shards 0 and 1 of 2 run on two streams into two buffers; their element-wise sum
    (what multigpu.merge_shards' all-reduce(SUM) produces) is compared with the oracle on EVERY pair.  1,700 samples = 14
    tiles = blocks (0,0), (0,1), (1,1) of 12 x 12 tiles dealt to shards 0, 1, 0."""
    import torch
    cfg = synth.CONFIGS["small"]
    p = synth.make_problem(3000, 1700, 0.1, 1.1, cfg[4], cfg[5], seed=5)
    n = p.n_samples
    want = O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, variant)
    args = B.to_device(p)
    torch.cuda.synchronize()
    s0, s1 = torch.cuda.Stream(), torch.cuda.Stream()
    a = B.unifrac_dm(*args, n, variant, B.FP32, shard=(0, 2), stream=s0)
    b = B.unifrac_dm(*args, n, variant, B.FP32, shard=(1, 2), stream=s1)
    torch.cuda.synchronize()
    assert int(torch.count_nonzero((a != 0) & (b != 0))) == 0          # disjoint owners
    assert int(torch.count_nonzero(a)) > 0 and int(torch.count_nonzero(b)) > 0
    check((a + b).cpu().numpy().astype(np.float64), want, 0)


def test_unifrac_dm_returns_before_the_stripe_kernel_finishes(B):
    """include/unifrac_b200.h: "after planning and embedding the stripe kernel is enqueued asynchronously and the call returns
    without waiting for it".  Medium-sized weighted call (~100 ms of a-5 kernels): an event recorded right after the call
    returns has not completed yet; the result is still correct once it has."""
    import torch
    cfg = synth.CONFIGS["medium"]
    p = synth.make_problem(30000, 6000, 0.05, 1.05, cfg[4], cfg[5], seed=2)
    args = B.to_device(p)
    B.unifrac_dm(*args, p.n_samples, W, B.FP32)                      # warm-up (module load, allocator)
    torch.cuda.synchronize()
    ev = torch.cuda.Event()
    out = B.unifrac_dm(*args, p.n_samples, W, B.FP32)
    ev.record()
    pending = not ev.query()
    torch.cuda.synchronize()
    assert pending, "unifrac_dm waited for its a-5 kernels"
    assert bool(torch.isfinite(out).all()) and float(out.max()) <= 1.0


def test_host_multi_matches_device_entry_point(B, O):
    """unifrac_dm_host_multi (both variants, inputs uploaded once, result copies overlapping the next variant's compute)
    returns what unifrac_dm returns; unifrac_release_host_pool afterwards."""
    import torch
    cfg = synth.CONFIGS["small"]
    p = synth.make_problem(3000, 300, 0.1, 1.1, cfg[4], cfg[5], seed=4)
    outs = B.unifrac_dm_host_multi(p.parent, p.branch_len, p.postorder, p.indptr, p.indices, p.counts, p.n_samples, [U, W], B.FP32)
    for v, got in zip((U, W), outs):
        dev = gpu_dm(B, p, v, 0)
        assert np.allclose(got.astype(np.float64), dev, rtol=2e-6, atol=1e-7)     # last bits: the tail's REDs arrive in arbitrary order
        check(got.astype(np.float64), O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, v), 0)
    one = B.unifrac_dm_host(p.parent, p.branch_len, p.postorder, p.indptr, p.indices, p.counts, p.n_samples, W, B.FP64)
    check(one, O.all_pairs(p.parent, p.branch_len, p.indptr, p.indices, p.counts, W), 1)
    B.unifrac_release_host_pool()
