"""Seeded synthetic inputs shaped like the paper's workloads (PAPER.md:15,21-23 -- EMP-sized,
sparse sample x feature tables over a phylogeny).  The EMP tree/table are not available, so
these stand in for them; shapes and distributions are BASELINE.json:7-11, the exact recipe is
DESIGN.md "Input recipe" (readings Q14-Q16 of SURVEY.md section 8c).

This module contains NO UniFrac arithmetic: it only draws trees and count tables.  It is the
one module shared by the CUDA path's tests/bench and the oracle's tests.
"""
from __future__ import annotations

import os
from dataclasses import dataclass, field

import numpy as np


@dataclass
class Problem:
    """A tree in parent-array form plus a CSR sample x tip count table.

    parent[v]      int32 [n_nodes]  parent node id, -1 for the single root
    branch_len[v]  float64 [n_nodes] length of the edge v -> parent[v] (root entry ignored)
    postorder      int32 [n_nodes]  permutation, children before parent, root last
    indptr         int64 [n_samples+1]
    indices        int32 [nnz]      tip NODE ids, strictly increasing within a row
    counts         int32 [nnz]      >= 0
    """
    parent: np.ndarray
    branch_len: np.ndarray
    postorder: np.ndarray
    indptr: np.ndarray
    indices: np.ndarray
    counts: np.ndarray
    name: str = "custom"
    meta: dict = field(default_factory=dict)

    @property
    def n_nodes(self) -> int:
        return int(self.parent.shape[0])

    @property
    def n_samples(self) -> int:
        return int(self.indptr.shape[0] - 1)

    @property
    def nnz(self) -> int:
        return int(self.indices.shape[0])

    @property
    def n_pairs(self) -> int:
        n = self.n_samples
        return n * (n - 1) // 2


# ----------------------------------------------------------------------------------------------
# trees
# ----------------------------------------------------------------------------------------------
def yule_parent(n_tips: int, rng: np.random.Generator) -> np.ndarray:
    """Yule topology: start with node 0 as the only tip; n_tips-1 times pick a uniformly random
    current tip and give it two new children (ids next, next+1).  2*n_tips-1 nodes, parent id <
    child id.  Uniform picks are floor(U_k * k) with U drawn in one call (fixed RNG order)."""
    n_nodes = 2 * n_tips - 1
    parent = np.full(n_nodes, -1, dtype=np.int32)
    if n_tips == 1:
        return parent
    u = rng.random(n_tips - 1)
    tips = [0] * n_tips
    nxt = 1
    picks = np.minimum((u * np.arange(1, n_tips)).astype(np.int64), np.arange(0, n_tips - 1))
    picks = picks.tolist()
    par = parent.tolist()
    for k in range(1, n_tips):
        j = picks[k - 1]
        p = tips[j]
        par[nxt] = p
        par[nxt + 1] = p
        tips[j] = nxt
        tips[k] = nxt + 1
        nxt += 2
    return np.asarray(par, dtype=np.int32)


def children_csr(parent: np.ndarray):
    """children lists in id order: (offsets int64[n+1], child ids int32)."""
    n = parent.shape[0]
    nonroot = np.nonzero(parent >= 0)[0]
    order = nonroot[np.argsort(parent[nonroot], kind="stable")]
    cnt = np.bincount(parent[nonroot], minlength=n)
    off = np.zeros(n + 1, dtype=np.int64)
    np.cumsum(cnt, out=off[1:])
    return off, order.astype(np.int32)


def dfs_postorder(parent: np.ndarray) -> np.ndarray:
    """True DFS post-order (children visited in id order), root last."""
    n = parent.shape[0]
    off, ch = children_csr(parent)
    off_l = off.tolist()
    ch_l = ch.tolist()
    root = int(np.nonzero(parent < 0)[0][0])
    out = []
    stack = [root]
    nxt = [off_l[v] for v in range(n)]
    while stack:
        v = stack[-1]
        i = nxt[v]
        if i < off_l[v + 1]:
            nxt[v] = i + 1
            stack.append(ch_l[i])
        else:
            out.append(v)
            stack.pop()
    return np.asarray(out, dtype=np.int32)


def tip_ids(parent: np.ndarray) -> np.ndarray:
    n = parent.shape[0]
    has_child = np.zeros(n, dtype=bool)
    has_child[parent[parent >= 0]] = True
    return np.nonzero(~has_child)[0].astype(np.int32)


# ----------------------------------------------------------------------------------------------
# tables
# ----------------------------------------------------------------------------------------------
def _distinct_ranks(k: int, cdf: np.ndarray, rng: np.random.Generator) -> np.ndarray:
    """Draw ranks iid by inverse CDF until k distinct ones have been seen (first-seen order)."""
    n = cdf.shape[0]
    k = min(k, n)
    got = np.empty(0, dtype=np.int64)
    while got.shape[0] < k:
        need = k - got.shape[0]
        m = 2 * need + 32
        r = np.searchsorted(cdf, rng.random(m), side="right")
        np.minimum(r, n - 1, out=r)
        allr = np.concatenate([got, r])
        _, first = np.unique(allr, return_index=True)
        first.sort()
        got = allr[first][:k]
    return got


_TAB = {}          # state inherited by forked workers (read-only)


def _sample_rows(lo: int, hi: int):
    """Rows lo..hi-1.  Sample s uses its own generator default_rng(SeedSequence(seed, spawn_key=(1, s))),
    so the table does not depend on how the samples are split over worker processes."""
    t = _TAB
    idx, cnt = [], []
    for s in range(lo, hi):
        rng = np.random.default_rng(np.random.SeedSequence(t["seed"], spawn_key=(1, s)))
        ranks = _distinct_ranks(int(t["ks"][s]), t["cdf"], rng)
        cols = np.sort(t["tips"][t["perm"][ranks]])
        idx.append(cols)
        cnt.append(t["count_draw"](cols.shape[0], rng))
    return lo, np.concatenate(idx).astype(np.int32), np.concatenate(cnt).astype(np.int32)


def make_table(tips: np.ndarray, n_samples: int, zipf_a: float, k_draw, count_draw,
               rng: np.random.Generator, seed: int = 0, workers: int | None = None):
    n_tips = tips.shape[0]
    perm = rng.permutation(n_tips)                 # rank r -> tips[perm[r]]
    w = np.arange(1, n_tips + 1, dtype=np.float64) ** (-zipf_a)
    cdf = np.cumsum(w)
    cdf /= cdf[-1]
    ks = k_draw(n_samples, rng)
    ks = np.clip(ks, 1, n_tips).astype(np.int64)
    indptr = np.zeros(n_samples + 1, dtype=np.int64)
    np.cumsum(ks, out=indptr[1:])
    _TAB.clear()
    _TAB.update(seed=seed, ks=ks, cdf=cdf, tips=tips, perm=perm, count_draw=count_draw)
    if workers is None:
        workers = min(os.cpu_count() or 1, 32) if int(indptr[-1]) > 2_000_000 else 1
    chunk = 256
    jobs = [(lo, min(lo + chunk, n_samples)) for lo in range(0, n_samples, chunk)]
    if workers > 1:
        import multiprocessing as mp
        with mp.get_context("fork").Pool(workers) as pool:
            parts = pool.starmap(_sample_rows, jobs)
    else:
        parts = [_sample_rows(lo, hi) for lo, hi in jobs]
    parts.sort(key=lambda p: p[0])
    indices = np.concatenate([p[1] for p in parts])
    counts = np.concatenate([p[2] for p in parts])
    _TAB.clear()
    return indptr, indices, counts


def _k_poisson40(n, rng):
    return rng.poisson(40.0, size=n) + 1


def _k_lognormal(mu, sigma):
    def f(n, rng):
        return np.maximum(1, np.rint(rng.lognormal(mu, sigma, size=n))).astype(np.int64)
    return f


def _c_geometric(n, rng):          # 1 + failures-before-success: numpy's support is 1,2,...
    return rng.geometric(0.2, size=n).astype(np.int32)


def _c_lognormal(n, rng):
    return np.minimum(np.maximum(1, np.rint(rng.lognormal(2.0, 1.5, size=n))), 2**30).astype(np.int32)


CONFIGS = {
    # name: (n_tips, n_samples, mean branch length, zipf a, k draw, count draw)   BASELINE.json:7-11
    "tiny":   (256,     64,     0.1,  1.1,  _k_poisson40,                      _c_geometric),
    "small":  (20_000,  2_048,  0.1,  1.1,  _k_lognormal(np.log(200.0), 0.5),  _c_lognormal),
    "medium": (100_000, 10_000, 0.05, 1.05, _k_lognormal(np.log(500.0), 0.6),  _c_lognormal),
    "emp":    (300_000, 25_000, 0.05, 1.05, _k_lognormal(np.log(800.0), 0.7),  _c_lognormal),
    "large":  (500_000, 50_000, 0.05, 1.05, _k_lognormal(np.log(800.0), 0.7),  _c_lognormal),
}


def make_problem(n_tips: int, n_samples: int, mean_len: float, zipf_a: float, k_draw, count_draw,
                 seed: int = 0, name: str = "custom") -> Problem:
    """RNG = numpy default_rng(seed), consumed in this order: Yule picks, branch lengths,
    popularity permutation, per-sample feature counts k; then sample s draws (ranks, counts)
    from its own default_rng(SeedSequence(seed, spawn_key=(1, s)))."""
    rng = np.random.default_rng(seed)
    parent = yule_parent(n_tips, rng)
    n_nodes = parent.shape[0]
    branch_len = rng.exponential(mean_len, size=n_nodes)
    branch_len[0] = 0.0
    post = dfs_postorder(parent)
    tips = tip_ids(parent)
    indptr, indices, counts = make_table(tips, n_samples, zipf_a, k_draw, count_draw, rng, seed=seed)
    return Problem(parent, branch_len.astype(np.float64), post, indptr, indices, counts, name=name,
                   meta=dict(n_tips=n_tips, seed=seed, mean_len=mean_len, zipf_a=zipf_a))


def make_config(name: str, seed: int = 0, n_samples: int | None = None) -> Problem:
    """One of BASELINE.json's five configs ('tiny','small','medium','emp','large').
    n_samples may be lowered for a scaled-down run of the same tree/distributions."""
    n_tips, n_s, mean_len, a, kd, cd = CONFIGS[name]
    if n_samples is not None:
        n_s = n_samples
    return make_problem(n_tips, n_s, mean_len, a, kd, cd, seed=seed, name=name)


# ----------------------------------------------------------------------------------------------
# small structured inputs for tests (still no UniFrac arithmetic)
# ----------------------------------------------------------------------------------------------
def problem_from_parent(parent, branch_len, rows, name="custom") -> Problem:
    """rows: list of {tip node id: count} dicts."""
    parent = np.asarray(parent, dtype=np.int32)
    post = dfs_postorder(parent)
    indptr = [0]
    idx, cnt = [], []
    for r in rows:
        for t in sorted(r):
            idx.append(t)
            cnt.append(r[t])
        indptr.append(len(idx))
    return Problem(parent, np.asarray(branch_len, dtype=np.float64), post,
                   np.asarray(indptr, dtype=np.int64), np.asarray(idx, dtype=np.int32),
                   np.asarray(cnt, dtype=np.int32), name=name)


def star_tree(n_tips: int, lengths) -> tuple[np.ndarray, np.ndarray]:
    """All tips are children of the root (node n_tips)."""
    parent = np.full(n_tips + 1, n_tips, dtype=np.int32)
    parent[n_tips] = -1
    bl = np.zeros(n_tips + 1, dtype=np.float64)
    bl[:n_tips] = lengths
    return parent, bl


def random_tree(n_nodes: int, rng: np.random.Generator, p_unary: float = 0.15,
                p_zero_len: float = 0.1) -> tuple[np.ndarray, np.ndarray]:
    """Random rooted tree with arbitrary arity (multifurcations, unary internal nodes, some
    zero-length branches).  Node ids are shuffled so that parent id is unrelated to child id."""
    parent = np.full(n_nodes, -1, dtype=np.int64)
    for v in range(1, n_nodes):
        if rng.random() < p_unary and v > 1:
            parent[v] = v - 1                   # chains -> unary nodes
        else:
            parent[v] = rng.integers(0, v)
    relabel = rng.permutation(n_nodes)
    new_parent = np.full(n_nodes, -1, dtype=np.int32)
    for v in range(n_nodes):
        if parent[v] >= 0:
            new_parent[relabel[v]] = relabel[parent[v]]
    bl = rng.exponential(1.0, size=n_nodes)
    bl[rng.random(n_nodes) < p_zero_len] = 0.0
    return new_parent, bl


def random_table(tips: np.ndarray, n_samples: int, rng: np.random.Generator, density: float = 0.3,
                 max_count: int = 20):
    rows = []
    for _ in range(n_samples):
        m = rng.random(tips.shape[0]) < density
        if not m.any():
            m[rng.integers(0, tips.shape[0])] = True
        rows.append({int(t): int(rng.integers(1, max_count + 1)) for t in tips[m]})
    return rows


def sample_pairs(n_samples: int, n_pairs: int, seed: int = 0) -> np.ndarray:
    """Seeded i<j pairs (with replacement across draws), shape [n_pairs, 2], int32."""
    rng = np.random.default_rng(seed + 7919)
    i = rng.integers(0, n_samples, size=n_pairs)
    j = rng.integers(0, n_samples - 1, size=n_pairs)
    j = np.where(j >= i, j + 1, j)
    lo = np.minimum(i, j)
    hi = np.maximum(i, j)
    return np.stack([lo, hi], axis=1).astype(np.int32)


def condensed_index(n: int, i, j):
    """scipy squareform order: idx(i,j) = i*(2n-i-1)/2 + (j-i-1), i<j."""
    i = np.asarray(i, dtype=np.int64)
    j = np.asarray(j, dtype=np.int64)
    return i * (2 * n - i - 1) // 2 + (j - i - 1)


def rows_of(p: Problem) -> list:
    """The table of `p` as a list of {tip node id: count} dicts (one per sample)."""
    return [{int(t): int(c) for t, c in zip(p.indices[p.indptr[s]:p.indptr[s + 1]], p.counts[p.indptr[s]:p.indptr[s + 1]])}
            for s in range(p.n_samples)]


def with_rows(p: Problem, rows, branch_len=None) -> Problem:
    """Same tree as `p` (optionally other branch lengths) with another table."""
    q = problem_from_parent(p.parent, p.branch_len if branch_len is None else branch_len, rows, name=p.name)
    q.postorder = p.postorder
    return q


def plant_near_duplicates(p: Problem, n_each: int, seed: int = 0):
    """Overwrite 3 * n_each samples of `p` with (a) exact copies, (b) integer multiples and (c) copies with one count
    changed by 1 and one feature dropped, of other samples, at positions spread so that sources and copies sit in different 128-sample tiles and
    on tile boundaries.  Returns (problem, pairs [3 * n_each, 2] int32 with i < j, kinds) -- kinds 0 / 1 / 2."""
    rng = np.random.default_rng(seed + 4242)
    rows = rows_of(p)
    n = p.n_samples
    boundary = [s for t in range(128, n, 128) for s in (t - 1, t)]
    pool = boundary + [int(x) for x in rng.permutation(n) if int(x) not in set(boundary)]
    dst = pool[:3 * n_each]
    taken = set(dst)
    src = [int(x) for x in rng.permutation(n) if int(x) not in taken][:3 * n_each]
    pairs, kinds = [], []
    for k, (a, b) in enumerate(zip(src, dst)):
        kind = k % 3
        r = dict(rows[a])
        if kind == 1:
            m = int(rng.integers(2, 9))
            r = {t: c * m for t, c in r.items()}
        elif kind == 2:
            keys = sorted(r)
            r[keys[int(rng.integers(0, len(keys)))]] += 1
            if len(keys) > 2:                           # and one feature dropped, so that presence changes as well
                del r[keys[int(rng.integers(0, len(keys)))]]
        rows[b] = r
        pairs.append((min(a, b), max(a, b)))
        kinds.append(kind)
    return with_rows(p, rows), np.asarray(pairs, dtype=np.int32), np.asarray(kinds)
