"""Second, independent formulation of UniFrac used ONLY to pin the oracle (tests).

Not the oracle and not the CUDA path: explicit ancestor-indicator matrix A[v, t] (1 if tip t is
below branch v), embeddings by one matrix product, then the ratios -- with the weighted
denominator taken from the closed form I1 (root-to-tip distances), so that a dropped term or a
wrong index in the oracle's tree walk cannot cancel out.  Exact rational variant included."""
from fractions import Fraction

import numpy as np


def ancestor_matrix(parent):
    parent = np.asarray(parent)
    n = parent.shape[0]
    has_child = np.zeros(n, bool)
    has_child[parent[parent >= 0]] = True
    tips = np.nonzero(~has_child)[0]
    A = np.zeros((n, tips.shape[0]), dtype=np.int64)
    for k, t in enumerate(tips):
        v = int(t)
        while parent[v] >= 0:
            A[v, k] = 1
            v = int(parent[v])
    return A, tips


def dense_counts(problem, tips):
    col = {int(t): k for k, t in enumerate(tips)}
    X = np.zeros((problem.n_samples, tips.shape[0]), dtype=np.int64)
    for s in range(problem.n_samples):
        for k in range(problem.indptr[s], problem.indptr[s + 1]):
            X[s, col[int(problem.indices[k])]] += int(problem.counts[k])
    return X


def unifrac_matrix_np(problem, variant):
    """Full N x N float64 matrix via E = X A^T (0 = unweighted, 1 = weighted-normalized)."""
    A, tips = ancestor_matrix(problem.parent)
    X = dense_counts(problem, tips)
    ell = np.where(problem.parent >= 0, problem.branch_len, 0.0)
    C = X @ A.T                                         # [N, n_nodes] subtree counts
    n = problem.n_samples
    D = np.zeros((n, n))
    if variant == 0:
        P = (C > 0)
        for a in range(n):
            x = np.logical_xor(P[a][None, :], P)
            o = np.logical_or(P[a][None, :], P)
            num = (x * ell).sum(1)
            den = (o * ell).sum(1)
            D[a] = np.where(den > 0, num / np.where(den > 0, den, 1), 0.0)
    else:
        T = X.sum(1, keepdims=True).astype(np.float64)
        U = C / T
        # I1: root-to-tip distances
        dist = (A * ell[:, None]).sum(0)                # D_t
        R = ((X / T) * dist[None, :]).sum(1)
        for a in range(n):
            num = (np.abs(U[a][None, :] - U) * ell).sum(1)
            den = R[a] + R
            D[a] = np.where(den > 0, num / np.where(den > 0, den, 1), 0.0)
    return D


def unifrac_pair_exact(problem, variant, a, b):
    """Exact rational d(a,b) (branch lengths must be integers or Fractions)."""
    A, tips = ancestor_matrix(problem.parent)
    X = dense_counts(problem, tips)
    C = X @ A.T
    Ta, Tb = int(X[a].sum()), int(X[b].sum())
    num = Fraction(0)
    den = Fraction(0)
    for v in range(problem.n_nodes):
        if problem.parent[v] < 0:
            continue
        l = Fraction(problem.branch_len[v]).limit_denominator(10**9)
        if variant == 0:
            xa, xb = C[a, v] > 0, C[b, v] > 0
            num += l * int(xa != xb)
            den += l * int(xa or xb)
        else:
            u, w = Fraction(int(C[a, v]), Ta), Fraction(int(C[b, v]), Tb)
            num += l * abs(u - w)
            den += l * (u + w)
    return num / den if den != 0 else Fraction(0)
