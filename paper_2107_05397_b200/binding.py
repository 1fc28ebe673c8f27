"""Thin ctypes binding of include/unifrac_b200.h -- same names, argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch is used here only for device
memory (the workspace allocator handed to the library is backed by ``torch.empty``) and for the
stream.  There is no CPU fallback: if the library cannot be loaded, ``load()`` raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

from . import build as _build

UNWEIGHTED, WEIGHTED_NORMALIZED = 0, 1
FP32, FP64 = 0, 1
FLAG_LITERAL, FLAG_TENSOR_GRAM, FLAG_SKIP_VALIDATION, FLAG_ABSDIFF = 1, 2, 4, 8
FLAG_NO_TAIL, FLAG_ALL_TAIL, FLAG_NO_TENSOR, FLAG_NO_MID, FLAG_SPARSE_STRIPE, FLAG_RICHNESS_ZONES = 16, 32, 64, 128, 256, 512

ABI_VERSION = 8          # unifrac_abi_version() of the header this binding was written against
OK = 0
ERR_INVALID_ARG, ERR_INVALID_TREE, ERR_INVALID_TABLE, ERR_EMPTY_SAMPLE = -1, -2, -3, -4
ERR_WORKSPACE, ERR_CUDA, ERR_UNSUPPORTED = -5, -6, -7

EXPORTS = ("unifrac_dm", "unifrac_dm_shard", "unifrac_shard_of_pair", "unifrac_dm_host", "unifrac_dm_host_multi", "unifrac_release_host_pool", "unifrac_mantel_pearson", "unifrac_mantel_pearson_noalloc", "unifrac_mantel_spearman", "unifrac_pcoa", "unifrac_measure_rates", "unifrac_last_stats", "unifrac_status_string",
           "unifrac_last_cuda_error", "unifrac_abi_version")


class CSR(C.Structure):
    _fields_ = [("indptr", C.c_void_p), ("indices", C.c_void_p), ("counts", C.c_void_p)]


class Stats(C.Structure):
    _fields_ = [("branches_embedded", C.c_uint64), ("updates_dense", C.c_uint64), ("updates_union", C.c_uint64),
                ("updates_inter", C.c_uint64), ("updates_executed", C.c_uint64), ("updates_executed_head", C.c_uint64),
                ("head_rows", C.c_uint64), ("tail_rows", C.c_uint64), ("tail_updates", C.c_uint64),
                ("tail_entries", C.c_uint64), ("mid_rows", C.c_uint64), ("mid_updates", C.c_uint64),
                ("rows_staged", C.c_uint64),
                ("embed_rows", C.c_uint64), ("workspace_bytes", C.c_uint64), ("skip_updates_executed", C.c_uint64),
                ("skip_row_pair_visits", C.c_uint64), ("mid_atomics", C.c_uint64), ("n_tile_pairs", C.c_uint32),
                ("n_levels", C.c_uint32), ("stripe_launches", C.c_uint32), ("tail_launches", C.c_uint32),
                ("kernel_launches", C.c_uint32), ("mid_launches", C.c_uint32), ("mid_F", C.c_uint32), ("gram", C.c_uint32), ("gram_k", C.c_uint32), ("gram_q", C.c_uint32), ("dense", C.c_uint32), ("skip", C.c_uint32), ("skip_rows", C.c_uint32), ("list_rows", C.c_uint32), ("guard_pairs", C.c_uint32), ("guard_capacity", C.c_uint32), ("mid_groups", C.c_uint32), ("mid_group_rows", C.c_uint32), ("quant_fallback", C.c_uint32), ("guard_theta", C.c_float), ("quant_err_ratio", C.c_float),
                ("ms_plan", C.c_float), ("ms_embed", C.c_float), ("ms_tail", C.c_float), ("ms_mid", C.c_float), ("ms_stripe", C.c_float),
                ("ms_total", C.c_float)]


class Rates(C.Structure):
    _fields_ = [("smem_atomic_conflict_free_per_s", C.c_double), ("smem_atomic_random_per_s", C.c_double),
                ("l2_red_random_per_s", C.c_double), ("fmnmx_per_s", C.c_double), ("fadd_per_s", C.c_double),
                ("fmnmx_fadd_per_s", C.c_double), ("fadd2_per_s", C.c_double), ("fmnmx2_fadd2_updates_per_s", C.c_double),
                ("dense16_mix_updates_per_s", C.c_double), ("sm_count", C.c_int32), ("sm_clock_khz", C.c_int32)]


ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)


class UnifracError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"unifrac_b200 status {status}: {msg}")
        self.status = status


_lib = None


def load(build_if_missing: bool = True) -> C.CDLL:
    """dlopen libunifrac_b200.so (built in-tree by build.py).  Raises if it cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if not os.path.exists(path) or (build_if_missing and _build.needs_build()):
        if not build_if_missing:
            raise FileNotFoundError(path)
        _build.build()              # a failed rebuild raises: a stale library is never loaded in its place
    lib = C.CDLL(path)
    lib.unifrac_abi_version.restype = C.c_int
    if lib.unifrac_abi_version() != ABI_VERSION:
        raise RuntimeError(f"{path}: ABI version {lib.unifrac_abi_version()} != {ABI_VERSION} (stale build; the Stats / "
                           f"Rates layouts of this binding would not match)")
    lib.unifrac_dm.restype = C.c_int
    lib.unifrac_dm.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, CSR, C.c_int32, C.c_int, C.c_int,
                               C.c_void_p, ALLOC_FN, C.c_void_p, C.c_uint32, C.c_void_p]
    lib.unifrac_dm_shard.restype = C.c_int
    lib.unifrac_dm_shard.argtypes = lib.unifrac_dm.argtypes + [C.c_int32, C.c_int32]
    lib.unifrac_shard_of_pair.restype = C.c_int32
    lib.unifrac_shard_of_pair.argtypes = [C.c_int32, C.c_int32, C.c_int32]
    lib.unifrac_dm_host.restype = C.c_int
    lib.unifrac_dm_host.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, CSR, C.c_int32, C.c_int, C.c_int,
                                    C.c_void_p, C.c_uint32]
    lib.unifrac_dm_host_multi.restype = C.c_int
    lib.unifrac_dm_host_multi.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, CSR, C.c_int32, C.c_int32,
                                          C.POINTER(C.c_int32), C.c_int, C.POINTER(C.c_void_p), C.c_uint32]
    lib.unifrac_release_host_pool.restype = C.c_int
    lib.unifrac_mantel_pearson.restype = C.c_int
    lib.unifrac_mantel_pearson.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_int32, C.c_void_p,
                                           ALLOC_FN, C.c_void_p, C.c_void_p]
    lib.unifrac_mantel_spearman.restype = C.c_int
    lib.unifrac_mantel_spearman.argtypes = lib.unifrac_mantel_pearson.argtypes
    lib.unifrac_mantel_pearson_noalloc.argtypes = [C.c_int32, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]
    lib.unifrac_mantel_pearson_noalloc.restype = C.c_int
    lib.unifrac_pcoa.restype = C.c_int
    lib.unifrac_pcoa.argtypes = [C.c_int32, C.c_void_p, C.c_int, C.c_int32, C.c_int32, C.c_double, C.c_void_p,
                                 C.POINTER(C.c_int32), ALLOC_FN, C.c_void_p, C.c_void_p]
    lib.unifrac_measure_rates.restype = C.c_int
    lib.unifrac_measure_rates.argtypes = [C.POINTER(Rates), C.c_void_p]
    lib.unifrac_last_stats.restype = C.c_int
    lib.unifrac_last_stats.argtypes = [C.POINTER(Stats)]
    lib.unifrac_status_string.restype = C.c_char_p
    lib.unifrac_status_string.argtypes = [C.c_int]
    lib.unifrac_last_cuda_error.restype = C.c_char_p
    lib.unifrac_abi_version.restype = C.c_int
    _lib = lib
    return lib


def _check(lib, rc: int):
    if rc != 0:
        msg = lib.unifrac_status_string(rc).decode()
        if rc == ERR_CUDA:
            msg += ": " + lib.unifrac_last_cuda_error().decode()
        raise UnifracError(rc, msg)


def unifrac_dm(tree_parent, branch_len, postorder, indptr, indices, counts, n_samples: int, variant: int,
               precision: int, out=None, flags: int = 0, stream=None, shard=None):
    """Device entry point (`shard=(index, count)` calls unifrac_dm_shard: this shard's blocks, 0 elsewhere).  All inputs are CUDA torch tensors (int32 / float64 / int32 / int64 / int32 /
    int32); returns the condensed matrix as a CUDA tensor (float32 or float64).  Asynchronous on
    `stream` (default: torch's current stream) after the plan/embedding steps."""
    import torch
    lib = load()
    dev = tree_parent.device
    assert dev.type == "cuda", "unifrac_dm takes device tensors; use unifrac_dm_host for host arrays"
    for t, dt in ((tree_parent, torch.int32), (branch_len, torch.float64), (postorder, torch.int32),
                  (indptr, torch.int64), (indices, torch.int32), (counts, torch.int32)):
        assert t.dtype == dt and t.is_contiguous() and t.device == dev
    n = int(n_samples)
    odt = torch.float32 if precision == FP32 else torch.float64
    assert indptr.numel() == n + 1, "indptr must have n_samples + 1 entries"
    assert branch_len.numel() == tree_parent.numel() == postorder.numel() and indices.numel() == counts.numel()
    if out is None:
        out = torch.empty(n * (n - 1) // 2, dtype=odt, device=dev)
    assert out.dtype == odt and out.device == dev and out.is_contiguous() and out.numel() == n * (n - 1) // 2, \
        "out must be a contiguous condensed vector of n(n-1)/2 elements of the call's precision on the inputs' device"
    held = []

    def _alloc(nbytes, _user):
        try:
            t = torch.empty(int(nbytes), dtype=torch.uint8, device=dev)
        except Exception:
            return None
        held.append(t)
        return t.data_ptr()

    cb = ALLOC_FN(_alloc)
    with torch.cuda.device(dev):
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        with torch.cuda.stream(s):
            common = (int(tree_parent.shape[0]), tree_parent.data_ptr(), branch_len.data_ptr(),
                      postorder.data_ptr(), CSR(indptr.data_ptr(), indices.data_ptr(), counts.data_ptr()),
                      n, int(variant), int(precision), out.data_ptr(), cb, None, int(flags), C.c_void_p(s.cuda_stream))
            if shard is None:
                rc = lib.unifrac_dm(*common)
            else:
                rc = lib.unifrac_dm_shard(*common, int(shard[0]), int(shard[1]))
    # workspace tensors were allocated under `s`; dropping them here is stream-ordered safe
    del held
    _check(lib, rc)
    return out


def unifrac_dm_host(tree_parent, branch_len, postorder, indptr, indices, counts, n_samples: int, variant: int,
                    precision: int, out: Optional[np.ndarray] = None, flags: int = 0) -> np.ndarray:
    """Host entry point: numpy arrays in, numpy condensed matrix out (synchronous; the library does
    the host<->device copies itself)."""
    lib = load()
    a = [np.ascontiguousarray(tree_parent, np.int32), np.ascontiguousarray(branch_len, np.float64),
         np.ascontiguousarray(postorder, np.int32), np.ascontiguousarray(indptr, np.int64),
         np.ascontiguousarray(indices, np.int32), np.ascontiguousarray(counts, np.int32)]
    n = int(n_samples)
    if out is None:
        out = np.empty(n * (n - 1) // 2, dtype=np.float32 if precision == FP32 else np.float64)
    rc = lib.unifrac_dm_host(int(a[0].shape[0]), a[0].ctypes.data, a[1].ctypes.data, a[2].ctypes.data,
                             CSR(a[3].ctypes.data, a[4].ctypes.data, a[5].ctypes.data), n, int(variant),
                             int(precision), out.ctypes.data, int(flags))
    _check(lib, rc)
    return out


def unifrac_dm_host_multi(tree_parent, branch_len, postorder, indptr, indices, counts, n_samples: int, variants,
                          precision: int, outs=None, flags: int = 0):
    """Host entry point for several variants of one table (inputs uploaded once, result copies overlap the next
    variant's compute).  Returns the list of condensed numpy arrays."""
    lib = load()
    a = [np.ascontiguousarray(tree_parent, np.int32), np.ascontiguousarray(branch_len, np.float64),
         np.ascontiguousarray(postorder, np.int32), np.ascontiguousarray(indptr, np.int64),
         np.ascontiguousarray(indices, np.int32), np.ascontiguousarray(counts, np.int32)]
    n, k = int(n_samples), len(variants)
    if outs is None:
        outs = [np.empty(n * (n - 1) // 2, dtype=np.float32 if precision == FP32 else np.float64) for _ in range(k)]
    vs = (C.c_int32 * k)(*[int(v) for v in variants])
    ptrs = (C.c_void_p * k)(*[o.ctypes.data for o in outs])
    rc = lib.unifrac_dm_host_multi(int(a[0].shape[0]), a[0].ctypes.data, a[1].ctypes.data, a[2].ctypes.data,
                                   CSR(a[3].ctypes.data, a[4].ctypes.data, a[5].ctypes.data), n, k, vs, int(precision), ptrs, int(flags))
    _check(lib, rc)
    return outs


def unifrac_release_host_pool() -> None:
    lib = load()
    _check(lib, lib.unifrac_release_host_pool())


def unifrac_last_stats() -> dict:
    lib = load()
    s = Stats()
    _check(lib, lib.unifrac_last_stats(C.byref(s)))
    return {k: getattr(s, k) for k, _ in Stats._fields_}


def unifrac_mantel_spearman(x_condensed, y_condensed, n_samples: int, perms, stream=None):
    """Mantel test with Spearman's rank correlation; same arguments and result layout as unifrac_mantel_pearson."""
    return unifrac_mantel_pearson(x_condensed, y_condensed, n_samples, perms, stream=stream, _entry="unifrac_mantel_spearman")


def unifrac_mantel_pearson(x_condensed, y_condensed, n_samples: int, perms, stream=None, _entry="unifrac_mantel_pearson"):
    """Mantel test (Pearson) on two condensed CUDA tensors (both float32 or both float64); perms: CUDA int32 [K, n].
    Returns a CUDA float64 tensor [4 + K]: r, p two-sided, p greater, p less, r_1 .. r_K.  Asynchronous on the stream."""
    import torch
    lib = load()
    dev = x_condensed.device
    n = int(n_samples)
    assert dev.type == "cuda" and y_condensed.device == dev and perms.device == dev
    assert x_condensed.dtype == y_condensed.dtype and x_condensed.dtype in (torch.float32, torch.float64)
    assert x_condensed.is_contiguous() and y_condensed.is_contiguous() and perms.is_contiguous() and perms.dtype == torch.int32
    assert x_condensed.numel() == n * (n - 1) // 2 == y_condensed.numel()
    K = int(perms.numel() // n) if perms.numel() else 0
    out = torch.empty(4 + K, dtype=torch.float64, device=dev)
    held = []

    def _alloc(nbytes, _user):
        try:
            t = torch.empty(int(nbytes), dtype=torch.uint8, device=dev)
        except Exception:
            return None
        held.append(t)
        return t.data_ptr()

    cb = ALLOC_FN(_alloc)
    with torch.cuda.device(dev):
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        with torch.cuda.stream(s):
            rc = getattr(lib, _entry)(n, x_condensed.data_ptr(), y_condensed.data_ptr(),
                                            FP32 if x_condensed.dtype == torch.float32 else FP64,
                                            perms.data_ptr() if K else None, K, out.data_ptr(), cb, None,
                                            C.c_void_p(s.cuda_stream))
    del held
    _check(lib, rc)
    return out


NOALLOC_MAX_SAMPLES = 1024       # UNIFRAC_NOALLOC_MAX_SAMPLES / _PERMS of the header
NOALLOC_MAX_PERMS = 999


def unifrac_mantel_pearson_noalloc(x_condensed, y_condensed, n_samples: int, perms, out, stream=None):
    """unifrac_mantel_pearson through the library's static device workspace: no allocation anywhere in the call, so `out`
    (CUDA float64 [4 + K]) is the caller's too.  n_samples <= 1024, K <= 999 (UnifracError otherwise).  Calls that overlap
    on the GPU race on the shared workspace.  Returns `out`.  Asynchronous on the stream."""
    import torch
    lib = load()
    dev = x_condensed.device
    n = int(n_samples)
    assert dev.type == "cuda" and y_condensed.device == dev and perms.device == dev and out.device == dev
    assert x_condensed.dtype == y_condensed.dtype and x_condensed.dtype in (torch.float32, torch.float64)
    assert x_condensed.is_contiguous() and y_condensed.is_contiguous() and perms.is_contiguous() and perms.dtype == torch.int32
    assert x_condensed.numel() == n * (n - 1) // 2 == y_condensed.numel()
    K = int(perms.numel() // n) if perms.numel() else 0
    assert out.dtype == torch.float64 and out.is_contiguous() and out.numel() == 4 + K
    with torch.cuda.device(dev):
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        rc = lib.unifrac_mantel_pearson_noalloc(n, C.c_void_p(x_condensed.data_ptr()), C.c_void_p(y_condensed.data_ptr()),
                                                FP32 if x_condensed.dtype == torch.float32 else FP64,
                                                C.c_void_p(perms.data_ptr()) if K else None, K, C.c_void_p(out.data_ptr()),
                                                C.c_void_p(s.cuda_stream))
    if rc == ERR_UNSUPPORTED:
        raise UnifracError(rc, lib.unifrac_status_string(rc).decode() + ": " + lib.unifrac_last_cuda_error().decode())
    _check(lib, rc)
    return out


def unifrac_pcoa(d_condensed, n_samples: int, k: int, max_iter: int = 200, tol: float = 1e-7, stream=None):
    """PCoA of a condensed CUDA distance vector (float32 / float64).  Returns (eigenvalues[k], proportion[k], coords[n, k])
    as CUDA float64 tensors and the number of B Q products used."""
    import torch
    lib = load()
    dev = d_condensed.device
    n, k = int(n_samples), int(k)
    assert dev.type == "cuda" and d_condensed.is_contiguous() and d_condensed.dtype in (torch.float32, torch.float64)
    assert d_condensed.numel() == n * (n - 1) // 2
    out = torch.empty(2 * k + n * k, dtype=torch.float64, device=dev)
    held = []

    def _alloc(nbytes, _user):
        try:
            t = torch.empty(int(nbytes), dtype=torch.uint8, device=dev)
        except Exception:
            return None
        held.append(t)
        return t.data_ptr()

    cb = ALLOC_FN(_alloc)
    its = C.c_int32(0)
    with torch.cuda.device(dev):
        s = stream if stream is not None else torch.cuda.current_stream(dev)
        with torch.cuda.stream(s):
            rc = lib.unifrac_pcoa(n, d_condensed.data_ptr(), FP32 if d_condensed.dtype == torch.float32 else FP64, k,
                                  int(max_iter), float(tol), out.data_ptr(), C.byref(its), cb, None, C.c_void_p(s.cuda_stream))
    del held
    _check(lib, rc)
    return out[:k], out[k:2 * k], out[2 * k:].view(n, k), int(its.value)


def unifrac_measure_rates(stream=None) -> dict:
    """Device-rate probes (shared-memory atomics, L2 REDs) on torch's current stream."""
    import torch
    lib = load()
    r = Rates()
    s = stream if stream is not None else torch.cuda.current_stream()
    _check(lib, lib.unifrac_measure_rates(C.byref(r), C.c_void_p(s.cuda_stream)))
    return {k: getattr(r, k) for k, _ in Rates._fields_}


def unifrac_shard_of_pair(i: int, j: int, shard_count: int) -> int:
    return int(load().unifrac_shard_of_pair(int(i), int(j), int(shard_count)))


def unifrac_status_string(status: int) -> str:
    return load().unifrac_status_string(int(status)).decode()


def unifrac_abi_version() -> int:
    return int(load().unifrac_abi_version())


def to_device(problem, device="cuda:0"):
    """Marshal a synth.Problem (numpy) into the six device tensors unifrac_dm takes."""
    import torch
    f = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(device)
    return (f(problem.parent.astype(np.int32)), f(problem.branch_len.astype(np.float64)),
            f(problem.postorder.astype(np.int32)), f(problem.indptr.astype(np.int64)),
            f(problem.indices.astype(np.int32)), f(problem.counts.astype(np.int32)))
