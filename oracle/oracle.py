"""ctypes wrapper + build step for oracle/unifrac_oracle.c -- TEST INFRASTRUCTURE ONLY.

The arithmetic lives in the C file (plain definition of UniFrac, PAPER.md:21-23 /
BASELINE.json:5); this module only builds it with gcc and marshals numpy arrays.
It imports nothing from the CUDA package."""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "unifrac_oracle.c")
_LIB = os.path.join(_HERE, "libunifrac_oracle.so")

UNWEIGHTED = 0
WEIGHTED_NORMALIZED = 1

OK, ERR_ARG, ERR_TREE, ERR_TABLE, ERR_EMPTY_SAMPLE, ERR_NOMEM = 0, -1, -2, -3, -4, -5


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        i32p, i64p, f64p = C.POINTER(C.c_int32), C.POINTER(C.c_int64), C.POINTER(C.c_double)
        _lib.oracle_validate.argtypes = [C.c_int32, i32p, f64p, i32p, C.c_int32, i64p, i32p, i32p]
        _lib.oracle_unifrac_all_pairs.argtypes = [C.c_int32, i32p, f64p, C.c_int32, i64p, i32p, i32p, C.c_int, f64p]
        _lib.oracle_unifrac_pair.argtypes = [C.c_int32, i32p, f64p, i64p, i32p, i32p, C.c_int, C.c_int32, C.c_int32, f64p]
        _lib.oracle_unifrac_pair_list.argtypes = [C.c_int32, i32p, f64p, C.c_int32, i64p, i32p, i32p, C.c_int,
                                                  C.c_int64, i32p, i32p, f64p]
        _lib.oracle_num_threads.restype = C.c_int
    return _lib


def _p(a, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def _arrs(parent, branch_len, indptr, indices, counts):
    return (np.ascontiguousarray(parent, dtype=np.int32), np.ascontiguousarray(branch_len, dtype=np.float64),
            np.ascontiguousarray(indptr, dtype=np.int64), np.ascontiguousarray(indices, dtype=np.int32),
            np.ascontiguousarray(counts, dtype=np.int32))


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__(f"oracle status {code}")
        self.code = code


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def validate(parent, branch_len, postorder, indptr, indices, counts) -> int:
    lib = _load()
    parent, branch_len, indptr, indices, counts = _arrs(parent, branch_len, indptr, indices, counts)
    postorder = np.ascontiguousarray(postorder, dtype=np.int32)
    return int(lib.oracle_validate(parent.shape[0], _p(parent, C.c_int32), _p(branch_len, C.c_double),
                                   _p(postorder, C.c_int32), indptr.shape[0] - 1, _p(indptr, C.c_int64),
                                   _p(indices, C.c_int32), _p(counts, C.c_int32)))


def all_pairs(parent, branch_len, indptr, indices, counts, variant) -> np.ndarray:
    """Condensed (scipy squareform order) float64 distances for every pair."""
    lib = _load()
    parent, branch_len, indptr, indices, counts = _arrs(parent, branch_len, indptr, indices, counts)
    n = indptr.shape[0] - 1
    out = np.zeros(n * (n - 1) // 2, dtype=np.float64)
    rc = lib.oracle_unifrac_all_pairs(parent.shape[0], _p(parent, C.c_int32), _p(branch_len, C.c_double), n,
                                      _p(indptr, C.c_int64), _p(indices, C.c_int32), _p(counts, C.c_int32),
                                      int(variant), _p(out, C.c_double))
    if rc != 0:
        raise OracleError(rc)
    return out


def pair(parent, branch_len, indptr, indices, counts, variant, a: int, b: int) -> float:
    lib = _load()
    parent, branch_len, indptr, indices, counts = _arrs(parent, branch_len, indptr, indices, counts)
    out = C.c_double(0.0)
    rc = lib.oracle_unifrac_pair(parent.shape[0], _p(parent, C.c_int32), _p(branch_len, C.c_double),
                                 _p(indptr, C.c_int64), _p(indices, C.c_int32), _p(counts, C.c_int32),
                                 int(variant), int(a), int(b), C.byref(out))
    if rc != 0:
        raise OracleError(rc)
    return float(out.value)


def pair_list(parent, branch_len, indptr, indices, counts, variant, pairs) -> np.ndarray:
    """float64 distances for the listed (a, b) pairs (int array [n_pairs, 2])."""
    lib = _load()
    parent, branch_len, indptr, indices, counts = _arrs(parent, branch_len, indptr, indices, counts)
    pairs = np.asarray(pairs)
    pa = np.ascontiguousarray(pairs[:, 0], dtype=np.int32)
    pb = np.ascontiguousarray(pairs[:, 1], dtype=np.int32)
    out = np.zeros(pa.shape[0], dtype=np.float64)
    rc = lib.oracle_unifrac_pair_list(parent.shape[0], _p(parent, C.c_int32), _p(branch_len, C.c_double),
                                      indptr.shape[0] - 1, _p(indptr, C.c_int64), _p(indices, C.c_int32),
                                      _p(counts, C.c_int32), int(variant), pa.shape[0],
                                      _p(pa, C.c_int32), _p(pb, C.c_int32), _p(out, C.c_double))
    if rc != 0:
        raise OracleError(rc)
    return out
