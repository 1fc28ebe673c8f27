"""The C-ABI library builds for sm_100a, loads without a GPU, and exports every symbol that
include/unifrac_b200.h declares (no compute calls here)."""
import os
import re
import subprocess

from paper_2107_05397_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "unifrac_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return set(re.findall(r"\b(unifrac_[a-z_]+)\s*\(", src)) - {"unifrac_alloc_fn"}


def test_header_symbols_are_exported_and_bound():
    lib = binding.load()
    declared = _declared()
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert getattr(lib, name) is not None
    out = subprocess.run(["nm", "-D", "--defined-only", build.LIB], capture_output=True, text=True).stdout
    for name in declared:
        assert re.search(rf"\bT {name}\b", out), name


def test_version_and_status_strings_without_gpu():
    assert binding.unifrac_abi_version() == binding.ABI_VERSION
    assert binding.unifrac_status_string(0) == "ok"
    assert "tree" in binding.unifrac_status_string(binding.ERR_INVALID_TREE)


def test_host_checkable_errors_return_before_any_cuda_work():
    import ctypes as C
    lib = binding.load()
    null = binding.CSR(None, None, None)
    rc = lib.unifrac_dm(10, None, None, None, null, 5, 0, 0, None, binding.ALLOC_FN(0), None, 0, None)
    assert rc == binding.ERR_INVALID_ARG
    rc = lib.unifrac_dm_host(10, None, None, None, null, 5, 0, 0, None, 0)
    assert rc == binding.ERR_INVALID_ARG


def test_library_is_built_for_sm_100a_with_tcgen05_tma_and_bulk_copies():
    sass = subprocess.run(["cuobjdump", "-sass", build.LIB], capture_output=True, text=True).stdout
    assert "sm_100a" in sass
    assert "UBLKCP" in sass            # cp.async.bulk (TMA bulk copy): Mantel row staging, debug stripe kernel
    assert "UTMALDG" in sass           # cp.async.bulk.tensor (TMA tile loads): k_dense16 / k_gram operand staging
    assert "UTCIMMA" in sass           # tcgen05.mma kind::i8: the Gram kernel did not fall back to CUDA cores
    assert "LDTM" in sass              # tcgen05.ld: TMEM accumulators read back by the Gram epilogue


def test_shard_of_pair_is_a_partition_by_blocks_of_12_tiles():
    """unifrac_shard_of_pair (host helper): symmetric, constant on 1536 x 1536 sample blocks, round-robin over blocks."""
    f = binding.unifrac_shard_of_pair
    assert f(0, 1, 1) == 0 and f(5, 5, 4) == -1
    assert f(3, 7, 4) == f(7, 3, 4) == 0                     # block (0, 0)
    assert f(0, 1535, 4) == 0 and f(0, 1536, 4) == 1         # block (0, 1) = linear index 1
    assert f(1536, 3071, 4) == 2 and f(0, 3072, 4) == 3      # (1, 1) -> 2, (0, 2) -> 3
    assert f(1536, 3072, 4) == 0 and f(3072, 3073, 4) == 1   # (1, 2) -> 4 % 4, (2, 2) -> 5 % 4
