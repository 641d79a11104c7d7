"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/ncclx_b200.h declares; host-side argument validation works without a GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    import __graft_entry__ as g
    g.build()
    from paper_2510_20171_b200 import binding
    return binding.lib()


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "ncclx_b200.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ncclx_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_all_exported(L):
    from paper_2510_20171_b200 import binding
    syms = declared_symbols()
    assert len(syms) >= 20
    assert sorted(binding.SYMBOLS) == syms, "binding.SYMBOLS out of sync with the header"
    for s in syms:
        assert hasattr(L, s), f"{s} not exported by libncclx_b200.so"


def test_version_and_strerror(L):
    assert L.ncclx_version() == 200
    assert L.ncclx_strerror(0) == b"ok"
    for code in range(1, 6):
        assert len(L.ncclx_strerror(code)) > 3
    assert L.ncclx_strerror(99) == b"unknown error code"


def test_calls_fail_loudly_without_init(L):
    """No GPU work here: before ncclx_init every entry point must refuse (no CPU fallback)."""
    from paper_2510_20171_b200 import binding
    assert L.ncclx_sm_count() == 0
    assert L.ncclx_alltoallv_dev(1, 1, 1, 2, 4, 0, None) == 3
    assert L.ncclx_allreduce_sum(1, 1, 8, 2, 0, None) == 3
    assert L.ncclx_reducescatter_sum(1, 1, 8, 2, 0, None) == 3
    assert L.ncclx_alltoallv_host(1, 1, 1, 2, 4, 0, None) == 3
    assert L.ncclx_alltoallv_prepare_dev(0, 1, 1, 1, 2, 4, 0, None) == 3
    assert L.ncclx_alltoallv_execute_dev(0, None) == 3
    assert L.ncclx_alltoallv_dynamic_prepare_dev(0, 1, 1, 4, 1, 4, 1, 2, 1, 1, 2, 0, None) == 3
    assert L.ncclx_moe_topk_prepare_dev(0, 1, 2, 4, None) == 3
    assert L.ncclx_moe_dispatch_topk_execute_dev(0, 1, 1, 1, 4, 2, 16, 0, None) == 3
    assert L.ncclx_moe_combine_topk_sum_execute_dev(0, 1, 1, 1, 4, 2, 16, 0, None) == 3
    assert L.ncclx_stream_probe_ctas(2, 32, 64, 32, 1, None) == 3
    with pytest.raises(binding.NcclxError):
        binding.ncclx_finalize()


def test_param_validation(L):
    from paper_2510_20171_b200 import binding as b
    assert L.ncclx_set_param(99, 1) == 1
    assert L.ncclx_set_param(b.PARAM_COPY_BULK_ENGINES, 3) == 1
    assert L.ncclx_set_param(b.PARAM_PDL, 2) == 1
    assert b.PARAM_COUNT <= 10                      # the tuning surface stays small
    assert L.ncclx_set_param(b.PARAM_BULK_MIN_BYTES, 8) == 1
    assert L.ncclx_set_param(b.PARAM_BULK_TILE_SHIFT, 20) == 1
    b.ncclx_set_param(b.PARAM_BULK_MIN_BYTES, 4096)
    assert b.ncclx_get_param(b.PARAM_BULK_MIN_BYTES) == 4096
    b.ncclx_set_param(b.PARAM_BULK_MIN_BYTES, 1024)


def test_init_without_gpu_reports_cuda_error(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    assert L.ncclx_init(64, 0) == 4      # NCCLX_ERR_CUDA, not a silent CPU path
    assert L.ncclx_last_cuda_error() != 0
    assert L.ncclx_init(0, 0) == 1 and L.ncclx_init(5000, 0) == 1


def test_missing_library_raises(tmp_path, monkeypatch):
    from paper_2510_20171_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(ImportError):
        binding.lib()


def test_static_entry_point_checks_sizes_before_touching_cuda(L):
    """ncclx_alltoallv_static_dev (the call for users who may not allocate) validates on the host first: its fixed
    built-in scratch stops at R = 32, and the refusal names that limit."""
    from paper_2510_20171_b200 import binding as b
    assert b.STATIC_MAX_RANKS == 32 and b.ERR_TOO_LARGE == 6
    assert L.ncclx_alltoallv_static_dev(1, 1, 1, 2, None, 33, 0, None) == 6
    assert L.ncclx_alltoallv_static_dev(1, 1, 1, 2, None, 1024, 0, None) == 6
    assert b"32" in L.ncclx_strerror(6)
    assert L.ncclx_alltoallv_static_dev(1, 1, 1, 2, None, 0, 0, None) == 1
    assert L.ncclx_alltoallv_static_dev(1, 1, 1, 1, None, 4, 0, None) == 1     # counts in == counts out
    assert L.ncclx_alltoallv_static_dev(None, 1, 1, 2, None, 4, 0, None) == 1
    assert L.ncclx_alltoallv_static_dev(1, 1, 1, 2, None, 4, 9, None) == 2
    import torch
    if not torch.cuda.is_available():
        assert L.ncclx_alltoallv_static_dev(1, 1, 1, 2, None, 4, 0, None) == 4   # no device: loud, no CPU path
