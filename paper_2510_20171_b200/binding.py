"""Thin ctypes binding over libncclx_b200.so -- argument marshalling only.

Same names as include/ncclx_b200.h.  Every step of the hot path runs in the library's CUDA
kernels; PyTorch appears only as the owner of device memory and streams.  There is NO
fallback: if the shared library is missing or fails to load, importing a symbol raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Sequence

HERE = os.path.dirname(os.path.abspath(__file__))
# NCCLX_B200_LIB selects another build of the same library (tests/test_zy_barrier_fallback.py's forced-time-out one); never a fallback
LIB_PATH = os.environ.get("NCCLX_B200_LIB") or os.path.join(HERE, "libncclx_b200.so")

BF16, F32, F16, U8 = 0, 1, 2, 3
DTYPE_ID = {"bf16": BF16, "f32": F32, "f16": F16, "u8": U8}

PARAM_BULK_MIN_BYTES = 0
PARAM_REDUCE_CTAS_PER_SM = 1
PARAM_PROFILE = 2
PARAM_BULK_TILE_SHIFT = 3
PARAM_PDL = 4
PARAM_COPY_KMAX = 5
PARAM_FUSED_MAX_RANKS = 6
PARAM_COPY_BULK_ENGINES = 7
PARAM_HOST_ZERO_COPY = 8
PARAM_REDUCECOPY_TMA = 9
PARAM_COUNT = 10
NUM_PLANS = 4
STATIC_MAX_RANKS = 32            # NCCLX_STATIC_MAX_RANKS
ERR_TOO_LARGE = 6                # NCCLX_ERR_TOO_LARGE

KERNEL_COUNTS, KERNEL_COPY, KERNEL_REDUCE, KERNEL_DYN, KERNEL_TOPK, KERNEL_FUSED = 0, 1, 2, 3, 4, 5

# every symbol include/ncclx_b200.h declares (tests check the .so exports all of them)
SYMBOLS = [
    "ncclx_init", "ncclx_finalize", "ncclx_strerror", "ncclx_last_cuda_error", "ncclx_last_cuda_error_string",
    "ncclx_version", "ncclx_alltoallv_dev", "ncclx_alltoallv_last_offsets", "ncclx_device_status",
    "ncclx_allreduce_sum", "ncclx_reducescatter_sum", "ncclx_alltoallv_host", "ncclx_allreduce_sum_host",
    "ncclx_reducescatter_sum_host", "ncclx_set_param", "ncclx_get_param", "ncclx_profile_read",
    "ncclx_profile_reset", "ncclx_launch_count", "ncclx_sm_count", "ncclx_init_dynamic", "ncclx_alltoallv_dynamic_dev",
    "ncclx_reducecopy_sum", "ncclx_moe_dispatch_topk_dev", "ncclx_moe_combine_topk_sum_dev",
    "ncclx_alltoallv_prepare_dev", "ncclx_alltoallv_execute_dev", "ncclx_stream_probe", "ncclx_stream_probe_ctas",
    "ncclx_alltoallv_dynamic_prepare_dev", "ncclx_moe_topk_prepare_dev", "ncclx_moe_dispatch_topk_execute_dev",
    "ncclx_moe_combine_topk_sum_execute_dev", "ncclx_alltoallv_static_dev",
]


class NcclxError(RuntimeError):
    def __init__(self, code: int, where: str):
        L = lib()
        msg = L.ncclx_strerror(code).decode()
        if code == 4:
            msg += f" ({L.ncclx_last_cuda_error()}: {L.ncclx_last_cuda_error_string().decode()})"
        super().__init__(f"{where}: {msg} [code {code}]")
        self.code = code


_lib = None


def lib() -> ctypes.CDLL:
    """Loads the CUDA library; fails loudly when it has not been built (no CPU fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                              "(nvcc, sm_100a). There is no CPU fallback.")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, i64p = ctypes.c_void_p, ctypes.c_int64, ctypes.POINTER(ctypes.c_int64)
        L.ncclx_init.argtypes = [ctypes.c_int, ctypes.c_int]
        L.ncclx_strerror.argtypes = [ctypes.c_int]
        L.ncclx_strerror.restype = ctypes.c_char_p
        L.ncclx_last_cuda_error_string.restype = ctypes.c_char_p
        L.ncclx_alltoallv_dev.argtypes = [vp, vp, vp, vp, ctypes.c_int, ctypes.c_int, vp]
        L.ncclx_alltoallv_static_dev.argtypes = [vp, vp, vp, vp, vp, ctypes.c_int, ctypes.c_int, vp]
        L.ncclx_alltoallv_prepare_dev.argtypes = [ctypes.c_int, vp, vp, vp, vp, ctypes.c_int, ctypes.c_int, vp]
        L.ncclx_alltoallv_execute_dev.argtypes = [ctypes.c_int, vp]
        L.ncclx_alltoallv_last_offsets.argtypes = [vp, vp, ctypes.c_int, vp]
        L.ncclx_device_status.argtypes = [ctypes.POINTER(ctypes.c_uint32), vp]
        for f in (L.ncclx_allreduce_sum, L.ncclx_reducescatter_sum, L.ncclx_allreduce_sum_host,
                  L.ncclx_reducescatter_sum_host):
            f.argtypes = [vp, vp, ctypes.c_size_t, ctypes.c_int, ctypes.c_int, vp]
        L.ncclx_alltoallv_host.argtypes = [vp, vp, vp, vp, ctypes.c_int, ctypes.c_int, vp]
        L.ncclx_init_dynamic.argtypes = [ctypes.c_int, i64]
        L.ncclx_alltoallv_dynamic_dev.argtypes = [vp, vp, ctypes.c_int, vp, ctypes.c_int, vp, ctypes.c_int, vp, vp,
                                                  ctypes.c_int, ctypes.c_int, vp]
        L.ncclx_reducecopy_sum.argtypes = [vp, vp, vp, vp, ctypes.c_size_t, ctypes.c_int, ctypes.c_size_t, ctypes.c_int, vp]
        L.ncclx_moe_dispatch_topk_dev.argtypes = [vp, vp, vp, vp, vp] + [ctypes.c_int] * 5 + [vp]
        L.ncclx_moe_combine_topk_sum_dev.argtypes = [vp, vp, vp, vp] + [ctypes.c_int] * 5 + [vp]
        L.ncclx_stream_probe.argtypes = [ctypes.c_int, vp, vp, ctypes.c_size_t, vp]
        L.ncclx_stream_probe_ctas.argtypes = [ctypes.c_int, vp, vp, ctypes.c_size_t, ctypes.c_int, vp]
        L.ncclx_alltoallv_dynamic_prepare_dev.argtypes = [ctypes.c_int, vp, vp, ctypes.c_int, vp, ctypes.c_int, vp, ctypes.c_int, vp, vp,
                                                          ctypes.c_int, ctypes.c_int, vp]
        L.ncclx_moe_topk_prepare_dev.argtypes = [ctypes.c_int, vp, vp, ctypes.c_int, vp]
        L.ncclx_moe_dispatch_topk_execute_dev.argtypes = [ctypes.c_int, vp, vp, vp] + [ctypes.c_int] * 4 + [vp]
        L.ncclx_moe_combine_topk_sum_execute_dev.argtypes = [ctypes.c_int, vp, vp, vp] + [ctypes.c_int] * 4 + [vp]
        L.ncclx_set_param.argtypes = [ctypes.c_int, i64]
        L.ncclx_get_param.argtypes = [ctypes.c_int, i64p]
        L.ncclx_profile_read.argtypes = [ctypes.c_int, ctypes.POINTER(ctypes.c_double), i64p]
        L.ncclx_launch_count.restype = i64
        _lib = L
    return _lib


def _ck(code: int, where: str) -> None:
    if code != 0:
        raise NcclxError(code, where)


def _dt(dtype) -> int:
    return DTYPE_ID[dtype] if isinstance(dtype, str) else int(dtype)


def _stream(stream) -> int:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return int(getattr(stream, "cuda_stream", stream))


def _ptr(x) -> int:
    """Device/host address of a torch tensor, numpy array or raw int."""
    if x is None:
        return 0
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    return int(x)


# ---- lifetime ------------------------------------------------------------------------------

def ncclx_init(max_ranks: int = 128, device: int = 0) -> None:
    _ck(lib().ncclx_init(max_ranks, device), "ncclx_init")


def ncclx_finalize() -> None:
    _ck(lib().ncclx_finalize(), "ncclx_finalize")


def ncclx_version() -> int:
    return lib().ncclx_version()


def ncclx_sm_count() -> int:
    return lib().ncclx_sm_count()


# ---- device entry points ---------------------------------------------------------------------

def device_ptr_table(tensors: Sequence, device=None):
    """DEVICE int64 tensor holding the data_ptr of each tensor (the `send` / `recv` tables)."""
    import torch
    dev = device if device is not None else tensors[0].device
    return torch.tensor([t.data_ptr() for t in tensors], dtype=torch.int64, device=dev)


def ncclx_alltoallv_dev(send_table, sendcounts_dev, recv_table, recvcounts_dev, R: int, dtype, stream=None) -> None:
    _ck(lib().ncclx_alltoallv_dev(_ptr(send_table), _ptr(sendcounts_dev), _ptr(recv_table), _ptr(recvcounts_dev),
                                  R, _dt(dtype), _stream(stream)), "ncclx_alltoallv_dev")


def ncclx_alltoallv_static_dev(send_table, sendcounts_dev, recv_table, recvcounts_dev, R: int, dtype, stream=None,
                               status_dev=None) -> None:
    """AllToAllv for callers that may not allocate device memory (a plug-in inside an application whose pool owns
    all of HBM, a phase in which the framework forbids cudaMalloc because it stalls every stream, a worker that is
    only handed finished buffers).  Needs no ncclx_init and allocates nothing: its scratch is a fixed 16.5 KiB array
    built into the library, hence R <= STATIC_MAX_RANKS (NcclxError code ERR_TOO_LARGE above that), one call in
    flight per GPU at a time, and the first call on a GPU (which does the one-time set-up) made outside stream
    capture.  Same arguments and results as ncclx_alltoallv_dev; `status_dev`: optional uint32 device tensor that
    gets bit 0 OR-ed in when a negative count was seen."""
    _ck(lib().ncclx_alltoallv_static_dev(_ptr(send_table), _ptr(sendcounts_dev), _ptr(recv_table), _ptr(recvcounts_dev),
                                         _ptr(status_dev), R, _dt(dtype), _stream(stream)), "ncclx_alltoallv_static_dev")


def ncclx_alltoallv_prepare_dev(plan: int, send_table, sendcounts_dev, recv_table, recvcounts_dev, R: int, dtype,
                                stream=None) -> None:
    _ck(lib().ncclx_alltoallv_prepare_dev(plan, _ptr(send_table), _ptr(sendcounts_dev), _ptr(recv_table),
                                          _ptr(recvcounts_dev), R, _dt(dtype), _stream(stream)), "ncclx_alltoallv_prepare_dev")


def ncclx_alltoallv_execute_dev(plan: int, stream=None) -> None:
    _ck(lib().ncclx_alltoallv_execute_dev(plan, _stream(stream)), "ncclx_alltoallv_execute_dev")


def ncclx_alltoallv_last_offsets(R: int, stream=None):
    import numpy as np
    soff = np.empty((R, R), np.int64)
    roff = np.empty((R, R), np.int64)
    _ck(lib().ncclx_alltoallv_last_offsets(soff.ctypes.data, roff.ctypes.data, R, _stream(stream)),
        "ncclx_alltoallv_last_offsets")
    return soff, roff


def ncclx_device_status(stream=None) -> int:
    st = ctypes.c_uint32(0)
    _ck(lib().ncclx_device_status(ctypes.byref(st), _stream(stream)), "ncclx_device_status")
    return st.value


def ncclx_init_dynamic(max_splits: int, max_segments: int) -> None:
    _ck(lib().ncclx_init_dynamic(max_splits, max_segments), "ncclx_init_dynamic")


def ncclx_alltoallv_dynamic_dev(send_table, split_lengths_dev, nsplits: int, indices_dev, max_indices: int, block_lens_dev,
                                max_block_len: int, recvbuffs_table, recv_all_split_lengths_dev, R: int, dtype,
                                stream=None) -> None:
    _ck(lib().ncclx_alltoallv_dynamic_dev(_ptr(send_table), _ptr(split_lengths_dev), nsplits, _ptr(indices_dev), max_indices,
                                          _ptr(block_lens_dev), max_block_len, _ptr(recvbuffs_table),
                                          _ptr(recv_all_split_lengths_dev), R, _dt(dtype), _stream(stream)),
        "ncclx_alltoallv_dynamic_dev")


def ncclx_alltoallv_dynamic_prepare_dev(plan: int, send_table, split_lengths_dev, nsplits: int, indices_dev, max_indices: int,
                                        block_lens_dev, max_block_len: int, recvbuffs_table, recv_all_split_lengths_dev,
                                        R: int, dtype, stream=None) -> None:
    _ck(lib().ncclx_alltoallv_dynamic_prepare_dev(plan, _ptr(send_table), _ptr(split_lengths_dev), nsplits, _ptr(indices_dev),
                                                  max_indices, _ptr(block_lens_dev), max_block_len, _ptr(recvbuffs_table),
                                                  _ptr(recv_all_split_lengths_dev), R, _dt(dtype), _stream(stream)),
        "ncclx_alltoallv_dynamic_prepare_dev")


def ncclx_moe_topk_prepare_dev(plan: int, sendcounts_rows_dev, recvcounts_rows_dev, R: int, stream=None) -> None:
    _ck(lib().ncclx_moe_topk_prepare_dev(plan, _ptr(sendcounts_rows_dev), _ptr(recvcounts_rows_dev), R, _stream(stream)),
        "ncclx_moe_topk_prepare_dev")


def ncclx_moe_dispatch_topk_execute_dev(plan: int, tokens_table, pos_dev, recv_table, T: int, k: int, width: int, dtype,
                                        stream=None) -> None:
    _ck(lib().ncclx_moe_dispatch_topk_execute_dev(plan, _ptr(tokens_table), _ptr(pos_dev), _ptr(recv_table), T, k, width,
                                                  _dt(dtype), _stream(stream)), "ncclx_moe_dispatch_topk_execute_dev")


def ncclx_moe_combine_topk_sum_execute_dev(plan: int, expert_out_table, pos_dev, out_table, T: int, k: int, width: int, dtype,
                                           stream=None) -> None:
    _ck(lib().ncclx_moe_combine_topk_sum_execute_dev(plan, _ptr(expert_out_table), _ptr(pos_dev), _ptr(out_table), T, k, width,
                                                     _dt(dtype), _stream(stream)), "ncclx_moe_combine_topk_sum_execute_dev")


def ncclx_allreduce_sum(send_table, recv_table, count: int, R: int, dtype, stream=None) -> None:
    _ck(lib().ncclx_allreduce_sum(_ptr(send_table), _ptr(recv_table), count, R, _dt(dtype), _stream(stream)),
        "ncclx_allreduce_sum")


def ncclx_moe_dispatch_topk_dev(tokens_table, pos_dev, sendcounts_rows_dev, recv_table, recvcounts_rows_dev, R: int, T: int,
                                k: int, width: int, dtype, stream=None) -> None:
    _ck(lib().ncclx_moe_dispatch_topk_dev(_ptr(tokens_table), _ptr(pos_dev), _ptr(sendcounts_rows_dev), _ptr(recv_table),
                                          _ptr(recvcounts_rows_dev), R, T, k, width, _dt(dtype), _stream(stream)),
        "ncclx_moe_dispatch_topk_dev")


def ncclx_moe_combine_topk_sum_dev(expert_out_table, pos_dev, sendcounts_rows_dev, out_table, R: int, T: int, k: int,
                                   width: int, dtype, stream=None) -> None:
    _ck(lib().ncclx_moe_combine_topk_sum_dev(_ptr(expert_out_table), _ptr(pos_dev), _ptr(sendcounts_rows_dev),
                                             _ptr(out_table), R, T, k, width, _dt(dtype), _stream(stream)),
        "ncclx_moe_combine_topk_sum_dev")


def ncclx_reducecopy_sum(a, b, out, fwd, count: int, dtype, chunk_bytes: int = 0, num_ctas: int = 0, stream=None) -> None:
    _ck(lib().ncclx_reducecopy_sum(_ptr(a), _ptr(b), _ptr(out), _ptr(fwd), count, _dt(dtype), chunk_bytes, num_ctas,
                                   _stream(stream)), "ncclx_reducecopy_sum")


def ncclx_reducescatter_sum(send_table, recv_table, recvcount: int, R: int, dtype, stream=None) -> None:
    _ck(lib().ncclx_reducescatter_sum(_ptr(send_table), _ptr(recv_table), recvcount, R, _dt(dtype), _stream(stream)),
        "ncclx_reducescatter_sum")


# ---- host-buffer entry points ------------------------------------------------------------------

def _host_table(bufs: Sequence):
    tab = (ctypes.c_void_p * len(bufs))()
    for i, b in enumerate(bufs):
        tab[i] = _ptr(b)
    return tab


def ncclx_alltoallv_host(send: Sequence, sendcounts_host, recv: Sequence, recvcounts_host, R: int, dtype,
                         stream=None) -> None:
    st, rt = _host_table(send), _host_table(recv)
    _ck(lib().ncclx_alltoallv_host(ctypes.addressof(st), _ptr(sendcounts_host), ctypes.addressof(rt),
                                   _ptr(recvcounts_host), R, _dt(dtype), _stream(stream)), "ncclx_alltoallv_host")


def ncclx_allreduce_sum_host(send: Sequence, recv: Sequence, count: int, R: int, dtype, stream=None) -> None:
    st, rt = _host_table(send), _host_table(recv)
    _ck(lib().ncclx_allreduce_sum_host(ctypes.addressof(st), ctypes.addressof(rt), count, R, _dt(dtype),
                                       _stream(stream)), "ncclx_allreduce_sum_host")


def ncclx_reducescatter_sum_host(send: Sequence, recv: Sequence, recvcount: int, R: int, dtype, stream=None) -> None:
    st, rt = _host_table(send), _host_table(recv)
    _ck(lib().ncclx_reducescatter_sum_host(ctypes.addressof(st), ctypes.addressof(rt), recvcount, R, _dt(dtype),
                                           _stream(stream)), "ncclx_reducescatter_sum_host")


# ---- tuning / measurement -------------------------------------------------------------------------

def ncclx_stream_probe(mode: int, src, dst, nbytes: int, stream=None) -> None:
    _ck(lib().ncclx_stream_probe(mode, _ptr(src), _ptr(dst), nbytes, _stream(stream)), "ncclx_stream_probe")


def ncclx_stream_probe_ctas(mode: int, src, dst, nbytes: int, num_ctas: int, stream=None) -> None:
    _ck(lib().ncclx_stream_probe_ctas(mode, _ptr(src), _ptr(dst), nbytes, num_ctas, _stream(stream)), "ncclx_stream_probe_ctas")


def ncclx_set_param(param: int, value: int) -> None:
    _ck(lib().ncclx_set_param(param, value), "ncclx_set_param")


def ncclx_get_param(param: int) -> int:
    v = ctypes.c_int64(0)
    _ck(lib().ncclx_get_param(param, ctypes.byref(v)), "ncclx_get_param")
    return v.value


def ncclx_profile_read(kernel: int):
    ms, n = ctypes.c_double(0), ctypes.c_int64(0)
    _ck(lib().ncclx_profile_read(kernel, ctypes.byref(ms), ctypes.byref(n)), "ncclx_profile_read")
    return ms.value, n.value


def ncclx_profile_reset() -> None:
    _ck(lib().ncclx_profile_reset(), "ncclx_profile_reset")


def ncclx_launch_count() -> int:
    return lib().ncclx_launch_count()
