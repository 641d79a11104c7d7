"""CPU oracle for the NCCLX on-device data path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

ctypes wrapper over oracle/ncclx_oracle.c (plain C, the definitions written out; see that
file's header for the paper citations).  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_2510_20171_b200 and shares no code with the CUDA path.

Arrays are numpy; bf16 / f16 values travel as uint16 bit patterns.
"""
from __future__ import annotations

import ctypes
from typing import Sequence

import numpy as np

from .build import build as _build

BF16, F32, F16, U8 = 0, 1, 2, 3
DTYPE_ID = {"bf16": BF16, "f32": F32, "f16": F16, "u8": U8}
NP_DTYPE = {BF16: np.uint16, F32: np.float32, F16: np.uint16, U8: np.uint8}

_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build())
        vp, i64p = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int64)
        L.oracle_alltoallv_offsets.argtypes = [i64p, ctypes.c_int, i64p, i64p, i64p]
        L.oracle_alltoallv_offsets.restype = ctypes.c_int
        L.oracle_alltoallv.argtypes = [vp, i64p, vp, i64p, i64p, i64p, ctypes.c_int, ctypes.c_int, ctypes.c_int]
        L.oracle_alltoallv.restype = ctypes.c_int
        for f in (L.oracle_allreduce_sum, L.oracle_reducescatter_sum):
            f.argtypes = [vp, vp, ctypes.c_size_t, ctypes.c_int, ctypes.c_int, ctypes.c_int]
            f.restype = ctypes.c_int
        L.oracle_reduce_samples.argtypes = [vp, vp, ctypes.c_size_t, ctypes.c_int, ctypes.c_int]
        L.oracle_reduce_samples.restype = ctypes.c_int
        L.oracle_alltoallv_dynamic.argtypes = [vp, i64p, ctypes.c_int, i64p, ctypes.c_int, i64p, ctypes.c_int, vp, i64p,
                                               ctypes.c_int, ctypes.c_int]
        L.oracle_alltoallv_dynamic.restype = ctypes.c_int
        i32p = ctypes.POINTER(ctypes.c_int32)
        L.oracle_moe_dispatch_topk.argtypes = [vp, i32p, i64p, vp, i64p, i64p, i64p] + [ctypes.c_int] * 5
        L.oracle_moe_dispatch_topk.restype = ctypes.c_int
        L.oracle_moe_combine_topk_sum.argtypes = [vp, i32p, i64p, vp] + [ctypes.c_int] * 5
        L.oracle_moe_combine_topk_sum.restype = ctypes.c_int
        L.oracle_f32_to_bf16_rne.argtypes = [ctypes.c_uint32]
        L.oracle_f32_to_bf16_rne.restype = ctypes.c_uint16
        L.oracle_f32_to_f16_rne.argtypes = [ctypes.c_uint32]
        L.oracle_f32_to_f16_rne.restype = ctypes.c_uint16
        _lib = L
    return _lib


def _dt(dtype) -> int:
    return DTYPE_ID[dtype] if isinstance(dtype, str) else int(dtype)


def _ptr_table(arrs: Sequence[np.ndarray]):
    tab = (ctypes.c_void_p * len(arrs))()
    for i, a in enumerate(arrs):
        assert a.flags["C_CONTIGUOUS"]
        tab[i] = a.ctypes.data
    return tab


def _i64p(a: np.ndarray):
    assert a.dtype == np.int64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))


def f32_to_bf16_rne(bits: int) -> int:
    return int(lib().oracle_f32_to_bf16_rne(bits & 0xFFFFFFFF))


def f32_to_f16_rne(bits: int) -> int:
    return int(lib().oracle_f32_to_f16_rne(bits & 0xFFFFFFFF))


def alltoallv_offsets(C: np.ndarray):
    """-> (RC, soff, roff, n_negative); all (R, R) int64, as SURVEY section 8(c.1) steps 1-3."""
    C = np.ascontiguousarray(C, dtype=np.int64)
    R = C.shape[0]
    assert C.shape == (R, R)
    RC, soff, roff = (np.empty((R, R), np.int64) for _ in range(3))
    neg = lib().oracle_alltoallv_offsets(_i64p(C), R, _i64p(RC), _i64p(soff), _i64p(roff))
    return RC, soff, roff, neg


def alltoallv(send: Sequence[np.ndarray], C: np.ndarray, recv: Sequence[np.ndarray], dtype, nthreads: int = 1):
    """Writes into the caller's recv arrays IN PLACE (they carry their pre-call bytes, e.g. the
    0xA5 sentinel) and returns (RC, soff, roff, n_negative).  send/recv are 1-D arrays whose
    itemsize equals the dtype's element size; counts are in elements."""
    dt = _dt(dtype)
    C = np.ascontiguousarray(C, dtype=np.int64)
    R = C.shape[0]
    assert C.shape == (R, R) and len(send) == R and len(recv) == R
    e = lib().oracle_elem_size(dt)
    Cc = np.maximum(C, 0)
    for s in range(R):
        assert send[s].itemsize == e and send[s].size >= int(Cc[s].sum()), "send buffer too small"
    for d in range(R):
        assert recv[d].itemsize == e and recv[d].size >= int(Cc[:, d].sum()), "recv buffer too small"
    RC, soff, roff = (np.empty((R, R), np.int64) for _ in range(3))
    st, rt = _ptr_table(send), _ptr_table(recv)
    neg = lib().oracle_alltoallv(st, _i64p(C), rt, _i64p(RC), _i64p(soff), _i64p(roff), R, dt, nthreads)
    assert neg >= 0
    return RC, soff, roff, neg


def alltoallv_dynamic(send: Sequence[np.ndarray], split_lengths: np.ndarray, indices: np.ndarray, block_lens: np.ndarray,
                      max_block_len: int, recvbuffs: Sequence[Sequence[np.ndarray]], dtype):
    """The paper's AllToAllvDynamic.  split_lengths (R, n), indices (R, maxIndices),
    block_lens (R, R); recvbuffs[d][s] are written IN PLACE at the sender's split offsets.
    -> (recvAllSplitLengths (R, R, n), status bits)."""
    dt = _dt(dtype)
    Ls = np.ascontiguousarray(split_lengths, dtype=np.int64)
    idx = np.ascontiguousarray(indices, dtype=np.int64)
    bl = np.ascontiguousarray(block_lens, dtype=np.int64)
    R, n = Ls.shape
    assert bl.shape == (R, R) and idx.shape[0] == R and len(send) == R and len(recvbuffs) == R
    e = lib().oracle_elem_size(dt)
    tot = np.maximum(Ls, 0).sum(axis=1)
    flat = []
    for d in range(R):
        assert len(recvbuffs[d]) == R
        for s in range(R):
            assert recvbuffs[d][s].itemsize == e and recvbuffs[d][s].size >= int(tot[s]), "recvbuff too small"
            flat.append(recvbuffs[d][s])
    for s in range(R):
        assert send[s].itemsize == e and send[s].size >= int(tot[s])
    out = np.empty((R, R, n), np.int64)
    st = lib().oracle_alltoallv_dynamic(_ptr_table(send), _i64p(Ls), n, _i64p(idx), idx.shape[1], _i64p(bl), max_block_len,
                                        _ptr_table(flat), _i64p(out), R, dt)
    assert st >= 0
    return out, st


def _i32p(a: np.ndarray):
    assert a.dtype == np.int32 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))


def moe_dispatch_topk(tokens: Sequence[np.ndarray], pos: np.ndarray, Crows: np.ndarray, recv: Sequence[np.ndarray], width: int, dtype):
    """Top-k dispatch (virtual sorted send buffer, see ncclx_oracle.c).  tokens[s]: (T*width,), pos: (R, T, k) int32,
    Crows: (R, R) rows; recv[d] written in place.  -> (RC rows, status)."""
    dt = _dt(dtype)
    pos = np.ascontiguousarray(pos, dtype=np.int32)
    C = np.ascontiguousarray(Crows, dtype=np.int64)
    R, T, k = pos.shape
    assert C.shape == (R, R)
    for s in range(R):
        assert tokens[s].size >= T * width
    for d in range(R):
        assert recv[d].size >= int(np.maximum(C[:, d], 0).sum()) * width
    RC, soff, roff = (np.empty((R, R), np.int64) for _ in range(3))
    st = lib().oracle_moe_dispatch_topk(_ptr_table(tokens), _i32p(pos), _i64p(C), _ptr_table(recv), _i64p(RC), _i64p(soff),
                                        _i64p(roff), R, T, k, width, dt)
    assert st >= 0
    return RC, st


def moe_combine_topk_sum(Y: Sequence[np.ndarray], pos: np.ndarray, Crows: np.ndarray, width: int, dtype):
    """Top-k combine fused with the fixed-order fp32 sum.  -> (list of R arrays (T*width,), status)."""
    dt = _dt(dtype)
    pos = np.ascontiguousarray(pos, dtype=np.int32)
    C = np.ascontiguousarray(Crows, dtype=np.int64)
    R, T, k = pos.shape
    out = [np.zeros(T * width, NP_DTYPE[dt]) for _ in range(R)]
    st = lib().oracle_moe_combine_topk_sum(_ptr_table(Y), _i32p(pos), _i64p(C), _ptr_table(out), R, T, k, width, dt)
    assert st >= 0
    return out, st


def allreduce_sum(send: Sequence[np.ndarray], dtype, nthreads: int = 1, out: Sequence[np.ndarray] | None = None):
    dt = _dt(dtype)
    R, n = len(send), send[0].size
    assert all(a.size == n and a.dtype == NP_DTYPE[dt] for a in send)
    if out is None:
        out = [np.empty(n, NP_DTYPE[dt]) for _ in range(R)]
    rc = lib().oracle_allreduce_sum(_ptr_table(send), _ptr_table(out), n, R, dt, nthreads)
    assert rc == 0
    return out


def reducescatter_sum(send: Sequence[np.ndarray], dtype, nthreads: int = 1, out: Sequence[np.ndarray] | None = None):
    dt = _dt(dtype)
    R, N = len(send), send[0].size
    assert N % R == 0 and all(a.size == N and a.dtype == NP_DTYPE[dt] for a in send)
    n = N // R
    if out is None:
        out = [np.empty(n, NP_DTYPE[dt]) for _ in range(R)]
    rc = lib().oracle_reducescatter_sum(_ptr_table(send), _ptr_table(out), n, R, dt, nthreads)
    assert rc == 0
    return out


def reduce_samples(vals: np.ndarray, dtype) -> np.ndarray:
    """vals: (R, T) gathered inputs for T sampled element positions -> (T,) reduced outputs."""
    dt = _dt(dtype)
    vals = np.ascontiguousarray(vals)
    assert vals.dtype == NP_DTYPE[dt] and vals.ndim == 2
    R, T = vals.shape
    out = np.empty(T, NP_DTYPE[dt])
    rc = lib().oracle_reduce_samples(vals.ctypes.data, out.ctypes.data, T, R, dt)
    assert rc == 0
    return out


def alltoallv_source_of(C: np.ndarray, d: int, pos: np.ndarray):
    """Sampled form for full-size parity: for element positions `pos` inside the packed part of
    recv[d], return (s, src_pos) such that recv[d][pos] = send[s][src_pos], computed one by one
    from the definition (linear walk over sources)."""
    RC, soff, roff, _ = alltoallv_offsets(C)
    R = RC.shape[0]
    s_out = np.empty(len(pos), np.int64)
    p_out = np.empty(len(pos), np.int64)
    for t, p in enumerate(pos):
        p = int(p)
        found = False
        for s in range(R):
            lo = int(roff[d, s])
            if lo <= p < lo + int(RC[d, s]):
                s_out[t], p_out[t] = s, int(soff[s, d]) + (p - lo)
                found = True
                break
        assert found, "position beyond the packed end"
    return s_out, p_out
