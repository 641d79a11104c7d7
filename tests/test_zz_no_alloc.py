"""-m gpu: ncclx_alltoallv_static_dev, the AllToAllv for callers that are not allowed to allocate.

Some users of this library cannot call cudaMalloc at the moment they need a collective: a plug-in living inside
an application whose memory pool has already taken all of HBM, a step phase during which the framework bans
allocator calls because cudaMalloc/cudaFree stall every stream of the device, a worker that only ever receives
ready-made buffers.  For them the library has one entry point that needs no ncclx_init and keeps its scratch
(claim counters, two offset matrices, a status word) in a fixed 16.5 KiB array compiled into the device image --
which is why it stops at R = 32 and why all calls on a GPU share, and leave their traces in, the same scratch.

What is checked here: on the same inputs the new call must produce exactly what the ordinary path
(ncclx_init + ncclx_alltoallv_dev) produces -- receive buffers compared byte for byte over their FULL capacity
(sentinel tail included) and the receive-count matrix; data movement has no tolerance, the bar is bit equality,
as in tests/test_gpu_alltoallv.py.  It is checked on two calls IN A ROW with different shapes and no
synchronisation in between, so that state left in the shared scratch by the first call would show in the second.

This file is named test_zz_* so that pytest collects it last: `pytest -x` stops at the first failure and a
failure here must not hide the rest of the suite.  It sets up and tears down its own library context, so it
passes alone in a fresh process as well as after all the other test modules.
"""
import numpy as np
import pytest
import torch

import paper_2510_20171_b200 as nx
from paper_2510_20171_b200 import workloads as W

pytestmark = pytest.mark.gpu

from gpu_util import ES, back, sentinel, to_dev  # noqa: E402


def _inputs(C, dtype, seed, mis_send=0, mis_recv=0, slack=16):
    """Device buffers for one AllToAllv: (send list, count matrix on the device, capacities in bytes)."""
    C = np.asarray(C, np.int64)
    R = C.shape[0]
    Cc = np.maximum(C, 0)
    send_np = [W.np_values(int(Cc[s].sum()), dtype, seed + s) for s in range(R)]
    send = [to_dev(a, mis_send) for a in send_np]
    cap = [(int(Cc[:, d].sum()) + slack) * ES[dtype] for d in range(R)]
    return send, torch.from_numpy(C).cuda(), cap, mis_recv


def _fresh_outputs(cap, mis_recv, Cd):
    return [sentinel(c, mis_recv) for c in cap], torch.full_like(Cd, -7)


def _counts(kind, R, rng):
    if kind == "ragged":          # element-granular, many zeros: segments land on odd addresses (vector list)
        C = rng.integers(0, 700, (R, R))
        C[rng.random((R, R)) < 0.3] = 0
        return C.astype(np.int64)
    if kind == "aligned":         # multiples of 512 elements: 16-byte aligned segments (bulk list, dynamic claims)
        return (rng.integers(0, 24, (R, R)) * 512).astype(np.int64)
    if kind == "big":             # ~250 MB in all: far more tiles than engines, the claim counters are in heavy use
        return (rng.integers(0, 64, (R, R)) * 4096).astype(np.int64)
    raise ValueError(kind)


CASES = [
    # (first call, second call): (R, dtype, kind)
    ((32, "bf16", "aligned"), (5, "u8", "ragged")),
    ((7, "f32", "ragged"), (32, "bf16", "ragged")),
    ((1, "bf16", "aligned"), (16, "f16", "aligned")),
    ((32, "bf16", "big"), (32, "bf16", "aligned")),
]


def test_works_without_ncclx_init_and_reports_negative_counts():
    """Runs FIRST in this file, before the fixture below creates a workspace (and drops any context another module
    may have left): with no ncclx_init at all the call must still work, and a negative count must move nothing and
    raise bit 0 of the caller's status word."""
    try:
        nx.ncclx_finalize()
    except nx.binding.NcclxError:
        pass
    R, dtype = 6, "bf16"
    C = np.arange(R * R, dtype=np.int64).reshape(R, R) * 3 + 1
    C[2, 4] = -9
    send, Cd, cap, _ = _inputs(C, dtype, 7)
    recv, RC = _fresh_outputs(cap, 0, Cd)
    status = torch.zeros(1, dtype=torch.int32, device="cuda")
    nx.ncclx_alltoallv_static_dev(nx.device_ptr_table(send), Cd, nx.device_ptr_table(recv), RC, R, dtype,
                                  status_dev=status)
    torch.cuda.synchronize()
    assert int(status.item()) == 1
    Cc = np.maximum(C, 0)
    assert (RC.cpu().numpy() == Cc.T).all()
    # packed by source rank ascending, nothing past the packed end
    for d in range(R):
        got = back(recv[d], "bf16")
        exp = np.concatenate([back(send[s], "bf16")[int(Cc[s, :d].sum()): int(Cc[s, :d + 1].sum())] for s in range(R)])
        assert got[:exp.size].tobytes() == exp.tobytes()
        assert (got[exp.size:] == 0xA5A5).all()
    with pytest.raises(nx.binding.NcclxError):          # the ordinary path really has no workspace now
        nx.ncclx_alltoallv_dev(nx.device_ptr_table(send), Cd, nx.device_ptr_table(recv), RC, R, dtype)


@pytest.fixture(scope="module")
def ordinary_path():
    """The existing path needs its workspace; the new one must work without -- see the ordering in the tests."""
    assert torch.cuda.is_available()
    nx.ncclx_init(128, 0)
    yield
    nx.ncclx_finalize()


@pytest.mark.parametrize("first,second", CASES)
def test_two_calls_in_a_row_match_the_ordinary_path(ordinary_path, first, second):
    rng = np.random.default_rng(20171)
    stream = torch.cuda.current_stream()
    prepared = []
    for i, (R, dtype, kind) in enumerate((first, second)):
        C = _counts(kind, R, rng)
        send, Cd, cap, mis = _inputs(C, dtype, 100 * (i + 1), mis_send=0, mis_recv=0)
        st = nx.device_ptr_table(send)
        recv_new, RC_new = _fresh_outputs(cap, mis, Cd)
        recv_old, RC_old = _fresh_outputs(cap, mis, Cd)
        prepared.append((R, dtype, send, Cd, st, recv_new, RC_new, nx.device_ptr_table(recv_new),
                         recv_old, RC_old, nx.device_ptr_table(recv_old)))
    torch.cuda.synchronize()

    # the two static calls back to back on one stream, nothing in between: they share the built-in scratch
    for (R, dtype, _send, Cd, st, _rn, RC_new, rt_new, *_rest) in prepared:
        nx.ncclx_alltoallv_static_dev(st, Cd, rt_new, RC_new, R, dtype, stream)
    # the same two transfers through the ordinary entry point
    for (R, dtype, _send, Cd, st, _rn, _RCn, _rtn, _ro, RC_old, rt_old) in prepared:
        nx.ncclx_alltoallv_dev(st, Cd, rt_old, RC_old, R, dtype, stream)
    torch.cuda.synchronize()

    for n, (R, dtype, _send, Cd, _st, recv_new, RC_new, _rtn, recv_old, RC_old, _rto) in enumerate(prepared):
        assert torch.equal(RC_new, RC_old), f"call {n}: receive counts differ"
        assert torch.equal(RC_new, Cd.t().contiguous()), f"call {n}: receive counts are not the transpose"
        moved = 0
        for d in range(R):
            a, b = back(recv_new[d], "u8"), back(recv_old[d], "u8")
            assert a.tobytes() == b.tobytes(), f"call {n}: recv[{d}] differs from ncclx_alltoallv_dev"
            moved += int((a != 0xA5).sum())
        assert moved > 0 or int(Cd.sum()) == 0


def test_sizes_beyond_the_built_in_scratch_are_refused():
    t = torch.zeros(4096, dtype=torch.int64, device="cuda")
    before = t.clone()
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_alltoallv_static_dev(t, t[:1], t, t[2048:], nx.binding.STATIC_MAX_RANKS + 1, "bf16")
    assert e.value.code == nx.binding.ERR_TOO_LARGE and "32" in str(e.value)
    torch.cuda.synchronize()
    assert torch.equal(t, before)                       # refused before anything was enqueued
