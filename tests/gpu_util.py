"""Helpers for the -m gpu parity tests: move seeded inputs to the device, call the C ABI
through the binding, bring results back for the oracle comparison.  No method arithmetic."""
import numpy as np
import torch

import paper_2510_20171_b200 as nx

SENT8 = 0xA5
NP_OF = {"bf16": np.uint16, "f16": np.uint16, "f32": np.float32, "u8": np.uint8}
ES = {"bf16": 2, "f16": 2, "f32": 4, "u8": 1}


def to_dev(a: np.ndarray, pad_front_bytes: int = 0) -> torch.Tensor:
    """uint8 device tensor holding a's bytes, optionally starting `pad_front_bytes` into a
    256B-aligned allocation (to create misaligned base pointers)."""
    raw = np.frombuffer(a.tobytes(), np.uint8)
    buf = torch.empty(raw.size + pad_front_bytes + 64, dtype=torch.uint8, device="cuda")
    view = buf[pad_front_bytes:pad_front_bytes + raw.size]
    view.copy_(torch.from_numpy(raw.copy()))
    return view


def sentinel(nbytes: int, pad_front_bytes: int = 0) -> torch.Tensor:
    buf = torch.full((nbytes + pad_front_bytes + 64,), SENT8, dtype=torch.uint8, device="cuda")
    return buf[pad_front_bytes:pad_front_bytes + nbytes]


def back(t: torch.Tensor, dtype: str) -> np.ndarray:
    return t.cpu().numpy().view(NP_OF[dtype])


def run_a2a(send_np, C, dtype, slack_elems=16, stream=None, mis_send=0, mis_recv=0):
    """-> (recv list of np arrays over FULL capacity, RC np, (soff, roff) np, status)"""
    C = np.asarray(C, np.int64)
    R = C.shape[0]
    es = ES[dtype]
    Cc = np.maximum(C, 0)
    send = [to_dev(a, mis_send) for a in send_np]
    cap = [int(Cc[:, d].sum()) + slack_elems for d in range(R)]
    recv = [sentinel(c * es, mis_recv) for c in cap]
    Cd = torch.from_numpy(C).cuda()
    RCd = torch.full_like(Cd, -7)
    st, rt = nx.device_ptr_table(send), nx.device_ptr_table(recv)
    nx.ncclx_alltoallv_dev(st, Cd, rt, RCd, R, dtype, stream)
    offs = nx.ncclx_alltoallv_last_offsets(R, stream)
    status = nx.ncclx_device_status(stream)
    torch.cuda.synchronize()
    return [back(r, dtype) for r in recv], RCd.cpu().numpy(), offs, status


def oracle_a2a(send_np, C, dtype, slack_elems=16):
    import oracle
    C = np.asarray(C, np.int64)
    R = C.shape[0]
    Cc = np.maximum(C, 0)
    exp = [np.frombuffer(bytes([SENT8]) * ((int(Cc[:, d].sum()) + slack_elems) * ES[dtype]), NP_OF[dtype]).copy()
           for d in range(R)]
    RC, soff, roff, neg = oracle.alltoallv(send_np, C, exp, dtype, nthreads=8)
    return exp, RC, soff, roff, neg


def assert_a2a_matches(send_np, C, dtype, **kw):
    got, RC, (soff, roff), status = run_a2a(send_np, C, dtype, **kw)
    exp, eRC, esoff, eroff, neg = oracle_a2a(send_np, C, dtype)
    assert (RC == eRC).all(), "recvcounts mismatch"
    assert (soff == esoff).all() and (roff == eroff).all(), "offset matrices mismatch"
    assert status == (1 if neg else 0)
    for d in range(len(exp)):
        assert got[d].tobytes() == exp[d].tobytes(), f"recv[{d}] differs from the oracle"
    return got, RC
