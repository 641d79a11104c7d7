"""Pins for the AllToAllv oracle (oracle/ncclx_oracle.c) against what the paper and the
definition fix -- none of these re-type the oracle's loops."""
import json
import os

import numpy as np
import pytest

import oracle
from paper_2510_20171_b200 import workloads as W

SENTINEL = 0xA5


def run(send, C, dtype, slack=7, nthreads=1):
    C = np.asarray(C, np.int64)
    R = C.shape[0]
    Cc = np.maximum(C, 0)
    npdt = send[0].dtype
    # sentinel-filled buffers of the element type
    recv = [np.frombuffer(bytes([SENTINEL]) * ((int(Cc[:, d].sum()) + slack) * npdt.itemsize), dtype=npdt).copy()
            for d in range(R)]
    RC, soff, roff, neg = oracle.alltoallv(send, C, recv, dtype, nthreads)
    return recv, RC, soff, roff, neg


def test_handworked_example(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "handworked_alltoallv.json")))
    names = sorted({x for row in g["send"] for x in row})
    code = {n: i + 1000 for i, n in enumerate(names)}
    send = [np.array([code[x] for x in row], np.uint16) for row in g["send"]]
    recv, RC, soff, roff, neg = run(send, g["C"], "bf16", slack=0)
    assert neg == 0
    assert RC.tolist() == g["RC"] and soff.tolist() == g["soff"] and roff.tolist() == g["roff"]
    for d in range(2):
        assert recv[d].tolist() == [code[x] for x in g["recv"][d]]
    back, RC2, *_ = run(recv, RC, "bf16", slack=0)
    assert RC2.tolist() == g["C"]
    for s in range(2):
        assert back[s].tolist() == [code[x] for x in g["inverse_recv"][s]]


def test_cfg1_counts_match_survey(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "cfg1_counts.json")))
    rows = W.cfg1_rows()
    assert rows.tolist() == g["rows"] and int(rows.sum()) == g["total_rows"]
    assert int(rows.sum()) * 128 * 2 == g["bytes_each_way"]


@pytest.mark.parametrize("R,seed", [(1, 0), (2, 1), (3, 2), (5, 3), (8, 4), (17, 5)])
@pytest.mark.parametrize("dtype", ["u8", "bf16", "f32"])
def test_bruteforce_definition(R, seed, dtype):
    """Tiny inputs, expected value = the definition as one comprehension over python lists."""
    rng = np.random.default_rng(seed)
    C = rng.integers(0, 6, (R, R))
    C[rng.random((R, R)) < 0.3] = 0
    npdt = oracle.NP_DTYPE[oracle.DTYPE_ID[dtype]]
    send = [W.np_values(int(C[s].sum()), dtype, 100 + s).astype(npdt, copy=False) for s in range(R)]
    recv, RC, soff, roff, neg = run(send, C, dtype, slack=3)
    for d in range(R):
        exp = [send[s][j] for s in range(R) for j in range(int(C[s, :d].sum()), int(C[s, :d + 1].sum()))]
        got = recv[d]
        assert got[:len(exp)].tobytes() == np.array(exp, npdt).tobytes()
        assert got[len(exp):].tobytes() == bytes([SENTINEL]) * (3 * npdt().itemsize)   # untouched tail
    assert (RC == C.T).all()
    assert (soff == np.cumsum(C, axis=1) - C).all()          # library routine, not the oracle's loop
    assert (roff == (np.cumsum(C, axis=0) - C).T).all()


@pytest.mark.parametrize("R", [4, 16, 64])
def test_conservation_and_roundtrip(R):
    rng = np.random.default_rng(R)
    C = rng.integers(0, 50, (R, R)) * rng.integers(0, 2, (R, R))
    send = [W.np_values(int(C[s].sum()), "bf16", s) for s in range(R)]
    recv, RC, soff, roff, _ = run(send, C, "bf16", slack=0)
    assert (RC.sum(axis=0) == C.sum(axis=1)).all()           # sum_d RC[d][s] == sum_d C[s][d]
    for d in range(R):
        assert recv[d].size == int(C[:, d].sum())
    assert sum(r.nbytes for r in recv) == sum(s.nbytes for s in send)
    a = np.sort(np.concatenate(send)); b = np.sort(np.concatenate(recv))
    assert (a == b).all()                                    # multiset of elements preserved
    back, RC2, *_ = run(recv, RC, "bf16", slack=0)           # inverse with C := RC
    assert (RC2 == C).all()
    for s in range(R):
        assert back[s].tobytes() == send[s].tobytes()


@pytest.mark.parametrize("R,c", [(2, 3), (4, 128), (8, 5), (16, 1)])
def test_uniform_counts_is_block_transpose(R, c):
    send = [W.np_values(R * c, "f32", 7 + s) for s in range(R)]
    recv, RC, *_ = run(send, np.full((R, R), c), "f32", slack=0)
    exp = np.stack(send).reshape(R, R, c).swapaxes(0, 1)     # numpy, independent of the oracle
    for d in range(R):
        assert recv[d].tobytes() == exp[d].tobytes()


def test_tagged_payload_closed_form():
    cfg = W.a2a_config(1)
    C = cfg.rows * 4                                          # u32 elements, small
    R = cfg.R
    send = [W.tagged_payload_u32(s, int(C[s].sum())).view(np.float32) for s in range(R)]
    recv, *_ = run(send, C, "f32", slack=0)
    excl = np.cumsum(C, axis=1) - C
    for d in range(R):
        exp = np.concatenate([(np.uint32(s) << np.uint32(24)) | (np.uint32(excl[s, d]) + np.arange(C[s, d], dtype=np.uint32))
                              for s in range(R)])
        assert (recv[d].view(np.uint32) == exp).all()


def test_R1_is_memcpy_and_zero_matrix_and_negative():
    x = W.np_values(37, "u8", 0)
    recv, RC, soff, roff, neg = run([x], [[37]], "u8", slack=5)
    assert recv[0][:37].tobytes() == x.tobytes() and (recv[0][37:] == SENTINEL).all() and RC.tolist() == [[37]]
    send = [W.np_values(4, "bf16", s) for s in range(3)]
    recv, RC, soff, roff, neg = run(send, np.zeros((3, 3), np.int64), "bf16", slack=4)
    assert neg == 0 and (RC == 0).all() and (soff == 0).all() and (roff == 0).all()
    assert all((r.view(np.uint8) == SENTINEL).all() for r in recv)
    C = np.array([[2, -5], [1, 1]])
    send = [W.np_values(2, "bf16", 0), W.np_values(2, "bf16", 1)]
    recv, RC, soff, roff, neg = run(send, C, "bf16", slack=0)
    assert neg == 1 and RC.tolist() == [[2, 1], [0, 1]]       # negative reported, treated as 0
    assert recv[0].tolist() == [send[0][0], send[0][1], send[1][0]] and recv[1].tolist() == [send[1][1]]


def test_threads_do_not_change_result_and_sampled_lookup():
    cfg = W.scaled_a2a(W.a2a_config(3), 256)
    C = cfg.rows * 8
    R = cfg.R
    send = [W.np_values(int(C[s].sum()), "bf16", s) for s in range(R)]
    r1, *_ = run(send, C, "bf16", nthreads=1)
    r8, *_ = run(send, C, "bf16", nthreads=8)
    assert all(a.tobytes() == b.tobytes() for a, b in zip(r1, r8))
    d = 0
    pos = np.random.default_rng(0).integers(0, int(C[:, d].sum()), 200)
    s_idx, p_idx = oracle.alltoallv_source_of(C, d, pos)
    assert all(r1[d][p] == send[s][q] for p, s, q in zip(pos, s_idx, p_idx))


def test_workload_shapes_match_survey():
    """cfg3 every source sends 16384 rows, segments 220 KB..54 MiB, rank 0 gets
    33.1 %; cfg5 7245 non-empty pairs, 32496 rows, largest message 114688 B."""
    r3 = W.cfg3_rows()
    assert (r3.sum(axis=1) == 16384).all() and r3.min() * 10240 == 225280
    assert abs(r3.max() * 10240 / 2**20 - 54.02) < 0.01 and abs(r3.sum(0)[0] / r3.sum() - 0.3312) < 1e-3
    r5 = W.cfg5_rows()
    assert int(r5.sum()) == 32496 and int((r5 > 0).sum()) == 7245 and int(r5.max()) * 14336 == 114688
