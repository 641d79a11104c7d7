"""Pins for the AllToAllvDynamic oracle: the paper's own Fig. 17 worked example,
brute force from the definition on tiny inputs, reduction to the plain AllToAllv when every rank's
index list is the identity partition."""
import json
import os

import numpy as np
import pytest

import oracle
from paper_2510_20171_b200 import workloads as W

SENT = 0xA5A5


def test_fig17_worked_example(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "fig17_alltoallvdynamic.json")))
    L0 = np.array(g["sendSplitLengths"], np.int64)
    n, R = len(L0), 2
    # rank 0 is the paper's example; rank 1 (not shown in the text) sends nothing
    Ls = np.stack([L0, np.zeros(n, np.int64)])
    idx = np.zeros((R, 8), np.int64)
    idx[0, :5] = g["sendIndices"]
    bl = np.array([g["sendIndicesBlockLens"], [0, 0]], np.int64)
    send = [np.arange(1, int(L0.sum()) + 1, dtype=np.uint16), np.zeros(0, np.uint16)]
    recv = [[np.full(int(L0.sum()), SENT, np.uint16), np.zeros(0, np.uint16)] for _ in range(R)]
    allL, st = oracle.alltoallv_dynamic(send, Ls, idx, bl, 3, recv, "bf16")
    assert st == 0
    off = np.concatenate([[0], np.cumsum(L0)])
    for d, splits in ((0, g["to_rank0_splits"]), (1, g["to_rank1_splits"])):
        exp = np.full(int(L0.sum()), SENT, np.uint16)
        for i in splits:
            exp[off[i]:off[i + 1]] = send[0][off[i]:off[i + 1]]
        assert (recv[d][0] == exp).all()
    # "index 0 are sent to both rank 0 and rank 1 due to duplicated experts"; amounts 128+256 and 128+256+128
    assert int((recv[0][0] != SENT).sum()) == g["to_rank0_amount"] and int((recv[1][0] != SENT).sum()) == g["to_rank1_amount"]
    # "on rank 1 receiver side, the data received from rank 0 contains the padding of index 1"
    assert (recv[1][0][off[1]:off[2]] == SENT).all()
    # every rank receives all sendSplitLengths (L439)
    assert (allL[0] == Ls).all() and (allL[1] == Ls).all()


def brute(send, Ls, idx, bl, recv):
    R, n = Ls.shape
    for s in range(R):
        pos = 0
        off = np.concatenate([[0], np.cumsum(Ls[s])])
        for d in range(R):
            for j in range(int(bl[s, d])):
                i = int(idx[s, pos + j])
                recv[d][s][off[i]:off[i + 1]] = send[s][off[i]:off[i + 1]]
            pos += int(bl[s, d])


@pytest.mark.parametrize("R,n,seed", [(2, 4, 0), (3, 5, 1), (4, 8, 2), (8, 16, 3)])
def test_bruteforce_random_lists_with_duplicates(R, n, seed):
    rng = np.random.default_rng(seed)
    Ls = rng.integers(0, 9, (R, n)).astype(np.int64)
    J = 3
    bl = rng.integers(0, J + 1, (R, R)).astype(np.int64)
    M = R * J
    idx = np.zeros((R, M), np.int64)
    for s in range(R):
        m = int(bl[s].sum())
        idx[s, :m] = rng.integers(0, n, m)                 # non-contiguous, repeats allowed
    send = [W.np_values(int(Ls[s].sum()), "bf16", 40 + s) for s in range(R)]
    mk = lambda: [[np.full(int(Ls[s].sum()), SENT, np.uint16) for s in range(R)] for _ in range(R)]
    got, exp = mk(), mk()
    allL, st = oracle.alltoallv_dynamic(send, Ls, idx, bl, J, got, "bf16")
    brute(send, Ls, idx, bl, exp)
    assert st == 0 and all((allL[d] == Ls).all() for d in range(R))
    for d in range(R):
        for s in range(R):
            assert got[d][s].tobytes() == exp[d][s].tobytes()


def test_identity_partition_reduces_to_plain_alltoallv():
    """If rank s's splits are 'one per destination' and its list is [0,1,...,R-1] with block length 1, the
    dynamic collective moves exactly the segments of the plain AllToAllv (C = split lengths)."""
    R = 5
    rng = np.random.default_rng(7)
    C = rng.integers(0, 20, (R, R)).astype(np.int64)
    idx = np.tile(np.arange(R, dtype=np.int64), (R, 1))
    bl = np.ones((R, R), np.int64)
    send = [W.np_values(int(C[s].sum()), "f32", 60 + s) for s in range(R)]
    recvd = [[np.zeros(int(C[s].sum()), np.float32) for s in range(R)] for _ in range(R)]
    oracle.alltoallv_dynamic(send, C, idx, bl, 1, recvd, "f32")
    packed = [np.zeros(int(C[:, d].sum()), np.float32) for d in range(R)]
    RC, soff, roff, _ = oracle.alltoallv(send, C, packed, "f32")
    for d in range(R):
        for s in range(R):
            a = recvd[d][s][soff[s, d]:soff[s, d] + C[s, d]]
            b = packed[d][roff[d, s]:roff[d, s] + C[s, d]]
            assert a.tobytes() == b.tobytes()


def test_status_bits_for_bad_metadata():
    Ls = np.array([[4, -2, 3], [1, 1, 1]], np.int64)
    idx = np.array([[0, 2, 7, 0], [1, 0, 0, 0]], np.int64)
    bl = np.array([[2, 1], [9, 0]], np.int64)
    send = [np.arange(7, dtype=np.uint16), np.arange(3, dtype=np.uint16)]
    recv = [[np.full(7, SENT, np.uint16), np.full(3, SENT, np.uint16)] for _ in range(2)]
    allL, st = oracle.alltoallv_dynamic(send, Ls, idx, bl, 2, recv, "bf16")
    assert st == 1 | 2 | 4
    assert allL[0, 0].tolist() == [4, 0, 3]
    assert recv[0][0].tolist() == [0, 1, 2, 3, 4, 5, 6]            # splits 0 and 2 (negative split 1 is empty)
    assert (recv[1][0] == SENT).all()                              # index 7 out of range: skipped
    assert recv[0][1].tolist() == [0, 1, SENT]                     # block length 9 clamped to 2: indices 1, 0
