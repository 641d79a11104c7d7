"""Pins for the top-k dispatch/combine oracle (NEXT-3): k = 1 reduces to the plain AllToAllv of the
permuted rows and its inverse; with identity experts combine(dispatch(X)) = k * X exactly for k in
{1,2,4} (power-of-two scaling is exact); brute force on tiny inputs; the hand-derived order vector."""
import numpy as np
import pytest

import oracle
from paper_2510_20171_b200 import workloads as W


def setup(R, T, k, width, dtype, seed, experts=None):
    pos, C = W.topk_routing(R, T, k, experts or 2 * R, seed)
    X = [W.np_values(T * width, dtype, 500 + s) for s in range(R)]
    recv = [np.zeros(int(C[:, d].sum()) * width, X[0].dtype) for d in range(R)]
    return pos, C, X, recv


@pytest.mark.parametrize("R,T,width", [(2, 5, 3), (4, 16, 8), (8, 33, 16)])
def test_k1_is_plain_alltoallv_of_permuted_rows_and_roundtrip(R, T, width):
    pos, C, X, recv = setup(R, T, 1, width, "bf16", 1)
    RC, st = oracle.moe_dispatch_topk(X, pos, C, recv, width, "bf16")
    assert st == 0 and (RC == C.T).all()
    V = []
    for s in range(R):
        v = np.empty((T, width), np.uint16)
        v[pos[s, :, 0]] = X[s].reshape(T, width)              # the materialised sorted send buffer
        V.append(v.reshape(-1))
    exp = [np.zeros_like(r) for r in recv]
    oracle.alltoallv(V, C * width, exp, "bf16")
    assert all(a.tobytes() == b.tobytes() for a, b in zip(recv, exp))
    Z, st = oracle.moe_combine_topk_sum(recv, pos, C, width, "bf16")
    assert st == 0 and all(z.tobytes() == x.tobytes() for z, x in zip(Z, X))


@pytest.mark.parametrize("k", [1, 2, 4])
@pytest.mark.parametrize("dtype", ["bf16", "f32", "f16"])
def test_identity_experts_give_k_times_x_exactly(k, dtype):
    R, T, width = 4, 40, 8
    pos, C, X, recv = setup(R, T, k, width, dtype, 2, experts=8)
    oracle.moe_dispatch_topk(X, pos, C, recv, width, dtype)
    Z, st = oracle.moe_combine_topk_sum(recv, pos, C, width, dtype)
    f = {"bf16": lambda a: (a.astype(np.uint32) << 16).view(np.float32), "f32": lambda a: a,
         "f16": lambda a: a.view(np.float16).astype(np.float32)}[dtype]
    for s in range(R):
        assert (f(Z[s]) == np.float32(k) * f(X[s])).all()      # N(0,1) values: no overflow / subnormal


def test_bruteforce_and_conservation():
    R, T, k, width = 3, 7, 2, 4
    pos, C, X, recv = setup(R, T, k, width, "f32", 3, experts=6)
    oracle.moe_dispatch_topk(X, pos, C, recv, width, "f32")
    soff = np.cumsum(C, axis=1) - C
    roff = (np.cumsum(C, axis=0) - C).T
    for s in range(R):
        assert sorted(pos[s].reshape(-1).tolist()) == list(range(T * k))          # a permutation
        for t in range(T):
            for j in range(k):
                p = int(pos[s, t, j])
                d = int(np.searchsorted(np.cumsum(C[s]), p, side="right"))
                row = int(roff[d, s] + p - soff[s, d])
                assert (recv[d].reshape(-1, width)[row] == X[s].reshape(T, width)[t]).all()
    assert sum(r.size for r in recv) == k * sum(x.size for x in X)


def test_order_vector_and_bad_positions():
    # one token, k = 4 copies whose returned values are [1, 2^-8, 2^-24, 2^-24] in router order (bf16 golden vector)
    R, T, k, width = 1, 1, 4, 1
    C = np.array([[4]], np.int64)
    pos = np.array([[[2, 0, 3, 1]]], np.int32)
    Y = [np.zeros(4, np.uint16)]
    for j, v in enumerate([0x3F80, 0x3B80, 0x3380, 0x3380]):
        Y[0][pos[0, 0, j]] = v
    Z, st = oracle.moe_combine_topk_sum(Y, pos, C, width, "bf16")
    assert st == 0 and int(Z[0][0]) == 0x3F80
    pos_rev = pos[:, :, ::-1].copy()
    Z, _ = oracle.moe_combine_topk_sum(Y, pos_rev, C, width, "bf16")
    assert int(Z[0][0]) == 0x3F81                                                   # order matters: j order is the contract
    bad = np.array([[[2, 9, -1, 1]]], np.int32)
    Z, st = oracle.moe_combine_topk_sum(Y, bad, C, width, "bf16")
    assert st == 2 and int(Z[0][0]) == oracle.allreduce_sum([Y[0][2:3], Y[0][1:2]], "bf16")[0][0]
    none = np.array([[[7, 9, -1, 5]]], np.int32)
    Z, st = oracle.moe_combine_topk_sum(Y, none, C, width, "bf16")
    assert st == 2 and int(Z[0][0]) == 0
