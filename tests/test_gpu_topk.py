"""-m gpu parity: top-k dispatch (duplication on the way) and combine (inverse AllToAllv fused with the
fixed-order fp32 sum) vs the CPU oracle, bit for bit over the full buffers."""
import numpy as np
import pytest
import torch

import oracle
import paper_2510_20171_b200 as nx
from paper_2510_20171_b200 import workloads as W

pytestmark = pytest.mark.gpu
from gpu_util import ES, NP_OF, back, sentinel, to_dev  # noqa: E402


@pytest.fixture(scope="module", autouse=True)
def ctx():
    nx.ncclx_init(128, 0)
    yield
    nx.ncclx_finalize()


def run_both(R, T, k, width, dtype, seed, experts=None, mis=0, scramble_y=True, plan=None):
    pos, C = W.topk_routing(R, T, k, experts or 2 * R, seed)
    X = [W.np_values(T * width, dtype, 700 + s) for s in range(R)]
    slack = 8
    # oracle
    erecv = [np.frombuffer(bytes([0xA5]) * ((int(C[:, d].sum()) + slack) * width * ES[dtype]), NP_OF[dtype]).copy() for d in range(R)]
    eRC, est = oracle.moe_dispatch_topk(X, pos, C, erecv, width, dtype)
    # gpu dispatch
    dX = [to_dev(x, mis) for x in X]
    drecv = [sentinel((int(C[:, d].sum()) + slack) * width * ES[dtype], mis) for d in range(R)]
    dpos = torch.from_numpy(pos).cuda()
    dC = torch.from_numpy(C).cuda()
    dRC = torch.zeros_like(dC)
    if plan is None:
        nx.ncclx_moe_dispatch_topk_dev(nx.device_ptr_table(dX), dpos, dC, nx.device_ptr_table(drecv), dRC, R, T, k, width, dtype)
    else:                           # plan-slot form: ONE metadata phase serves the dispatch and (below) the combine
        n0 = nx.ncclx_launch_count()
        nx.ncclx_moe_topk_prepare_dev(plan, dC, dRC, R)
        nx.ncclx_moe_dispatch_topk_execute_dev(plan, nx.device_ptr_table(dX), dpos, nx.device_ptr_table(drecv), T, k, width, dtype)
        assert nx.ncclx_launch_count() - n0 == 2
    st = nx.ncclx_device_status()
    torch.cuda.synchronize()
    assert st == est and (dRC.cpu().numpy() == eRC).all()
    for d in range(R):
        assert back(drecv[d], dtype).tobytes() == erecv[d].tobytes(), f"dispatch recv[{d}]"
    # "experts": perturb the received rows so the k copies of a token differ (then order matters)
    Y = []
    for d in range(R):
        y = erecv[d][: int(C[:, d].sum()) * width].copy()
        if scramble_y:
            y = np.roll(y, 3 * d + 1)
        Y.append(y)
    dY = [to_dev(y, mis) for y in Y]
    eZ, est2 = oracle.moe_combine_topk_sum(Y, pos, C, width, dtype)
    dZ = [sentinel(T * width * ES[dtype], mis) for _ in range(R)]
    if plan is None:
        nx.ncclx_moe_combine_topk_sum_dev(nx.device_ptr_table(dY), dpos, dC, nx.device_ptr_table(dZ), R, T, k, width, dtype)
    else:
        n0 = nx.ncclx_launch_count()
        nx.ncclx_moe_combine_topk_sum_execute_dev(plan, nx.device_ptr_table(dY), dpos, nx.device_ptr_table(dZ), T, k, width, dtype)
        assert nx.ncclx_launch_count() - n0 == 1           # the combine reuses the dispatch's offsets: no metadata kernel
    st2 = nx.ncclx_device_status()
    torch.cuda.synchronize()
    assert st2 == est2
    for s in range(R):
        assert back(dZ[s], dtype).tobytes() == eZ[s].tobytes(), f"combine out[{s}]"
    return X, eZ


@pytest.mark.parametrize("dtype", ["bf16", "f32", "f16"])
@pytest.mark.parametrize("R,T,k,width", [(2, 5, 1, 16), (4, 33, 2, 64), (8, 100, 4, 128), (16, 64, 8, 80), (64, 32, 4, 512)])
def test_dispatch_and_combine_match_oracle(dtype, R, T, k, width):
    run_both(R, T, k, width, dtype, seed=R + k)


@pytest.mark.parametrize("plan", [0, 2])
@pytest.mark.parametrize("R,T,k,width,dtype", [(8, 100, 4, 128, "bf16"), (64, 128, 4, 5120, "bf16"), (32, 256, 1, 5120, "bf16"),
                                               (16, 64, 8, 80, "f32")])
def test_plan_slot_form_matches_oracle(plan, R, T, k, width, dtype):
    """ncclx_moe_topk_prepare_dev + the two execute calls (PAPER.md L483 double buffering for the k > 1 flow), incl.
    Table 3's decode shapes (k in {1, 4}, 128 / 256 tokens per rank, hidden 5120)."""
    run_both(R, T, k, width, dtype, seed=3 * R + k, plan=plan)


def test_plan_slot_kinds_are_checked():
    R = 4
    C = torch.from_numpy(np.full((R, R), 3, np.int64)).cuda()
    RC = torch.zeros_like(C)
    t = torch.zeros(64, dtype=torch.int64, device="cuda")
    nx.ncclx_moe_topk_prepare_dev(1, C, RC, R)
    n0 = nx.ncclx_launch_count()
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_alltoallv_execute_dev(1)                       # slot 1 holds a top-k plan, not a work list
    assert e.value.code == 1
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_moe_dispatch_topk_execute_dev(3, t, t, t, 4, 2, 16, "bf16")     # slot 3 was never prepared
    assert e.value.code == 1
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_moe_dispatch_topk_execute_dev(1, t, t, t, 4, 0, 16, "bf16")     # k = 0
    assert e.value.code == 1
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_moe_topk_prepare_dev(1, C, C, R)                                # aliased count matrices
    assert e.value.code == 1
    assert nx.ncclx_launch_count() == n0, "an argument error must not enqueue anything"
    torch.cuda.synchronize()


@pytest.mark.parametrize("mis,width", [(2, 16), (16, 24), (0, 7), (6, 33)])
def test_unaligned_rows_and_bases(mis, width):
    run_both(4, 50, 2, width, "bf16", seed=9, mis=mis)


def test_identity_experts_k_times_x_and_hidden_5120():
    X, Z = run_both(8, 64, 4, 5120, "bf16", seed=5, scramble_y=False)
    for s in range(8):
        xf = (X[s].astype(np.uint32) << 16).view(np.float32)
        zf = (Z[s].astype(np.uint32) << 16).view(np.float32)
        assert (zf == np.float32(4) * xf).all()


def test_bad_positions_and_errors():
    R, T, k, width = 2, 4, 2, 16
    pos, C = W.topk_routing(R, T, k, 4, 1)
    pos = pos.copy(); pos[0, 1, 0] = 999; pos[1, 2, 1] = -3
    Y = [W.np_values(int(C[:, d].sum()) * width, "bf16", 30 + d) for d in range(R)]
    eZ, est = oracle.moe_combine_topk_sum(Y, pos, C, width, "bf16")
    dZ = [sentinel(T * width * 2) for _ in range(R)]
    dY = [to_dev(y) for y in Y]
    nx.ncclx_moe_combine_topk_sum_dev(nx.device_ptr_table(dY), torch.from_numpy(pos).cuda(), torch.from_numpy(C).cuda(),
                                      nx.device_ptr_table(dZ), R, T, k, width, "bf16")
    assert nx.ncclx_device_status() == est == 2
    for s in range(R):
        assert back(dZ[s], "bf16").tobytes() == eZ[s].tobytes()
    t = torch.zeros(8, dtype=torch.int64, device="cuda")
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_moe_combine_topk_sum_dev(t, t, t, t, 2, 4, 33, 16, "bf16")
    assert e.value.code == 1
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_moe_combine_topk_sum_dev(t, t, t, t, 2, 4, 2, 16, "u8")
    assert e.value.code == 2
