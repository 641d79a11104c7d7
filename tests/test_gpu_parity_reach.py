"""-m gpu parity, the reach the round-2 review asked for: shapes under which code paths run that the other test
modules never enter while the oracle is watching.
  * top-k dispatch / combine with more tokens than the grid has warps (148 x 16 CTAs x 4 warps = 9 472), so the
    kernels' grid-stride loops take several trips (Table 3);
  * top-k and AllToAllvDynamic above 128 ranks: dyn_build_kernel's R > 128 branch, and counts_kernel's block-sum +
    grid-barrier phase 1 with no pointer tables;
  * a fused (R <= 32) AllToAllv between a top-k prepare and its executes in plan slot 0;
  * two host threads driving the library at once (the header promises one internal mutex).
Everything is compared with the CPU oracle bit for bit over the full buffers (sentinel tails included)."""
import threading

import numpy as np
import pytest
import torch

import oracle
import paper_2510_20171_b200 as nx
from paper_2510_20171_b200 import workloads as W

pytestmark = pytest.mark.gpu
from gpu_util import ES, NP_OF, assert_a2a_matches, back, sentinel, to_dev  # noqa: E402
from test_gpu_topk import run_both  # noqa: E402

SENT = 0xA5A5


@pytest.fixture(scope="module", autouse=True)
def ctx():
    nx.ncclx_init(1024, 0)
    nx.ncclx_init_dynamic(512, 4 * 4 * 130_000)
    yield
    nx.ncclx_finalize()


# ---- top-k beyond one grid wave ------------------------------------------------------------------------------

@pytest.mark.parametrize("plan", [None, 1])
@pytest.mark.parametrize("R,T,k,width,dtype", [
    (64, 512, 4, 256, "bf16"),       # 32 768 tokens = 3.5 trips per warp, 256-bit row path
    (64, 512, 1, 256, "bf16"),       # k = 1: pos is a permutation
    (64, 512, 2, 7, "f32"),          # 28-byte rows: the scalar row path loops too
    (16, 2048, 4, 24, "f16"),        # 48-byte rows (16 B- but not 32 B-multiples)
])
def test_topk_grid_stride_loops_take_several_trips(R, T, k, width, dtype, plan):
    assert R * T > 3 * 9472
    run_both(R, T, k, width, dtype, seed=17 * R + k, plan=plan)


# ---- top-k above 128 ranks -----------------------------------------------------------------------------------

@pytest.mark.parametrize("plan", [None, 2])
@pytest.mark.parametrize("R,T,k,width", [(129, 24, 2, 16), (200, 16, 4, 32), (512, 8, 2, 16)])
def test_topk_above_128_ranks(R, T, k, width, plan):
    run_both(R, T, k, width, "bf16", seed=R, plan=plan)


# ---- AllToAllvDynamic above 128 ranks ------------------------------------------------------------------------

def dynamic_case(R, n, J, scale, seed, full_blocks=False):
    rng = np.random.default_rng(seed)
    Ls = (rng.integers(0, scale, (R, n)) * rng.integers(0, 2, (R, n))).astype(np.int64)
    Ls[:, 0] = (Ls[:, 0] // 8) * 8 + 8                         # some 16 B-aligned splits -> bulk list as well
    bl = np.full((R, R), J, np.int64) if full_blocks else rng.integers(0, J + 1, (R, R)).astype(np.int64)
    idx = np.zeros((R, R * J), np.int64)
    for s in range(R):
        m = int(bl[s].sum())
        idx[s, :m] = rng.integers(0, n, m)
    send = [W.np_values(int(Ls[s].sum()), "bf16", 900 + s) for s in range(R)]
    return send, Ls, idx, bl


def check_dynamic_slab(send_np, Ls, idx, bl, J, plan=None):
    """Like test_gpu_dynamic.check, but the R*R receive arrays are rows of ONE slab (R = 512 has 262 144 of them)."""
    R, n = Ls.shape
    tot = np.maximum(Ls, 0).sum(axis=1)
    cap = (int(tot.max()) + 15) // 8 * 8
    eslab = np.full((R * R, cap), SENT, np.uint16)
    exp = [[eslab[d * R + s][: int(tot[s])] for s in range(R)] for d in range(R)]
    eall, est = oracle.alltoallv_dynamic(send_np, Ls, idx, bl, J, exp, "bf16")

    send = [torch.from_numpy(a.view(np.int16)).cuda() if a.size else torch.zeros(8, dtype=torch.int16, device="cuda") for a in send_np]
    slab = torch.full((R * R, cap), -23131, dtype=torch.int16, device="cuda")
    rt = torch.from_numpy(slab.data_ptr() + np.arange(R * R, dtype=np.int64) * (cap * 2)).cuda()
    st = nx.device_ptr_table(send)
    Ld, Id, Bd = (torch.from_numpy(np.ascontiguousarray(x, dtype=np.int64)).cuda() for x in (Ls, idx, bl))
    allL = torch.full((R, R, n), -1, dtype=torch.int64, device="cuda")
    if plan is None:
        nx.ncclx_alltoallv_dynamic_dev(st, Ld, n, Id, idx.shape[1], Bd, J, rt, allL, R, "bf16")
    else:
        nx.ncclx_alltoallv_dynamic_prepare_dev(plan, st, Ld, n, Id, idx.shape[1], Bd, J, rt, allL, R, "bf16")
        nx.ncclx_alltoallv_execute_dev(plan)
    status = nx.ncclx_device_status()
    torch.cuda.synchronize()
    assert status == est
    assert (allL.cpu().numpy() == eall).all()
    got = slab.cpu().numpy().view(np.uint16)
    bad = np.nonzero((got != eslab).any(axis=1))[0]
    assert bad.size == 0, f"recvbuffs[d][s] differ from the oracle for (d, s) = {[(int(q) // R, int(q) % R) for q in bad[:8]]}"
    assert int((eslab != SENT).sum()) > 0


@pytest.mark.parametrize("R,n,J,scale,full,plan", [(129, 24, 3, 300, False, None), (160, 16, 2, 200, True, 3),
                                                   (200, 32, 3, 120, False, None), (512, 6, 2, 40, False, None),
                                                   (512, 4, 1, 64, True, 1)])
def test_dynamic_above_128_ranks(R, n, J, scale, full, plan):
    send, Ls, idx, bl = dynamic_case(R, n, J, scale, seed=R + J, full_blocks=full)
    check_dynamic_slab(send, Ls, idx, bl, J, plan=plan)


# ---- a fused AllToAllv between a top-k prepare and its executes in slot 0 (round-2 advisor finding) ----------

def test_fused_alltoallv_leaves_a_topk_plan_in_slot_0_intact():
    R, T, k, width, dtype = 8, 96, 4, 64, "bf16"
    pos, C = W.topk_routing(R, T, k, 2 * R, 77)
    X = [W.np_values(T * width, dtype, 40 + s) for s in range(R)]
    slack = 8
    erecv = [np.full((int(C[:, d].sum()) + slack) * width, SENT, np.uint16) for d in range(R)]
    eRC, est = oracle.moe_dispatch_topk(X, pos, C, erecv, width, dtype)
    dX = [to_dev(x) for x in X]
    drecv = [sentinel((int(C[:, d].sum()) + slack) * width * 2) for d in range(R)]
    dpos, dC = torch.from_numpy(pos).cuda(), torch.from_numpy(C).cuda()
    dRC = torch.zeros_like(dC)
    nx.ncclx_moe_topk_prepare_dev(0, dC, dRC, R)

    # an unrelated small AllToAllv (one fused kernel, different R and counts) while slot 0 holds the top-k plan
    C2 = (np.random.default_rng(3).integers(0, 90, (5, 5)) * 7).astype(np.int64)
    send2 = [W.np_values(int(C2[s].sum()), "bf16", 60 + s) for s in range(5)]
    n0 = nx.ncclx_launch_count()
    assert_a2a_matches(send2, C2, "bf16")
    assert nx.ncclx_launch_count() - n0 == 1, "R = 5 must have taken the single-launch path"

    nx.ncclx_moe_dispatch_topk_execute_dev(0, nx.device_ptr_table(dX), dpos, nx.device_ptr_table(drecv), T, k, width, dtype)
    Y = [np.roll(erecv[d][: int(C[:, d].sum()) * width], 5 * d + 1) for d in range(R)]
    dY = [to_dev(y) for y in Y]
    eZ, est2 = oracle.moe_combine_topk_sum(Y, pos, C, width, dtype)
    dZ = [sentinel(T * width * 2) for _ in range(R)]
    nx.ncclx_moe_combine_topk_sum_execute_dev(0, nx.device_ptr_table(dY), dpos, nx.device_ptr_table(dZ), T, k, width, dtype)
    assert nx.ncclx_device_status() == (est | est2) == 0
    torch.cuda.synchronize()
    assert (dRC.cpu().numpy() == eRC).all()
    for d in range(R):
        assert back(drecv[d], dtype).tobytes() == erecv[d].tobytes(), f"dispatch recv[{d}] after the interleaved call"
    for s in range(R):
        assert back(dZ[s], dtype).tobytes() == eZ[s].tobytes(), f"combine out[{s}] after the interleaved call"


# ---- two host threads (include/ncclx_b200.h: "entry points may be called from several host threads") ---------

def test_two_host_threads_share_the_library():
    """One thread enqueues reductions, the other parameter / status traffic plus launch counting, all on ONE stream
    (the workspace rule): nothing may crash, deadlock or lose a launch, and every reduction must match the oracle."""
    R, n, rounds = 4, 30_000, 40
    xs_np = [W.np_values(n, "bf16", 800 + r) for r in range(R)]
    xs = [to_dev(a) for a in xs_np]
    outs = [[sentinel(n * 2) for _ in range(R)] for _ in range(rounds)]
    xt = nx.device_ptr_table(xs)
    ots = [nx.device_ptr_table(o) for o in outs]
    stream = torch.cuda.current_stream()
    torch.cuda.synchronize()
    n0 = nx.ncclx_launch_count()
    errors = []

    def reducer():
        try:
            for i in range(rounds):
                nx.ncclx_allreduce_sum(xt, ots[i], n, R, "bf16", stream)
        except Exception as e:  # noqa: BLE001
            errors.append(e)

    def meddler():
        try:
            for i in range(rounds * 5):
                nx.ncclx_set_param(nx.PARAM_COPY_KMAX, 1 + i % 8)
                assert 1 <= nx.ncclx_get_param(nx.PARAM_COPY_KMAX) <= 8
                nx.ncclx_launch_count()
        except Exception as e:  # noqa: BLE001
            errors.append(e)

    th = [threading.Thread(target=reducer), threading.Thread(target=meddler)]
    for t in th:
        t.start()
    for t in th:
        t.join(60)
    assert not any(t.is_alive() for t in th), "a library call did not return"
    nx.ncclx_set_param(nx.PARAM_COPY_KMAX, 6)
    torch.cuda.synchronize()
    assert not errors, errors
    assert nx.ncclx_launch_count() - n0 == rounds
    exp = oracle.allreduce_sum(xs_np, "bf16", nthreads=4)
    for i in range(rounds):
        for r in range(R):
            assert back(outs[i][r], "bf16").tobytes() == exp[r].tobytes(), (i, r)
