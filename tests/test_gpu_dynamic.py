"""-m gpu parity: ncclx_alltoallv_dynamic_dev (the paper's full AllToAllvDynamic interface, PAPER.md
L429-439) vs the CPU oracle, byte for byte over every recvbuffs[d][s] incl. the reserved padding."""
import json
import os

import numpy as np
import pytest
import torch

import oracle
import paper_2510_20171_b200 as nx
from paper_2510_20171_b200 import workloads as W

pytestmark = pytest.mark.gpu
SENT = 0xA5A5


@pytest.fixture(scope="module", autouse=True)
def ctx():
    nx.ncclx_init(128, 0)
    nx.ncclx_init_dynamic(512, 4 * 4 * 130_000)
    yield
    nx.ncclx_finalize()


def run_gpu(send_np, Ls, idx, bl, J, dtype="bf16", plan=None):
    R, n = Ls.shape
    tot = np.maximum(Ls, 0).sum(axis=1)
    send = [torch.from_numpy(a.view(np.int16)).cuda() if a.size else torch.zeros(8, dtype=torch.int16, device="cuda") for a in send_np]
    recv = [[torch.full((max(int(tot[s]), 8),), -23131, dtype=torch.int16, device="cuda") for s in range(R)] for _ in range(R)]
    st = nx.device_ptr_table(send)
    rt = nx.device_ptr_table([recv[d][s] for d in range(R) for s in range(R)])
    Ld, Id, Bd = (torch.from_numpy(np.ascontiguousarray(x, dtype=np.int64)).cuda() for x in (Ls, idx, bl))
    allL = torch.full((R, R, n), -1, dtype=torch.int64, device="cuda")
    if plan is None:
        nx.ncclx_alltoallv_dynamic_dev(st, Ld, n, Id, idx.shape[1], Bd, J, rt, allL, R, dtype)
    else:                                                   # split-phase form: metadata into a plan slot, then the payload
        nx.ncclx_alltoallv_dynamic_prepare_dev(plan, st, Ld, n, Id, idx.shape[1], Bd, J, rt, allL, R, dtype)
        nx.ncclx_alltoallv_execute_dev(plan)
    status = nx.ncclx_device_status()
    torch.cuda.synchronize()
    got = [[recv[d][s].cpu().numpy().view(np.uint16)[: int(tot[s])] for s in range(R)] for d in range(R)]
    return got, allL.cpu().numpy(), status


def run_oracle(send_np, Ls, idx, bl, J):
    R, n = Ls.shape
    tot = np.maximum(Ls, 0).sum(axis=1)
    exp = [[np.full(int(tot[s]), SENT, np.uint16) for s in range(R)] for _ in range(R)]
    allL, st = oracle.alltoallv_dynamic(send_np, Ls, idx, bl, J, exp, "bf16")
    return exp, allL, st


def check(send_np, Ls, idx, bl, J, plan=None):
    got, allL, st = run_gpu(send_np, Ls, idx, bl, J, plan=plan)
    exp, eall, est = run_oracle(send_np, Ls, idx, bl, J)
    assert st == est and (allL == eall).all()
    R = Ls.shape[0]
    for d in range(R):
        for s in range(R):
            assert got[d][s].tobytes() == exp[d][s].tobytes(), (d, s)


def test_fig17_worked_example(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "fig17_alltoallvdynamic.json")))
    L0 = np.array(g["sendSplitLengths"], np.int64)
    Ls = np.stack([L0, np.zeros(4, np.int64)])
    idx = np.zeros((2, 8), np.int64); idx[0, :5] = g["sendIndices"]
    bl = np.array([g["sendIndicesBlockLens"], [0, 0]], np.int64)
    send = [np.arange(1, int(L0.sum()) + 1, dtype=np.uint16), np.zeros(0, np.uint16)]
    got, allL, st = run_gpu(send, Ls, idx, bl, 3)
    off = np.concatenate([[0], np.cumsum(L0)])
    for d, splits in ((0, g["to_rank0_splits"]), (1, g["to_rank1_splits"])):
        exp = np.full(int(L0.sum()), SENT, np.uint16)
        for i in splits:
            exp[off[i]:off[i + 1]] = send[0][off[i]:off[i + 1]]
        assert (got[d][0] == exp).all()
    assert st == 0 and (allL[0] == Ls).all() and (allL[1] == Ls).all()


@pytest.mark.parametrize("R,n,J,scale,seed", [(2, 4, 2, 9, 0), (4, 8, 3, 5000, 1), (8, 16, 3, 40000, 2), (16, 64, 4, 3000, 3),
                                              (64, 128, 3, 2000, 4), (100, 40, 3, 300, 5), (40, 300, 9, 200, 6),
                                              (64, 480, 2, 100, 7)])
def test_random_lists_with_duplicates(R, n, J, scale, seed):
    rng = np.random.default_rng(seed)
    Ls = (rng.integers(0, scale, (R, n)) * rng.integers(0, 2, (R, n))).astype(np.int64)
    Ls[:, 0] = (Ls[:, 0] // 8) * 8 + 8                         # some 16B-aligned splits -> bulk path
    bl = rng.integers(0, J + 1, (R, R)).astype(np.int64)
    idx = np.zeros((R, R * J), np.int64)
    for s in range(R):
        m = int(bl[s].sum())
        idx[s, :m] = rng.integers(0, n, m)
    send = [W.np_values(int(Ls[s].sum()), "bf16", 90 + s) for s in range(R)]
    check(send, Ls, idx, bl, J)


@pytest.mark.parametrize("R,n,J,scale", [(32, 64, 128, 40), (64, 64, 64, 24), (128, 32, 32, 16), (17, 48, 240, 24),
                                         (4, 64, 130_000, 6)])
def test_long_columns_full_blocks_search_without_shared_index(R, n, J, scale):
    """Columns of R*J slots whose coarse index does not fit the copy kernel's 16 KB of shared memory (R*ceil(R*J/32) >
    2048), every block full: claims locate their segment with the 128-ary search in L2.  R*J in 3969..4096 and around
    520 000 are the lengths at which the search's last round leaves exactly 32 candidates (round-1 ADVICE: the
    window then has to start at the first candidate's predecessor and still hold all of them).  The last shape has
    more slots per column than DYN_SMEM_SLOTS, so the metadata kernel stages its slots in the table itself."""
    rng = np.random.default_rng(R * 1000 + J)
    Ls = rng.integers(1, scale, (R, n)).astype(np.int64)
    Ls[:, :4] = (Ls[:, :4] // 8 + 1) * 8 * 70                  # a few 16B-aligned kilobyte splits -> bulk list too
    bl = np.full((R, R), J, np.int64)
    idx = rng.integers(0, n, (R, R * J)).astype(np.int64)
    send = [W.np_values(int(Ls[s].sum()), "bf16", 400 + s) for s in range(R)]
    check(send, Ls, idx, bl, J)


@pytest.mark.parametrize("plan", [1, 3])
def test_split_phase_form_in_plan_slots(plan):
    R, n, J = 16, 64, 4
    rng = np.random.default_rng(plan)
    Ls = (rng.integers(0, 3000, (R, n)) * rng.integers(0, 2, (R, n))).astype(np.int64)
    bl = rng.integers(0, J + 1, (R, R)).astype(np.int64)
    idx = np.zeros((R, R * J), np.int64)
    for s in range(R):
        m = int(bl[s].sum())
        idx[s, :m] = rng.integers(0, n, m)
    send = [W.np_values(int(Ls[s].sum()), "bf16", 500 + s) for s in range(R)]
    check(send, Ls, idx, bl, J, plan=plan)


def test_double_buffered_dynamic_pair_in_a_graph():
    """Two AllToAllvDynamic calls (two MoE layers' dispatches) in one graph: the second call's metadata kernel runs on a
    forked stream beside the first call's payload, each in its own plan slot (PAPER.md L483 double buffering)."""
    R, n, J = 8, 32, 3
    rng = np.random.default_rng(11)

    def problem(seed):
        Ls = (rng.integers(0, 4000, (R, n)) * 8).astype(np.int64)
        bl = rng.integers(0, J + 1, (R, R)).astype(np.int64)
        idx = np.zeros((R, R * J), np.int64)
        for s in range(R):
            m = int(bl[s].sum()); idx[s, :m] = rng.integers(0, n, m)
        send_np = [W.np_values(int(Ls[s].sum()), "bf16", seed + s) for s in range(R)]
        tot = Ls.sum(axis=1)
        send = [torch.from_numpy(a.view(np.int16)).cuda() for a in send_np]
        recv = [[torch.full((int(tot[s]),), -23131, dtype=torch.int16, device="cuda") for s in range(R)] for _ in range(R)]
        dev = dict(st=nx.device_ptr_table(send), rt=nx.device_ptr_table([recv[d][s] for d in range(R) for s in range(R)]),
                   L=torch.from_numpy(Ls).cuda(), I=torch.from_numpy(idx).cuda(), B=torch.from_numpy(bl).cuda(),
                   all=torch.full((R, R, n), -1, dtype=torch.int64, device="cuda"), send=send)
        return send_np, Ls, idx, bl, recv, dev
    P = [problem(600), problem(700)]
    side = torch.cuda.Stream()

    def enqueue():
        main = torch.cuda.current_stream()
        a, b = P[0][5], P[1][5]
        nx.ncclx_alltoallv_dynamic_prepare_dev(0, a["st"], a["L"], n, a["I"], R * J, a["B"], J, a["rt"], a["all"], R, "bf16")
        side.wait_stream(main)
        with torch.cuda.stream(side):
            nx.ncclx_alltoallv_dynamic_prepare_dev(1, b["st"], b["L"], n, b["I"], R * J, b["B"], J, b["rt"], b["all"], R, "bf16")
        nx.ncclx_alltoallv_execute_dev(0)
        main.wait_stream(side)
        nx.ncclx_alltoallv_execute_dev(1)
    warm = torch.cuda.Stream(); warm.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(warm):
        enqueue()
    torch.cuda.current_stream().wait_stream(warm)
    torch.cuda.synchronize()
    for p in P:
        for row in p[4]:
            for r in row:
                r.fill_(-23131)
        p[5]["all"].fill_(-1)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        enqueue()
    g.replay(); torch.cuda.synchronize()
    for send_np, Ls, idx, bl, recv, dev in P:
        exp, eall, est = run_oracle(send_np, Ls, idx, bl, J)
        assert (dev["all"].cpu().numpy() == eall).all()
        for d in range(R):
            for s in range(R):
                assert recv[d][s].cpu().numpy().view(np.uint16).tobytes() == exp[d][s].tobytes(), (d, s)
    assert nx.ncclx_device_status() == 0


def test_moe_shaped_expert_splits_aligned_rows():
    """Config-3 shape at 1/64 scale: 128 experts, 2 per rank + 1 redundant copy of the hottest expert on
    rank R-1 (duplicated experts), rows of 5120 bf16 (16B-aligned -> all bulk)."""
    R, E, width = 64, 128, 5120
    rng = np.random.default_rng(2)
    p = (np.arange(E) + 1.0) ** -1.1; p /= p.sum()
    per_expert = np.stack([rng.multinomial(256, p) for _ in range(R)])
    Ls = (per_expert * width).astype(np.int64)
    J = 3
    bl = np.full((R, R), 2, np.int64); bl[:, R - 1] = 3
    idx = np.zeros((R, 2 * R + 1), np.int64)
    for s in range(R):
        lst = []
        for d in range(R):
            lst += [2 * d, 2 * d + 1] + ([0] if d == R - 1 else [])
        idx[s, :len(lst)] = lst
    send = [W.np_values(int(Ls[s].sum()), "bf16", 200 + s) for s in range(R)]
    check(send, Ls, idx, bl, J)


def test_bad_metadata_status_bits_and_capacity_errors():
    Ls = np.array([[4, -2, 3], [1, 1, 1]], np.int64)
    idx = np.array([[0, 2, 7, 0], [1, 0, 0, 0]], np.int64)
    bl = np.array([[2, 1], [9, 0]], np.int64)
    send = [np.arange(7, dtype=np.uint16), np.arange(3, dtype=np.uint16)]
    got, allL, st = run_gpu(send, Ls, idx, bl, 2)
    exp, eall, est = run_oracle(send, Ls, idx, bl, 2)
    assert st == est == 7 and (allL == eall).all()
    assert all(got[d][s].tobytes() == exp[d][s].tobytes() for d in range(2) for s in range(2))
    t = torch.zeros(16, dtype=torch.int64, device="cuda")
    n0 = nx.ncclx_launch_count()
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_alltoallv_dynamic_dev(t, t, 9999, t, 4, t, 2, t, t, 2, "bf16")     # nsplits > max_splits
    assert e.value.code == 3
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_alltoallv_dynamic_dev(t, t, 4, t, 4, t, 1 << 24, t, t, 2, "bf16")  # work list larger than ncclx_init_dynamic's
    assert e.value.code == 3
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_alltoallv_dynamic_prepare_dev(7, t, t, 4, t, 4, t, 2, t, t, 2, "bf16")   # no such plan slot
    assert e.value.code == 1
    assert nx.ncclx_launch_count() == n0, "an argument error must not enqueue anything"


def test_graph_replay_follows_device_metadata():
    R, n, J = 4, 8, 2
    rng = np.random.default_rng(5)
    cap = 4096
    send_np = [W.np_values(cap * n, "bf16", 300 + s) for s in range(R)]
    send = [torch.from_numpy(a.view(np.int16)).cuda() for a in send_np]
    recv = [[torch.empty(cap * n, dtype=torch.int16, device="cuda") for s in range(R)] for _ in range(R)]
    st = nx.device_ptr_table(send); rt = nx.device_ptr_table([recv[d][s] for d in range(R) for s in range(R)])
    Ld = torch.zeros((R, n), dtype=torch.int64, device="cuda")
    Id = torch.zeros((R, R * J), dtype=torch.int64, device="cuda")
    Bd = torch.zeros((R, R), dtype=torch.int64, device="cuda")
    allL = torch.zeros((R, R, n), dtype=torch.int64, device="cuda")
    call = lambda: nx.ncclx_alltoallv_dynamic_dev(st, Ld, n, Id, R * J, Bd, J, rt, allL, R, "bf16")
    side = torch.cuda.Stream(); side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        call()
    torch.cuda.current_stream().wait_stream(side)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        call()
    for trial in range(3):
        Ls = (rng.integers(0, cap // 8, (R, n)) * 8).astype(np.int64)
        bl = rng.integers(0, J + 1, (R, R)).astype(np.int64)
        idx = np.zeros((R, R * J), np.int64)
        for s in range(R):
            m = int(bl[s].sum()); idx[s, :m] = rng.integers(0, n, m)
        for row in recv:
            for r in row:
                r.fill_(-23131)
        Ld.copy_(torch.from_numpy(Ls)); Id.copy_(torch.from_numpy(idx)); Bd.copy_(torch.from_numpy(bl))
        g.replay(); torch.cuda.synchronize()
        exp = [[np.full(cap * n, SENT, np.uint16) for s in range(R)] for _ in range(R)]
        eall, est = oracle.alltoallv_dynamic(send_np, Ls, idx, bl, J, exp, "bf16")
        assert (allL.cpu().numpy() == eall).all()
        for d in range(R):
            for s in range(R):
                assert recv[d][s].cpu().numpy().view(np.uint16).tobytes() == exp[d][s].tobytes()
