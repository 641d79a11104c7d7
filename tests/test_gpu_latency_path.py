"""-m gpu parity for SURVEY.md 8(f) NEXT-4 (section 6.2): the single-launch small-R path of
ncclx_alltoallv_dev, and the split-phase prepare/execute form with plan slots (double buffering).  Neither
adds arithmetic: the expected values are the AllToAllv oracle's, byte for byte over the full capacity."""
import numpy as np
import pytest
import torch

import paper_2510_20171_b200 as nx
from paper_2510_20171_b200 import workloads as W

pytestmark = pytest.mark.gpu

from gpu_util import ES, NP_OF, SENT8, assert_a2a_matches, back, oracle_a2a, run_a2a, sentinel, to_dev  # noqa: E402


@pytest.fixture(scope="module", autouse=True)
def ctx():
    assert torch.cuda.is_available()
    nx.ncclx_init(128, 0)
    yield
    nx.ncclx_finalize()


@pytest.fixture(autouse=True)
def default_params():
    yield
    nx.ncclx_set_param(nx.PARAM_FUSED_MAX_RANKS, 32)
    nx.ncclx_set_param(nx.PARAM_BULK_MIN_BYTES, 1024)
    nx.ncclx_set_param(nx.PARAM_BULK_TILE_SHIFT, 15)


def make_send(C, dtype, seed=0):
    C = np.maximum(np.asarray(C), 0)
    return [W.np_values(int(C[s].sum()), dtype, seed + s) for s in range(C.shape[0])]


def launches_of(fn):
    n0 = nx.ncclx_launch_count()
    fn()
    return nx.ncclx_launch_count() - n0


# ---- single-launch path ------------------------------------------------------------------------------

def test_small_R_call_is_one_kernel_and_large_R_is_two():
    C = W.a2a_config(1).counts
    send = make_send(C, "bf16", 1)
    # run_a2a makes exactly one ncclx_alltoallv_dev call
    assert launches_of(lambda: run_a2a(send, C, "bf16")) == 1
    nx.ncclx_set_param(nx.PARAM_FUSED_MAX_RANKS, 0)
    assert launches_of(lambda: run_a2a(send, C, "bf16")) == 2
    nx.ncclx_set_param(nx.PARAM_FUSED_MAX_RANKS, 32)
    R = 33
    C = np.full((R, R), 64)
    assert launches_of(lambda: run_a2a(make_send(C, "bf16", 2), C, "bf16")) == 2


@pytest.mark.parametrize("fused", [32, 0])
@pytest.mark.parametrize("R", [1, 2, 3, 4, 7, 16, 31, 32])
@pytest.mark.parametrize("dtype", ["u8", "bf16"])
def test_fused_and_two_kernel_paths_match_the_oracle(R, dtype, fused):
    """Element-granular random counts (arbitrary alignment, zero rows / columns, negative entries)."""
    nx.ncclx_set_param(nx.PARAM_FUSED_MAX_RANKS, fused)
    rng = np.random.default_rng(100 * R + ES[dtype])
    C = rng.integers(0, max(2, 2_000_000 // (R * R)), (R, R))
    C[rng.random((R, R)) < 0.3] = 0
    if R > 2:
        C[R // 2, :] = 0
        C[:, R // 3] = 0
        C[0, R - 1] = -3
    assert_a2a_matches(make_send(C, dtype, 5), C, dtype)


@pytest.mark.parametrize("total_mib", [0.002, 0.3, 6, 48, 300])
@pytest.mark.parametrize("min_shift", [12])
def test_fused_tile_size_regimes_and_self_resetting_counters(total_mib, min_shift):
    """The device picks the tile size from the byte total: cover totals from below one tile per engine (no
    atomics at all) to thousands of tiles per engine (dynamic claims).  Two calls back to back: the second
    one only works if the first one's last CTA reset the claim counters."""
    R, rowbytes = 8, 512
    rng = np.random.default_rng(int(total_mib * 1000) + min_shift)
    p = rng.random((R, R)) ** 3
    rows = np.floor(p / p.sum() * total_mib * (1 << 20) / rowbytes).astype(np.int64)
    C = rows * (rowbytes // 2)
    send = make_send(C, "bf16", 7)
    assert_a2a_matches(send, C, "bf16")
    assert_a2a_matches(send, C, "bf16")
    # ragged variant of the same size: byte counts, every segment on the vector path or with bulk tails
    Cb = rows * rowbytes + rng.integers(0, 16, (R, R)) * (rows > 0)
    assert_a2a_matches(make_send(Cb, "u8", 9), Cb, "u8")


def test_fused_cfg1_roundtrip_in_a_graph_with_counts_by_reference():
    """Config 1 dispatch + inverse captured as TWO single-kernel calls; counts rewritten between replays (L401)."""
    cfg = W.a2a_config(1)
    R, width = cfg.R, cfg.width
    rng = np.random.default_rng(3)
    cap = 256 * R * width
    send_np = [W.np_values(cap, "bf16", 20 + s) for s in range(R)]
    send = [to_dev(a) for a in send_np]
    recv = [sentinel(cap * 2) for _ in range(R)]
    bk = [sentinel(cap * 2) for _ in range(R)]
    Cd = torch.from_numpy(cfg.counts).cuda()
    RCd, C2d = torch.zeros_like(Cd), torch.zeros_like(Cd)
    st, rt, bt = nx.device_ptr_table(send), nx.device_ptr_table(recv), nx.device_ptr_table(bk)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        nx.ncclx_alltoallv_dev(st, Cd, rt, RCd, R, "bf16")
    torch.cuda.current_stream().wait_stream(side)
    graph = torch.cuda.CUDAGraph()
    n0 = nx.ncclx_launch_count()
    with torch.cuda.graph(graph):
        nx.ncclx_alltoallv_dev(st, Cd, rt, RCd, R, "bf16")
        nx.ncclx_alltoallv_dev(rt, RCd, bt, C2d, R, "bf16")
    assert nx.ncclx_launch_count() - n0 == 2
    import oracle
    for it in range(4):
        C = cfg.counts if it == 0 else rng.integers(0, 257, (R, R)) * width * (rng.random((R, R)) < 0.7)
        C = C.astype(np.int64)
        for r in recv + bk:
            r.fill_(SENT8)
        Cd.copy_(torch.from_numpy(C), non_blocking=True)
        graph.replay()
        torch.cuda.synchronize()
        exp = [np.full(cap, 0xA5A5, np.uint16) for _ in range(R)]
        RC, *_ = oracle.alltoallv(send_np, C, exp, "bf16", nthreads=4)
        assert (RCd.cpu().numpy() == RC).all() and (C2d.cpu().numpy() == C).all()
        for d in range(R):
            assert back(recv[d], "bf16").tobytes() == exp[d].tobytes()
        for s in range(R):
            n = int(C[s].sum())
            got = back(bk[s], "bf16")
            assert got[:n].tobytes() == send_np[s][:n].tobytes() and (got[n:] == 0xA5A5).all()


# ---- split-phase form and plan slots --------------------------------------------------------------------

def a2a_buffers(send_np, C, dtype, slack=16):
    R = C.shape[0]
    es = ES[dtype]
    send = [to_dev(a) for a in send_np]
    recv = [sentinel((int(np.maximum(C, 0)[:, d].sum()) + slack) * es) for d in range(R)]
    Cd = torch.from_numpy(np.asarray(C, np.int64)).cuda()
    RCd = torch.full_like(Cd, -7)
    return send, recv, Cd, RCd, nx.device_ptr_table(send), nx.device_ptr_table(recv)


@pytest.mark.parametrize("R", [4, 64, 128])
@pytest.mark.parametrize("plan", [0, 1, 3])
def test_prepare_then_execute_matches_the_oracle_and_execute_is_repeatable(R, plan):
    rng = np.random.default_rng(R + plan)
    C = rng.integers(0, max(2, 4_000_000 // (R * R)), (R, R)) * 8
    C[rng.random((R, R)) < 0.3] = 0
    send_np = make_send(C, "bf16", 11)
    send, recv, Cd, RCd, st, rt = a2a_buffers(send_np, C, "bf16")
    exp, eRC, *_ = oracle_a2a(send_np, C, "bf16")
    assert launches_of(lambda: nx.ncclx_alltoallv_prepare_dev(plan, st, Cd, rt, RCd, R, "bf16")) == 1
    torch.cuda.synchronize()
    assert (RCd.cpu().numpy() == eRC).all()                          # metadata exchange done ...
    assert all((back(r, "u8") == SENT8).all() for r in recv)          # ... and no payload moved yet
    for _ in range(3):                                                # same work list, executed three times
        for r in recv:
            r.fill_(SENT8)
        assert launches_of(lambda: nx.ncclx_alltoallv_execute_dev(plan)) == 1
        torch.cuda.synchronize()
        for d in range(R):
            assert back(recv[d], "bf16").tobytes() == exp[d].tobytes()


def test_plan_slots_are_independent():
    """Two different calls prepared into two slots, executed in the opposite order."""
    R = 48
    rng = np.random.default_rng(1)
    CA = rng.integers(0, 3000, (R, R)) * 8
    CB = rng.integers(0, 500, (R, R)) * 8 * (rng.random((R, R)) < 0.5)
    sA, sB = make_send(CA, "bf16", 30), make_send(CB, "f32", 31)
    bufA, bufB = a2a_buffers(sA, CA, "bf16"), a2a_buffers(sB, CB, "f32")
    nx.ncclx_alltoallv_prepare_dev(1, bufA[4], bufA[2], bufA[5], bufA[3], R, "bf16")
    nx.ncclx_alltoallv_prepare_dev(2, bufB[4], bufB[2], bufB[5], bufB[3], R, "f32")
    nx.ncclx_alltoallv_execute_dev(2)
    nx.ncclx_alltoallv_execute_dev(1)
    torch.cuda.synchronize()
    for (send_np, C, dtype, buf) in ((sA, CA, "bf16", bufA), (sB, CB, "f32", bufB)):
        exp, eRC, *_ = oracle_a2a(send_np, C, dtype)
        assert (buf[3].cpu().numpy() == eRC).all()
        for d in range(R):
            assert back(buf[1][d], dtype).tobytes() == exp[d].tobytes()


def test_execute_argument_errors():
    nx.ncclx_finalize()
    nx.ncclx_init(128, 0)                    # fresh context: no slot prepared
    for plan in (0, 1, -1, nx.NUM_PLANS):
        with pytest.raises(nx.binding.NcclxError) as e:
            nx.ncclx_alltoallv_execute_dev(plan)
        assert e.value.code == 1
    t = torch.zeros(16, dtype=torch.int64, device="cuda")
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_alltoallv_prepare_dev(nx.NUM_PLANS, t, t, t, t[8:], 2, "bf16")
    assert e.value.code == 1
    n0 = nx.ncclx_launch_count()
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_alltoallv_prepare_dev(1, t, t, t, t, 2, "bf16")       # aliased count matrices
    assert e.value.code == 1
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_alltoallv_dev(t, t, t, t, 40, "bf16")                 # same, on the one-call entry point (two-kernel path)
    assert e.value.code == 1
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_alltoallv_dev(t, t, t, t[8:], 40, 9)                  # unknown dtype
    assert e.value.code == 2
    assert nx.ncclx_launch_count() == n0, "an argument error must not enqueue anything (header: error contract)"


def test_one_call_entry_point_leaves_slot_0_executable():
    """ncclx_alltoallv_dev == prepare(0) + execute(0) for R > 32: slot 0 then holds that call's plan, so its payload
    phase can be repeated; after a top-k call slot 0 holds a top-k plan and execute(0) is refused (round-1 ADVICE:
    the one-call entry points used to overwrite slot 0's tables without updating its state)."""
    R = 40
    rng = np.random.default_rng(77)
    C = rng.integers(0, 2000, (R, R)) * 8
    send_np = make_send(C, "bf16", 12)
    send, recv, Cd, RCd, st, rt = a2a_buffers(send_np, C, "bf16")
    exp, eRC, *_ = oracle_a2a(send_np, C, "bf16")
    nx.ncclx_alltoallv_dev(st, Cd, rt, RCd, R, "bf16")
    for r in recv:
        r.fill_(SENT8)
    nx.ncclx_alltoallv_execute_dev(0)
    torch.cuda.synchronize()
    for d in range(R):
        assert back(recv[d], "bf16").tobytes() == exp[d].tobytes()
    Crow = torch.from_numpy(np.full((4, 4), 2, np.int64)).cuda()
    nx.ncclx_moe_topk_prepare_dev(0, Crow, torch.zeros_like(Crow), 4)
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_alltoallv_execute_dev(0)
    assert e.value.code == 1
    torch.cuda.synchronize()


@pytest.mark.parametrize("use_graph", [False, True])
def test_double_buffered_dispatch_and_combine(use_graph):
    """The paper's double buffering (L483) in this build's terms: the combine's metadata phase (slot 1, counts =
    the dispatch's recvcounts) runs on a second stream while the dispatch's payload (slot 0) moves; then the
    combine's payload.  Config-5-shaped traffic; the round trip must be the identity and the dispatch must
    match the oracle; replayed with new counts when captured."""
    cfg = W.scaled_a2a(W.a2a_config(5), 1)
    R, width = cfg.R, cfg.width
    rng = np.random.default_rng(8)
    cap = 8 * R * width
    send_np = [W.np_values(cap, "bf16", 60 + s) for s in range(R)]
    send = [to_dev(a) for a in send_np]
    recv = [sentinel(cap * 2) for _ in range(R)]
    bk = [sentinel(cap * 2) for _ in range(R)]
    Cd = torch.from_numpy(cfg.counts).cuda()
    RCd, C2d = torch.zeros_like(Cd), torch.zeros_like(Cd)
    st, rt, bt = nx.device_ptr_table(send), nx.device_ptr_table(recv), nx.device_ptr_table(bk)
    side = torch.cuda.Stream()

    def enqueue():
        main = torch.cuda.current_stream()
        nx.ncclx_alltoallv_prepare_dev(0, st, Cd, rt, RCd, R, "bf16")
        side.wait_stream(main)                                        # fork after the dispatch's metadata phase
        with torch.cuda.stream(side):
            nx.ncclx_alltoallv_prepare_dev(1, rt, RCd, bt, C2d, R, "bf16")
        nx.ncclx_alltoallv_execute_dev(0)
        main.wait_stream(side)                                        # join
        nx.ncclx_alltoallv_execute_dev(1)

    warm = torch.cuda.Stream()
    warm.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(warm):
        enqueue()
    torch.cuda.current_stream().wait_stream(warm)
    torch.cuda.synchronize()
    graph = None
    if use_graph:
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            enqueue()
    import oracle
    for it in range(3):
        rows = cfg.rows if it == 0 else rng.integers(0, 9, (R, R)) * (rng.random((R, R)) < 0.5)
        C = (rows * width).astype(np.int64)
        for r in recv + bk:
            r.fill_(SENT8)
        Cd.copy_(torch.from_numpy(C), non_blocking=True)
        if graph is not None:
            graph.replay()
        else:
            enqueue()
        torch.cuda.synchronize()
        exp = [np.full(cap, 0xA5A5, np.uint16) for _ in range(R)]
        RC, *_ = oracle.alltoallv(send_np, C, exp, "bf16", nthreads=8)
        assert (RCd.cpu().numpy() == RC).all() and (C2d.cpu().numpy() == C).all()
        for d in range(R):
            assert back(recv[d], "bf16").tobytes() == exp[d].tobytes()
        for s in range(R):
            n = int(C[s].sum())
            got = back(bk[s], "bf16")
            assert got[:n].tobytes() == send_np[s][:n].tobytes() and (got[n:] == 0xA5A5).all()


@pytest.mark.parametrize("R", [8, 48])
def test_graph_with_memcpy_and_memset_nodes_before_the_call(R):
    """The metadata kernels are launched with programmatic stream serialisation; inside a captured graph their
    predecessor may be a memcpy or memset node instead of a kernel (the router's output copied into the count
    matrix).  One-kernel (R = 8) and two-kernel (R = 48) paths; counts by reference through the captured copy."""
    rng = np.random.default_rng(R)
    cap_rows, width = 64, 128
    rowsA = rng.integers(0, cap_rows // 2, (R, R))
    rowsB = rng.integers(0, cap_rows // 2, (R, R)) * (rng.random((R, R)) < 0.5)
    cap = cap_rows * R * width
    send_np = [W.np_values(cap, "bf16", 90 + s) for s in range(R)]
    send = [to_dev(a) for a in send_np]
    recv = [sentinel(cap * 2) for _ in range(R)]
    staging = torch.from_numpy((rowsA * width).astype(np.int64)).cuda()      # "router output"
    Cd = torch.zeros_like(staging)
    RCd = torch.zeros_like(staging)
    st, rt = nx.device_ptr_table(send), nx.device_ptr_table(recv)

    def enqueue():
        for r in recv:
            r.fill_(SENT8)                                                    # fill kernels / memset nodes
        RCd.zero_()
        Cd.copy_(staging)                                                     # D2D memcpy node right before the call
        nx.ncclx_alltoallv_dev(st, Cd, rt, RCd, R, "bf16")

    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        enqueue()
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        enqueue()
    import oracle
    for rows in (rowsA, rowsB):
        C = (rows * width).astype(np.int64)
        staging.copy_(torch.from_numpy(C))
        graph.replay()
        torch.cuda.synchronize()
        exp = [np.full(cap, 0xA5A5, np.uint16) for _ in range(R)]
        RC, *_ = oracle.alltoallv(send_np, C, exp, "bf16", nthreads=4)
        assert (RCd.cpu().numpy() == RC).all()
        for d in range(R):
            assert back(recv[d], "bf16").tobytes() == exp[d].tobytes()
