"""-m gpu parity: ncclx_alltoallv_dev (C ABI) vs the CPU oracle, byte for byte over the FULL
receive capacity (so writes past the packed end are caught), plus RC and the offset matrices."""
import json
import os

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
    nx.ncclx_init(1024, 0)
    yield
    nx.ncclx_finalize()


@pytest.fixture(autouse=True)
def default_params():
    yield
    nx.ncclx_set_param(nx.PARAM_BULK_MIN_BYTES, 1024)
    nx.ncclx_set_param(nx.PARAM_BULK_TILE_SHIFT, 15)
    nx.ncclx_set_param(nx.PARAM_COPY_BULK_ENGINES, 0)
    nx.ncclx_set_param(nx.PARAM_COPY_KMAX, 6)
    nx.ncclx_set_param(nx.PARAM_PDL, 1)


def make_send(C, dtype, seed=0):
    return [W.np_values(int(np.maximum(np.asarray(C)[s], 0).sum()), dtype, seed + s) for s in range(np.asarray(C).shape[0])]


def test_handworked_example(golden_dir):
    g = json.load(open(os.path.join(golden_dir, "handworked_alltoallv.json")))
    names = sorted({x for row in g["send"] for x in row})
    code = {n: i + 1000 for i, n in enumerate(names)}
    send = [np.array([code[x] for x in row], np.uint16) for row in g["send"]]
    got, RC, (soff, roff), _ = run_a2a(send, g["C"], "bf16", slack_elems=0)
    assert RC.tolist() == g["RC"] and soff.tolist() == g["soff"] and roff.tolist() == g["roff"]
    for d in range(2):
        assert got[d].tolist() == [code[x] for x in g["recv"][d]]


def test_cfg1_and_inverse():
    cfg = W.a2a_config(1)
    C = cfg.counts
    send = make_send(C, "bf16", 10)
    got, RC = assert_a2a_matches(send, C, "bf16")
    packed = [got[d][: int(C[:, d].sum())] for d in range(cfg.R)]
    back_, RC2 = assert_a2a_matches(packed, RC, "bf16")
    assert (RC2 == C).all()
    for s in range(cfg.R):
        assert back_[s][: send[s].size].tobytes() == send[s].tobytes()


@pytest.mark.parametrize("R", [1, 2, 3, 5, 8, 17, 33, 64, 100, 128])
@pytest.mark.parametrize("dtype", ["u8", "bf16", "f32"])
def test_random_counts_any_alignment(R, dtype):
    """Element-granular counts: segments start at arbitrary element offsets, so source and
    destination misalignment differ; zero rows/columns included; spans several tiles and tails."""
    rng = np.random.default_rng(R * 7 + ES[dtype])
    hi = max(2, 3_000_000 // (R * R))
    C = rng.integers(0, hi, (R, R))
    C[rng.random((R, R)) < 0.3] = 0
    if R > 2:
        C[R // 2, :] = 0
        C[:, R // 3] = 0
    send = make_send(C, dtype, 3)
    assert_a2a_matches(send, C, dtype)


@pytest.mark.parametrize("mis_send,mis_recv", [(0, 0), (2, 2), (2, 6), (16, 32), (4, 0), (1, 3)])
def test_misaligned_base_pointers(mis_send, mis_recv):
    dtype = "u8" if (mis_send | mis_recv) & 1 else "bf16"
    R = 6
    rng = np.random.default_rng(5)
    C = rng.integers(0, 70_000, (R, R)) * 8          # multiples of 16 B so only the bases misalign
    send = make_send(C, dtype, 9)
    got, RC, offs, status = run_a2a(send, C, dtype, mis_send=mis_send, mis_recv=mis_recv)
    exp, eRC, *_ = oracle_a2a(send, C, dtype)
    assert all(g.tobytes() == e.tobytes() for g, e in zip(got, exp)) and (RC == eRC).all()


@pytest.mark.parametrize("rowbytes", [16, 256, 1024, 10240, 14336])
def test_aligned_rows_mixed_sizes_bulk_and_vector(rowbytes):
    """16B-aligned rows: segments above BULK_MIN_BYTES take cp.async.bulk, the rest the vector path;
    includes segments of many tiles, exactly one tile, and zero."""
    R = 16
    rng = np.random.default_rng(rowbytes)
    rows = rng.integers(0, max(2, (1 << 20) // rowbytes), (R, R))
    rows[rng.random((R, R)) < 0.25] = 0
    rows[0, 0] = (3 << 20) // rowbytes + 1           # a long one
    rows[1, 2] = max(1, 32768 // rowbytes)           # ~ one tile
    rows[2, 1] = 1
    C = rows * (rowbytes // 2)
    send = make_send(C, "bf16", 1)
    assert_a2a_matches(send, C, "bf16")


def test_ragged_bulk_tail_and_tiny_segments():
    """Aligned sources/destinations but byte lengths not multiple of 16 (u8): the bulk path moves
    floor16 and the engine copies the < 16 B tail; later segments become unaligned -> vector."""
    R = 4
    C = np.array([[40000 + 5, 16, 1, 0], [7, 131072 + 15, 3, 32768], [0, 0, 0, 0], [65536, 15, 17, 100001]])
    send = make_send(C, "u8", 2)
    assert_a2a_matches(send, C, "u8")
    # first segment of every destination is 16B-aligned with ragged length: exercise bulk tail on each
    C2 = np.zeros((R, R), np.int64)
    C2[0] = [32768 * 3 + 9, 2048 + 1, 1024 + 15, 5000]
    send = make_send(C2, "u8", 3)
    assert_a2a_matches(send, C2, "u8")


# BULK_MIN_BYTES = 2^40 sends every segment down the vector list (TMA-staged pieces + warp stores) although all are aligned
@pytest.mark.parametrize("param,value", [("BULK_MIN_BYTES", 1 << 40), ("BULK_MIN_BYTES", 16), ("BULK_MIN_BYTES", 1 << 20),
                                         ("BULK_TILE_SHIFT", 12), ("BULK_TILE_SHIFT", 16),
                                         ("COPY_BULK_ENGINES", 1), ("COPY_BULK_ENGINES", 2), ("COPY_BULK_ENGINES", 4),
                                         ("COPY_KMAX", 1), ("COPY_KMAX", 17), ("PDL", 0)])
def test_launch_configurations_agree(param, value):
    nx.ncclx_set_param(getattr(nx, "PARAM_" + param), value)
    cfg = W.scaled_a2a(W.a2a_config(3), 64)
    C = cfg.counts
    send = make_send(C, "bf16", 4)
    assert_a2a_matches(send, C, "bf16")


@pytest.mark.parametrize("engines", [2, 4])
def test_small_R_and_cfg5_shapes_with_several_bulk_engines(engines):
    """E bulk engine warps per CTA (ring split E ways) on the single-launch path and on short-segment traffic."""
    nx.ncclx_set_param(nx.PARAM_COPY_BULK_ENGINES, engines)
    rng = np.random.default_rng(engines)
    C = rng.integers(0, 60_000, (8, 8)) * 8
    assert_a2a_matches(make_send(C, "bf16", 21), C, "bf16")
    cfg = W.scaled_a2a(W.a2a_config(5), 2)
    assert_a2a_matches(make_send(cfg.counts, "bf16", 22), cfg.counts, "bf16")


def test_cfg5_small_messages_full_compare():
    cfg = W.a2a_config(5)
    C = cfg.counts
    send = make_send(C, "bf16", 40)
    got, RC = assert_a2a_matches(send, C, "bf16")
    # by-bytes accounting (padding-free): bytes moved == sum of counts
    assert sum(int(C[:, d].sum()) for d in range(cfg.R)) * 2 == int(cfg.rows.sum()) * 14336


def test_uniform_counts_block_transpose():
    R, c = 32, 4096
    send = make_send(np.full((R, R), c), "f32", 8)
    got, RC, _, _ = run_a2a(send, np.full((R, R), c), "f32", slack_elems=0)
    exp = np.stack(send).reshape(R, R, c).swapaxes(0, 1)
    for d in range(R):
        assert got[d].tobytes() == exp[d].tobytes()


def test_tagged_payload_closed_form():
    cfg = W.a2a_config(1)
    C = cfg.rows * 64
    send = [W.tagged_payload_u32(s, int(C[s].sum())).view(np.float32) for s in range(cfg.R)]
    got, *_ = run_a2a(send, C, "f32", slack_elems=0)
    excl = np.cumsum(C, axis=1) - C
    for d in range(cfg.R):
        exp = np.concatenate([(np.uint32(s) << np.uint32(24)) | (np.uint32(excl[s, d]) + np.arange(C[s, d], dtype=np.uint32))
                              for s in range(cfg.R)])
        assert (got[d].view(np.uint32) == exp).all()


def test_zero_matrix_negative_counts_and_R_limits():
    R = 5
    send = [W.np_values(8, "bf16", s) for s in range(R)]
    got, RC, (soff, roff), status = run_a2a(send, np.zeros((R, R), np.int64), "bf16")
    assert status == 0 and (RC == 0).all() and (soff == 0).all() and (roff == 0).all()
    assert all((g.view(np.uint8) == SENT8).all() for g in got)
    C = np.array([[2, -5], [1, 1]])
    send = [W.np_values(2, "bf16", 0), W.np_values(2, "bf16", 1)]
    assert_a2a_matches(send, C, "bf16")              # status == 1, negative treated as 0
    assert nx.ncclx_device_status() == 0             # cleared by the read
    t = torch.zeros(4, dtype=torch.int64, device="cuda")
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_alltoallv_dev(t, t, t, t, 2, "bf16")  # same count buffer for in and out
    assert e.value.code == 1
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_alltoallv_dev(t, t, t, t[1:], 2000, "bf16")
    assert e.value.code == 3
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_alltoallv_dev(t, t, t, t[1:], 2, 9)
    assert e.value.code == 2


@pytest.mark.parametrize("R", [256, 1024])
def test_large_R(R):
    rng = np.random.default_rng(R)
    C = rng.integers(0, 40, (R, R))
    C[rng.random((R, R)) < 0.5] = 0
    C[1, 2] = 300_000
    send = make_send(C, "bf16", 6)
    assert_a2a_matches(send, C, "bf16")


@pytest.mark.parametrize("R", [129, 160, 512])
def test_large_R_metadata_barrier_in_plan_slots_and_graph_replays(R):
    """Above 128 ranks the metadata kernel's CTAs exchange block sums through a self-resetting grid barrier in the plan
    slot's control block: a dispatch and its inverse prepared into two slots (the second on a side stream, beside the
    first one's payload kernel, which holds every SM), captured once and replayed with the counts rewritten between
    replays -- offsets, receive counts and every byte against the oracle each time."""
    import oracle
    rng = np.random.default_rng(R)
    hi = max(3, 6_000_000 // (R * R))
    cap = hi * R                                               # elements a rank can send / receive at most
    send_np = [W.np_values(cap, "bf16", 700 + s) for s in range(R)]
    send = [to_dev(a) for a in send_np]
    recv = [sentinel(cap * 2) for _ in range(R)]
    bk = [sentinel(cap * 2) for _ in range(R)]
    Cd = torch.zeros((R, R), dtype=torch.int64, device="cuda")
    RCd, C2d = torch.zeros_like(Cd), torch.zeros_like(Cd)
    st, rt, bt = nx.device_ptr_table(send), nx.device_ptr_table(recv), nx.device_ptr_table(bk)
    side = torch.cuda.Stream()

    def pair():
        main = torch.cuda.current_stream()
        nx.ncclx_alltoallv_prepare_dev(2, st, Cd, rt, RCd, R, "bf16")
        side.wait_stream(main)
        with torch.cuda.stream(side):
            nx.ncclx_alltoallv_prepare_dev(3, rt, RCd, bt, C2d, R, "bf16")
        nx.ncclx_alltoallv_execute_dev(2)
        main.wait_stream(side)
        nx.ncclx_alltoallv_execute_dev(3)
    warm = torch.cuda.Stream()
    warm.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(warm):
        pair()
    torch.cuda.current_stream().wait_stream(warm)
    torch.cuda.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        pair()
    for it in range(3):
        C = rng.integers(0, hi, (R, R)).astype(np.int64)
        C[rng.random((R, R)) < 0.4] = 0
        if it == 1:
            C[:, R // 2] = 0
        for r in recv + bk:
            r.fill_(SENT8)
        Cd.copy_(torch.from_numpy(C), non_blocking=True)
        graph.replay()
        torch.cuda.synchronize()
        exp = [np.full(cap, 0xA5A5, np.uint16) for _ in range(R)]
        RC, *_ = oracle.alltoallv(send_np, C, exp, "bf16", nthreads=4)
        assert (RCd.cpu().numpy() == RC).all() and (C2d.cpu().numpy() == C).all()
        for d in range(R):
            assert back(recv[d], "bf16").tobytes() == exp[d].tobytes(), f"replay {it} recv[{d}]"
        for s in range(R):
            n = int(C[s].sum())
            got = back(bk[s], "bf16")
            assert got[:n].tobytes() == send_np[s][:n].tobytes() and (got[n:] == 0xA5A5).all(), f"replay {it} round trip {s}"


def test_graph_capture_counts_by_reference():
    """counts may change until the collective executes.  Capture once with one
    count matrix, rewrite the device-resident counts between replays, outputs must follow."""
    R, width = 8, 256
    rng = np.random.default_rng(11)
    rowsA = rng.integers(0, 300, (R, R))
    rowsB = rng.integers(0, 300, (R, R)); rowsB[rng.random((R, R)) < 0.4] = 0
    rowsC = np.zeros((R, R), np.int64); rowsC[3, 5] = 299
    cap_rows = 300 * R
    send_np = [W.np_values(cap_rows * width, "bf16", 50 + s) for s in range(R)]
    send = [to_dev(a) for a in send_np]
    recv = [sentinel(cap_rows * width * 2) for _ in range(R)]
    Cd = torch.from_numpy(rowsA * width).cuda()
    RCd = torch.zeros_like(Cd)
    st, rt = nx.device_ptr_table(send), nx.device_ptr_table(recv)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        nx.ncclx_alltoallv_dev(st, Cd, rt, RCd, R, "bf16")   # warm-up outside capture
    torch.cuda.current_stream().wait_stream(side)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        nx.ncclx_alltoallv_dev(st, Cd, rt, RCd, R, "bf16")
    import oracle
    for rows in (rowsA, rowsB, rowsC, rowsA):
        C = (rows * width).astype(np.int64)
        for r in recv:
            r.fill_(SENT8)
        Cd.copy_(torch.from_numpy(C), non_blocking=True)       # stream-ordered rewrite of the metadata
        graph.replay()
        torch.cuda.synchronize()
        exp = [np.full(cap_rows * width, 0xA5A5, np.uint16) for _ in range(R)]
        RC, *_ = oracle.alltoallv(send_np, C, exp, "bf16", nthreads=4)
        assert (RCd.cpu().numpy() == RC).all()
        for d in range(R):
            assert back(recv[d], "bf16").tobytes() == exp[d].tobytes()


@pytest.mark.parametrize("mode", ["pinned_zero_copy", "pinned_staged", "pageable"])
def test_host_buffer_form(mode):
    """Host-buffer entry point: pinned buffers are accessed by the kernels directly (zero-copy), pageable ones
    (or NCCLX_PARAM_HOST_ZERO_COPY = 0) are staged through device memory; same result either way."""
    nx.ncclx_set_param(nx.PARAM_HOST_ZERO_COPY, 0 if mode == "pinned_staged" else 1)
    try:
        cfg = W.scaled_a2a(W.a2a_config(3), 128)
        C = cfg.counts
        R = cfg.R
        send_np = make_send(C, "bf16", 70)
        if mode == "pageable":
            src = [a.copy() for a in send_np]
            out = [np.full(int(C[:, d].sum()) + 8, 0xA5A5, np.uint16) for d in range(R)]
        else:
            src = [torch.from_numpy(a.view(np.int16)).pin_memory() for a in send_np]
            out = [torch.full((int(C[:, d].sum()) + 8,), -23131, dtype=torch.int16).pin_memory() for d in range(R)]
        RCh = np.zeros((R, R), np.int64)
        nx.ncclx_alltoallv_host(src, np.ascontiguousarray(C), out, RCh, R, "bf16")
        exp, eRC, *_ = oracle_a2a(send_np, C, "bf16", slack_elems=8)
        assert (RCh == eRC).all()
        for d in range(R):
            got = out[d] if mode == "pageable" else out[d].numpy().view(np.uint16)
            assert got.tobytes() == exp[d].tobytes()          # incl. the untouched 0xA5 tail
    finally:
        nx.ncclx_set_param(nx.PARAM_HOST_ZERO_COPY, 1)


@pytest.mark.parametrize("fused", [32, 0])
def test_every_source_destination_misalignment_pair(fused):
    """All 16 x 16 combinations of source / destination base misalignment modulo 16 with odd byte counts: co-aligned
    pairs take the 16-byte vector path, the others the funnel-shift path (aligned vectors on both sides), each
    with its own head and tail bytes; small enough for the whole receive capacity to be compared every time."""
    nx.ncclx_set_param(nx.PARAM_FUSED_MAX_RANKS, fused)
    try:
        rng = np.random.default_rng(77)
        C = np.array([[4099, 63, 1], [777, 20001, 64], [65, 0, 129]], np.int64)
        send = make_send(C, "u8", 12)
        exp, eRC, *_ = oracle_a2a(send, C, "u8")
        for ms in range(16):
            for md in range(16):
                got, RC, _, _ = run_a2a(send, C, "u8", mis_send=ms, mis_recv=md)
                assert (RC == eRC).all()
                for d in range(3):
                    assert got[d].tobytes() == exp[d].tobytes(), f"mis_send={ms} mis_recv={md} recv[{d}]"
    finally:
        nx.ncclx_set_param(nx.PARAM_FUSED_MAX_RANKS, 32)


@pytest.mark.parametrize("fused", [32, 0])
def test_vector_pieces_around_the_staging_boundaries(fused):
    """The vector engines stage a tile in pieces of at most 4 KiB whose ends follow the DESTINATION's 16-byte grid, realign
    each piece in shared memory and store its body with one bulk copy: segment lengths 0..80 (no body at all, head and
    tail only) and every length around one and two pieces (tiny trailing piece copied by lanes, body of a single vector),
    each with source and destination misaligned alike, differently, and not at all.  One call holds all lengths (a
    segment per (s, d) pair), so the full receive capacity incl. every neighbour's bytes is compared each time."""
    nx.ncclx_set_param(nx.PARAM_FUSED_MAX_RANKS, fused)
    try:
        lens = list(range(0, 81)) + list(range(4060, 4140)) + list(range(8170, 8215)) + [16384, 16385, 16399, 32769]
        R = 15
        assert R * R >= len(lens)
        C = np.zeros((R, R), np.int64)
        for i, n in enumerate(lens):
            C[i // R, i % R] = n
        send = make_send(C, "u8", 91)
        exp, eRC, *_ = oracle_a2a(send, C, "u8")
        for ms, md in ((0, 0), (5, 5), (3, 9), (9, 3), (0, 15), (1, 0), (15, 14)):
            got, RC, _, _ = run_a2a(send, C, "u8", mis_send=ms, mis_recv=md)
            assert (RC == eRC).all()
            for d in range(R):
                assert got[d].tobytes() == exp[d].tobytes(), f"mis_send={ms} mis_recv={md} recv[{d}]"
    finally:
        nx.ncclx_set_param(nx.PARAM_FUSED_MAX_RANKS, 32)


def test_randomised_shapes_alignments_and_paths():
    """Seeded sweep over what the other tests fix one at a time: R (incl. 1, 31..33, 128..129), dtype, count
    distributions (dense, sparse, one huge segment among tiny ones, multiples of 8, tiny, heavy-tailed, empty columns),
    base misalignment of send and receive buffers, single-launch vs two-kernel path -- metadata and every byte of the
    full receive capacity against the oracle (120 cases; the same generator ran 28 400 cases clean during development)."""
    try:
        for it in range(120):
            rng = np.random.default_rng(50_000 + it)
            R = int(rng.choice([1, 2, 3, 4, 7, 16, 31, 32, 33, 40, 64, 100, 128, 129, 200]))
            dtype = str(rng.choice(["u8", "bf16", "f32"]))
            mode = int(rng.integers(0, 6))
            budget = int(rng.choice([20_000, 400_000, 4_000_000, 30_000_000])) // ES[dtype]
            if mode == 0:
                C = rng.integers(0, max(2, budget // (R * R)), (R, R))
            elif mode == 1:
                C = rng.integers(0, max(2, budget // (R * R)), (R, R)) * (rng.random((R, R)) < 0.2)
            elif mode == 2:
                C = rng.integers(0, 6, (R, R))
                C[rng.integers(0, R), rng.integers(0, R)] = budget
            elif mode == 3:
                C = rng.integers(0, max(2, budget // (R * R * 8)), (R, R)) * 8
            elif mode == 4:
                C = rng.integers(0, 70, (R, R))
            else:
                C = np.round(rng.pareto(1.2, (R, R)) * max(1, budget // (R * R * 4))).astype(np.int64)
            C = np.minimum(C.astype(np.int64), budget)
            if rng.random() < 0.2:
                C[:, rng.integers(0, R)] = 0
            fused = int(rng.choice([0, 32]))
            ms, md = (int(rng.integers(0, 16)), int(rng.integers(0, 16))) if rng.random() < 0.7 else (0, 0)
            ms -= ms % ES[dtype]
            md -= md % ES[dtype]
            nx.ncclx_set_param(nx.PARAM_FUSED_MAX_RANKS, fused)
            send = make_send(C, dtype, 1000 * it)
            got, RC, (soff, roff), _ = run_a2a(send, C, dtype, mis_send=ms, mis_recv=md)
            exp, eRC, esoff, eroff, _ = oracle_a2a(send, C, dtype)
            what = f"case {it}: R={R} {dtype} mode={mode} fused={fused} mis=({ms},{md})"
            assert (RC == eRC).all() and (soff == esoff).all() and (roff == eroff).all(), what
            for d in range(R):
                assert got[d].tobytes() == exp[d].tobytes(), what + f" recv[{d}]"
    finally:
        nx.ncclx_set_param(nx.PARAM_FUSED_MAX_RANKS, 32)
