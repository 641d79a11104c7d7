"""-m gpu parity: ncclx_allreduce_sum / ncclx_reducescatter_sum (C ABI) vs the CPU oracle,
bit for bit (tolerance 0: fixed-order fp32 accumulation has one correct result)."""
import os

import numpy as np
import pytest
import torch

import oracle
import paper_2510_20171_b200 as nx
from paper_2510_20171_b200 import workloads as W

pytestmark = pytest.mark.gpu

from gpu_util import ES, NP_OF, back, to_dev  # noqa: E402


@pytest.fixture(scope="module", autouse=True)
def ctx():
    assert torch.cuda.is_available()
    nx.ncclx_init(1024, 0)
    yield
    nx.ncclx_finalize()


def gpu_allreduce(xs_np, dtype, mis=0, inplace=False):
    R, n = len(xs_np), xs_np[0].size
    xs = [to_dev(a, mis) for a in xs_np]
    outs = xs if inplace else [torch.zeros(n * ES[dtype] + 64, dtype=torch.uint8, device="cuda")[mis:mis + n * ES[dtype]]
                               for _ in range(R)]
    nx.ncclx_allreduce_sum(nx.device_ptr_table(xs), nx.device_ptr_table(outs), n, R, dtype)
    torch.cuda.synchronize()
    return [back(o, dtype) for o in outs]


def gpu_reducescatter(xs_np, dtype, mis=0):
    R, N = len(xs_np), xs_np[0].size
    n = N // R
    xs = [to_dev(a, mis) for a in xs_np]
    outs = [torch.zeros(n * ES[dtype] + 64, dtype=torch.uint8, device="cuda")[mis:mis + n * ES[dtype]] for _ in range(R)]
    nx.ncclx_reducescatter_sum(nx.device_ptr_table(xs), nx.device_ptr_table(outs), n, R, dtype)
    torch.cuda.synchronize()
    return [back(o, dtype) for o in outs]


def inject_specials(a: np.ndarray, dtype: str, seed: int) -> np.ndarray:
    """Sprinkle inf / nan / subnormal / signed-zero bit patterns (reading 13/14 of DESIGN.md)."""
    rng = np.random.default_rng(seed)
    a = a.copy()
    idx = rng.integers(0, a.size, max(1, a.size // 50))
    if dtype == "f32":
        pats = np.array([0x7F800000, 0xFF800000, 0x7FC00001, 0xFFFFFFFF, 1, 0x80000001, 0x007FFFFF, 0x80000000, 0], np.uint32)
        a.view(np.uint32)[idx] = rng.choice(pats, idx.size)
    elif dtype == "bf16":
        pats = np.array([0x7F80, 0xFF80, 0x7FC1, 0xFFFF, 1, 0x8001, 0x007F, 0x8000, 0, 0x7F7F, 0xFF7F], np.uint16)
        a[idx] = rng.choice(pats, idx.size)
    else:
        pats = np.array([0x7C00, 0xFC00, 0x7E01, 0xFFFF, 1, 0x8001, 0x03FF, 0x8000, 0, 0x7BFF, 0xFBFF], np.uint16)
        a[idx] = rng.choice(pats, idx.size)
    return a


def test_golden_vectors(golden_dir):
    for line in open(os.path.join(golden_dir, "bf16_sum_vectors.txt")):
        line = line.split("#")[0].strip()
        if not line:
            continue
        lhs, rhs = line.split("->")
        ins, exp = [int(t, 16) for t in lhs.split()], int(rhs, 16)
        for n in (1, 8, 9):                           # scalar-tail, vector, vector + tail
            outs = gpu_allreduce([np.full(n, v, np.uint16) for v in ins], "bf16")
            assert all((o == exp).all() for o in outs), (line, n, [hex(int(o[0])) for o in outs])


def test_cfg2_allreduce_full():
    cfg = W.reduce_config(2)
    xs = [W.np_values(cfg.count, "bf16", cfg.seed * 100 + k) for k in range(cfg.R)]
    got = gpu_allreduce(xs, "bf16")
    exp = oracle.allreduce_sum(xs, "bf16", nthreads=8)
    for r in range(cfg.R):
        assert got[r].tobytes() == exp[r].tobytes()


@pytest.mark.parametrize("R", [1, 2, 3, 4, 5, 8, 9, 16, 17, 40, 64])
@pytest.mark.parametrize("dtype", ["bf16", "f32", "f16"])
def test_random_R_ragged_sizes_with_specials(R, dtype):
    n = 8 * 256 * 5 + 8 * 77 + 3                      # several tiles + ragged tile + scalar tail
    xs = [inject_specials(W.np_values(n, dtype, 100 * R + k, 1.0 if k % 2 else 1e-3), dtype, k) for k in range(R)]
    got = gpu_allreduce(xs, dtype)
    exp = oracle.allreduce_sum(xs, dtype, nthreads=4)
    for r in range(R):
        assert got[r].tobytes() == exp[r].tobytes(), (R, dtype, r)


@pytest.mark.parametrize("dtype", ["bf16", "f32", "f16"])
@pytest.mark.parametrize("R,n", [(4, 8 * 1000), (16, 8 * 300 + 8), (3, 1001), (16, 5)])
def test_reducescatter_matches_oracle_and_allreduce_slices(dtype, R, n):
    xs = [inject_specials(W.np_values(R * n, dtype, 7 * R + k), dtype, 50 + k) for k in range(R)]
    rs = gpu_reducescatter(xs, dtype)
    ers = oracle.reducescatter_sum(xs, dtype, nthreads=4)
    ar = gpu_allreduce(xs, dtype)
    for r in range(R):
        assert rs[r].tobytes() == ers[r].tobytes()
        assert rs[r].tobytes() == ar[0][r * n:(r + 1) * n].tobytes()   # cross-API invariant
        assert ar[r].tobytes() == ar[0].tobytes()


@pytest.mark.parametrize("mis", [2, 4, 8, 6])
def test_misaligned_pointers_scalar_path(mis):
    R, n = 5, 4099
    xs = [W.np_values(n, "bf16", 900 + k) for k in range(R)]
    assert all(g.tobytes() == e.tobytes() for g, e in zip(gpu_allreduce(xs, "bf16", mis=mis), oracle.allreduce_sum(xs, "bf16")))
    xs = [W.np_values(R * 1003, "bf16", 950 + k) for k in range(R)]
    assert all(g.tobytes() == e.tobytes() for g, e in zip(gpu_reducescatter(xs, "bf16", mis=mis), oracle.reducescatter_sum(xs, "bf16")))


def test_inplace_allreduce_and_all_bf16_patterns():
    R, n = 8, 8 * 4096 + 5
    xs = [W.np_values(n, "bf16", 300 + k) for k in range(R)]
    got = gpu_allreduce(xs, "bf16", inplace=True)
    exp = oracle.allreduce_sum(xs, "bf16", nthreads=4)
    assert all(g.tobytes() == e.tobytes() for g, e in zip(got, exp))
    allb = np.arange(65536, dtype=np.uint16)
    assert gpu_allreduce([allb], "bf16")[0].tobytes() == oracle.allreduce_sum([allb], "bf16")[0].tobytes()
    assert gpu_allreduce([allb], "f16")[0].tobytes() == oracle.allreduce_sum([allb], "f16")[0].tobytes()
    # every bf16 pattern plus every other pattern shifted: exercises the final RNE over many exponents
    b = np.roll(allb, 12345)
    assert gpu_allreduce([allb, b], "bf16")[0].tobytes() == oracle.allreduce_sum([allb, b], "bf16")[0].tobytes()
    assert gpu_allreduce([allb, b], "f16")[0].tobytes() == oracle.allreduce_sum([allb, b], "f16")[0].tobytes()


def test_small_integer_sums_exact():
    R, n = 64, 8 * 513
    rng = np.random.default_rng(0)
    ints = rng.integers(-2, 3, (R, n))
    xs = [torch.from_numpy(ints[k].astype(np.float32)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16) for k in range(R)]
    got = gpu_allreduce(xs, "bf16")[0]
    val = (got.astype(np.uint32) << 16).view(np.float32)
    assert (val == ints.sum(axis=0)).all()


def test_errors_and_noop():
    t = torch.zeros(8, dtype=torch.int64, device="cuda")
    nx.ncclx_allreduce_sum(t, t, 0, 2, "bf16")         # count == 0: no-op
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_allreduce_sum(t, t, 8, 2, "u8")
    assert e.value.code == 2
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_reducescatter_sum(t, t, 8, 0, "bf16")
    assert e.value.code == 1


@pytest.mark.parametrize("mode", ["pinned_zero_copy", "pinned_staged", "pageable"])
def test_host_buffer_forms(mode):
    nx.ncclx_set_param(nx.PARAM_HOST_ZERO_COPY, 0 if mode == "pinned_staged" else 1)
    try:
        R, n = 4, 8 * 5000
        xs = [W.np_values(R * n, "bf16", 600 + k) for k in range(R)]
        if mode == "pageable":
            src = [a.copy() for a in xs]
            out_ar = [np.zeros(R * n, np.uint16) for _ in range(R)]
            out_rs = [np.zeros(n, np.uint16) for _ in range(R)]
            view = lambda t: t
        else:
            src = [torch.from_numpy(a.view(np.int16)).pin_memory() for a in xs]
            out_ar = [torch.empty(R * n, dtype=torch.int16).pin_memory() for _ in range(R)]
            out_rs = [torch.empty(n, dtype=torch.int16).pin_memory() for _ in range(R)]
            view = lambda t: t.numpy().view(np.uint16)
        nx.ncclx_allreduce_sum_host(src, out_ar, R * n, R, "bf16")
        nx.ncclx_reducescatter_sum_host(src, out_rs, n, R, "bf16")
        exp = oracle.allreduce_sum(xs, "bf16", nthreads=4)
        for r in range(R):
            assert view(out_ar[r]).tobytes() == exp[r].tobytes()
            assert view(out_rs[r]).tobytes() == exp[0][r * n:(r + 1) * n].tobytes()
    finally:
        nx.ncclx_set_param(nx.PARAM_HOST_ZERO_COPY, 1)


# ---- NEXT-2: FTAR-style ReduceCopy step -------------------------------------------------

@pytest.mark.parametrize("dtype", ["bf16", "f32", "f16"])
@pytest.mark.parametrize("n,chunk,ctas", [(8 * 1024 * 1024 // 2 * 3 + 8 * 100 + 5, 8 << 20, 2), (100_003, 4096, 1),
                                          (16 * 512 * 4 * 3, 16 * 512 * 4 * 2, 3), (777, 0, 0)])
@pytest.mark.parametrize("tma", [0, 1])
def test_reducecopy_matches_two_rank_oracle(dtype, n, chunk, ctas, tma):
    """Both inner loops (NCCLX_PARAM_REDUCECOPY_TMA: pipelined register loads / TMA-fed shared-memory ring)."""
    nx.ncclx_set_param(nx.PARAM_REDUCECOPY_TMA, tma)
    try:
        _reducecopy_case(dtype, n, chunk, ctas)
    finally:
        nx.ncclx_set_param(nx.PARAM_REDUCECOPY_TMA, 0)


def _reducecopy_case(dtype, n, chunk, ctas):
    a = inject_specials(W.np_values(n, dtype, 1), dtype, 1)
    b = inject_specials(W.np_values(n, dtype, 2, 1e-3), dtype, 2)
    exp = oracle.allreduce_sum([a, b], dtype, nthreads=4)[0]
    da, db = to_dev(a), to_dev(b)
    nb = n * ES[dtype]
    out = torch.zeros(nb + 64, dtype=torch.uint8, device="cuda")[:nb]
    fwd = torch.zeros(nb + 64, dtype=torch.uint8, device="cuda")[:nb]
    nx.ncclx_reducecopy_sum(da, db, out, fwd, n, dtype, chunk, ctas)            # ReduceCopy with local result
    torch.cuda.synchronize()
    assert back(out, dtype).tobytes() == exp.tobytes() and back(fwd, dtype).tobytes() == exp.tobytes()
    fwd.zero_()
    nx.ncclx_reducecopy_sum(da, db, None, fwd, n, dtype, chunk, ctas)           # intermediate step: forward only
    nx.ncclx_reducecopy_sum(da, db, db, None, n, dtype, chunk, ctas)            # Reduce, in place on the local chunk
    torch.cuda.synchronize()
    assert back(fwd, dtype).tobytes() == exp.tobytes() and back(db, dtype).tobytes() == exp.tobytes()


def test_reducecopy_misaligned_and_errors():
    n = 5001
    a, b = W.np_values(n, "bf16", 3), W.np_values(n, "bf16", 4)
    da, db = to_dev(a, 2), to_dev(b, 6)
    out = torch.zeros(2 * n + 64, dtype=torch.uint8, device="cuda")[10:10 + 2 * n]
    nx.ncclx_reducecopy_sum(da, db, out, None, n, "bf16", 1000, 2)
    torch.cuda.synchronize()
    assert back(out, "bf16").tobytes() == oracle.allreduce_sum([a, b], "bf16")[0].tobytes()
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_reducecopy_sum(da, db, None, None, n, "bf16")
    assert e.value.code == 1
    with pytest.raises(nx.binding.NcclxError) as e:
        nx.ncclx_reducecopy_sum(da, db, out, None, n, "u8")
    assert e.value.code == 2


def test_stream_probe_few_cta_form():
    """Per-SM ceiling probe (fixed small grid of 1024-thread CTAs): same copy semantics."""
    n = 32 * 70_001
    src = torch.randint(0, 255, (n,), dtype=torch.uint8, device="cuda")
    dst = torch.full((n + 32,), 0xA5, dtype=torch.uint8, device="cuda")
    for ctas in (1, 2, 4):
        dst.fill_(0xA5)
        nx.ncclx_stream_probe_ctas(2, src, dst, n, ctas)
        torch.cuda.synchronize()
        assert torch.equal(dst[:n], src) and bool((dst[n:] == 0xA5).all())
    with pytest.raises(nx.binding.NcclxError):
        nx.ncclx_stream_probe_ctas(2, src, dst, n, 0)


def test_stream_probe_modes():
    """Measurement aid: copy mode copies, read-only leaves both buffers alone, write-only fills."""
    n = 32 * 100_003
    src = torch.randint(0, 255, (n,), dtype=torch.uint8, device="cuda")
    dst = torch.full((n + 32,), 0xA5, dtype=torch.uint8, device="cuda")
    ref = src.clone()
    nx.ncclx_stream_probe(0, src, None, n)
    torch.cuda.synchronize()
    assert torch.equal(src, ref) and bool((dst == 0xA5).all())
    nx.ncclx_stream_probe(2, src, dst, n)
    torch.cuda.synchronize()
    assert torch.equal(dst[:n], ref) and bool((dst[n:] == 0xA5).all())
    nx.ncclx_stream_probe(1, None, dst, n)
    torch.cuda.synchronize()
    w = dst[:n].view(torch.int32).view(-1, 8).cpu()
    assert bool((w[:, 0] == torch.arange(n // 32, dtype=torch.int32)).all()) and bool((w[:, 1:] == torch.arange(1, 8, dtype=torch.int32)).all())
    assert bool((dst[n:] == 0xA5).all())
    with pytest.raises(nx.binding.NcclxError):
        nx.ncclx_stream_probe(2, src, dst, n + 1)
    chunk = 32 * 1024
    big = torch.full((5 * chunk + 64,), 0xA5, dtype=torch.uint8, device="cuda")
    nx.ncclx_stream_probe(3, None, big, 5 * chunk)               # TMA bulk stores of a fixed 32 KiB pattern
    torch.cuda.synchronize()
    w = big[:5 * chunk].view(torch.int32).view(5, chunk // 4).cpu()
    assert bool((w == torch.arange(chunk // 4, dtype=torch.int32)).all()) and bool((big[5 * chunk:] == 0xA5).all())
