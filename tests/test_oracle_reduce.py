"""Pins for the sum-reduction oracle: IEEE rounding vectors worked by hand (tests/golden),
exact small-integer sums, library special cases (numpy float32 add, torch's bf16 cast),
fp64 error bound, cross-API invariants."""
import os

import numpy as np
import pytest
import torch

import oracle
from paper_2510_20171_b200 import workloads as W


def bf16_bits(x_f32: np.ndarray) -> np.ndarray:
    """torch's fp32->bf16 cast (library routine, independent of the oracle)."""
    return torch.from_numpy(np.ascontiguousarray(x_f32, np.float32)).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16)


def bf16_to_f64(bits: np.ndarray) -> np.ndarray:
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def golden_vectors(golden_dir):
    out = []
    for line in open(os.path.join(golden_dir, "bf16_sum_vectors.txt")):
        line = line.split("#")[0].strip()
        if line:
            lhs, rhs = line.split("->")
            out.append(([int(t, 16) for t in lhs.split()], int(rhs, 16)))
    return out


def test_golden_rounding_order_zero_nan_vectors(golden_dir):
    vecs = golden_vectors(golden_dir)
    assert len(vecs) >= 15
    for ins, exp in vecs:
        send = [np.array([v], np.uint16) for v in ins]
        out = oracle.allreduce_sum(send, "bf16")
        assert all(int(o[0]) == exp for o in out), (list(map(hex, ins)), hex(int(out[0][0])), hex(exp))
        rs = oracle.reducescatter_sum([np.repeat(s, len(ins)) for s in send], "bf16")
        assert all(int(o[0]) == exp for o in rs)


def test_bf16_rne_against_torch_cast():
    rng = np.random.default_rng(0)
    bits = rng.integers(0, 2**32, 200_000, dtype=np.uint64).astype(np.uint32)
    edge = np.array([0x3F808000, 0x3F818000, 0x3F808001, 0x3F807FFF, 0x7F7FFFFF, 0x7F800000, 0xFF800000,
                     0x00000001, 0x00008000, 0x00018000, 0x80008000, 0x7F7F8000, 0x477FE000], np.uint32)
    bits = np.concatenate([bits, edge])
    f = bits.view(np.float32)
    finite_or_inf = ~np.isnan(f)
    exp = bf16_bits(f)
    got = np.array([oracle.f32_to_bf16_rne(int(b)) for b in bits], np.uint16)
    assert (got[finite_or_inf] == exp[finite_or_inf]).all()
    assert (got[~finite_or_inf] == 0x7FFF).all()             # reading 13: canonical NaN


def test_f16_rne_against_numpy_cast():
    rng = np.random.default_rng(1)
    # exponents around half's range incl. subnormal and overflow regions
    e = rng.integers(127 - 30, 127 + 18, 200_000).astype(np.uint32)
    m = rng.integers(0, 2**23, 200_000).astype(np.uint32)
    m[::3] &= np.uint32(0x7FE000)                            # many exact ties / representables
    m[1::7] = (m[1::7] & np.uint32(0x7FE000)) | np.uint32(0x1000)
    s = rng.integers(0, 2, 200_000).astype(np.uint32) << np.uint32(31)
    bits = s | (e << np.uint32(23)) | m
    bits = np.concatenate([bits, np.array([0, 0x80000000, 0x7F800000, 0xFF800000, 0x477FE000, 0x477FF000,
                                           0x33000000, 0x33000001, 0x33800000, 0x387FC000, 0x387FE000, 1], np.uint32)])
    with np.errstate(over="ignore"):
        exp = bits.view(np.float32).astype(np.float16).view(np.uint16)
    got = np.array([oracle.f32_to_f16_rne(int(b)) for b in bits], np.uint16)
    assert (got == exp).all()
    # widening: every finite/inf half pattern survives f16 -> f32 -> f16 through an R=1 reduction
    allh = np.arange(65536, dtype=np.uint16)
    isn = np.isnan(allh.view(np.float16))
    out = oracle.allreduce_sum([allh], "f16")[0]
    assert (out[~isn] == allh[~isn]).all() and (out[isn] == 0x7FFF).all()


def test_R1_identity_all_bf16_patterns():
    allb = np.arange(65536, dtype=np.uint16)
    isn = np.isnan((allb.astype(np.uint32) << 16).view(np.float32))
    out = oracle.allreduce_sum([allb], "bf16")[0]
    assert (out[~isn] == allb[~isn]).all() and (out[isn] == 0x7FFF).all()


@pytest.mark.parametrize("R", [2, 3, 8, 16, 64])
def test_small_integer_sums_are_exact(R):
    rng = np.random.default_rng(R)
    n = 4096
    ints = rng.integers(-2, 3, (R, n))
    send = [bf16_bits(ints[k].astype(np.float32)) for k in range(R)]
    out = oracle.allreduce_sum(send, "bf16")
    exp = bf16_bits(ints.sum(axis=0).astype(np.float32))     # |sum| <= 128: exact in bf16
    got_val = bf16_to_f64(out[0]); exp_val = bf16_to_f64(exp)
    assert (got_val == exp_val).all()                        # value-equal (0 vs -0 not distinguished here)
    for o in out[1:]:
        assert o.tobytes() == out[0].tobytes()


def test_R2_and_fp32_reduce_to_numpy_float32_adds():
    a, b, c = (W.np_values(10_000, "f32", s) for s in (1, 2, 3))
    out = oracle.allreduce_sum([a, b], "f32")[0]
    assert out.tobytes() == (a + b).tobytes()                # one IEEE add: library routine
    assert oracle.allreduce_sum([b, a], "f32")[0].tobytes() == out.tobytes()   # commutative
    out3 = oracle.allreduce_sum([a, b, c], "f32")[0]
    assert out3.tobytes() == ((a + b) + c).astype(np.float32).tobytes()
    xa, xb = W.np_values(10_000, "bf16", 4), W.np_values(10_000, "bf16", 5)
    fa, fb = ((x.astype(np.uint32) << 16).view(np.float32) for x in (xa, xb))
    assert oracle.allreduce_sum([xa, xb], "bf16")[0].tobytes() == bf16_bits(fa + fb).tobytes()


def test_R2_f16_reduces_to_numpy_half_widen_add_narrow():
    """Direct pin of the oracle's f16 -> f32 widening (until now reached only through the 65 536-pattern round trip):
    numpy's float16 -> float32 cast is exact, float32 add is one IEEE add, float32 -> float16 rounds to nearest even.
    Includes subnormal halves, both zeros and +-65504; the sum of two finite halves never overflows binary32, and
    NaN/Inf inputs are excluded because the oracle canonicalises NaN while numpy keeps payloads."""
    rng = np.random.default_rng(12)
    xa = rng.integers(0, 1 << 16, 200_000).astype(np.uint16)
    xb = rng.integers(0, 1 << 16, 200_000).astype(np.uint16)
    edge = np.array([0x0000, 0x8000, 0x0001, 0x8001, 0x03FF, 0x0400, 0x7BFF, 0xFBFF, 0x3C00, 0xBC00], np.uint16)
    xa = np.concatenate([xa, np.repeat(edge, edge.size)])
    xb = np.concatenate([xb, np.tile(edge, edge.size)])
    finite = ((xa & 0x7C00) != 0x7C00) & ((xb & 0x7C00) != 0x7C00)
    xa, xb = np.ascontiguousarray(xa[finite]), np.ascontiguousarray(xb[finite])
    with np.errstate(over="ignore"):
        want = (xa.view(np.float16).astype(np.float32) + xb.view(np.float16).astype(np.float32)).astype(np.float16)
    got = oracle.allreduce_sum([xa, xb], "f16")[0]
    assert got.tobytes() == want.view(np.uint16).tobytes()


@pytest.mark.parametrize("R,std", [(8, 1.0), (16, 1e-3)])
def test_error_bound_against_fp64(R, std):
    n = 50_000
    send = [W.np_values(n, "bf16", 10 + k, std) for k in range(R)]
    out = bf16_to_f64(oracle.allreduce_sum(send, "bf16")[0])
    xs = np.stack([bf16_to_f64(s) for s in send])
    exact = xs.sum(axis=0)
    ulp = 2.0 ** (np.floor(np.log2(np.maximum(np.abs(out), 1e-300))) - 7)
    bound = (R - 1) * 2.0**-24 * np.abs(xs).sum(axis=0) + 0.5 * ulp + 2.0**-133
    assert (np.abs(out - exact) <= bound).all()


@pytest.mark.parametrize("dtype", ["bf16", "f32", "f16"])
def test_cross_api_invariants(dtype):
    R, n = 4, 1000
    std = 1.0
    send = [W.np_values(R * n, dtype, 20 + k, std) for k in range(R)]
    ar = oracle.allreduce_sum(send, dtype, nthreads=3)
    rs = oracle.reducescatter_sum(send, dtype, nthreads=2)
    for r in range(R):
        assert ar[r].tobytes() == ar[0].tobytes()
        assert rs[r].tobytes() == ar[0][r * n:(r + 1) * n].tobytes()
    sampled = oracle.reduce_samples(np.stack(send)[:, ::7], dtype)
    assert sampled.tobytes() == ar[0][::7].tobytes()


def test_fp32_nan_canonical_and_inf():
    nan_payload = np.array([0x7FC12345], np.uint32).view(np.float32)
    one = np.array([1.0], np.float32)
    assert oracle.allreduce_sum([nan_payload, one], "f32")[0].view(np.uint32)[0] == 0x7FFFFFFF
    assert oracle.allreduce_sum([nan_payload], "f32")[0].view(np.uint32)[0] == 0x7FFFFFFF
    inf = np.array([np.inf], np.float32)
    assert oracle.allreduce_sum([inf, one], "f32")[0][0] == np.inf
    assert oracle.allreduce_sum([inf, -inf], "f32")[0].view(np.uint32)[0] == 0x7FFFFFFF
    sub = np.array([1], np.uint32).view(np.float32)          # smallest fp32 subnormal, no FTZ
    assert oracle.allreduce_sum([sub, sub], "f32")[0].view(np.uint32)[0] == 2
