"""Seeded synthetic input generators for the five BASELINE.json configs.

This module serves BOTH the CUDA path's tests/bench and the oracle's tests.  It
holds none of the method's arithmetic: it only draws count matrices and payload
values.  No offsets, no transposes, no sums, no rounding rules live here (the
fp32 -> bf16 cast of *inputs* is numpy/torch's own cast; the bytes it produces,
not the generator, are the contract: both sides consume the same buffers).

Recipes (SURVEY.md section 8(c.3) readings 17-20, section 8(d) table; the paper's traffic
shapes are PAPER.md L90/L369/L471 (MoE dispatch, < 128 KB per peer), L387
(skewed expert load) and L337/L373 (gradient AllReduce up to 256M messages)):

  cfg1  AllToAllv  R=4   rows of 128 bf16, C = default_rng(0).integers(0,257,(4,4)) rows
  cfg2  AllReduce  R=8   4,194,304 bf16 per rank, N(0,1), seed 1
  cfg3  AllToAllv  R=64  16,384 tokens/rank x 5120 bf16, top-1 over 128 experts,
                         Zipf(1.1) popularity p_e ~ (e+1)^-1.1, one multinomial per
                         source rank from default_rng(2), expert e lives on rank e//2
  cfg4  ReduceScatter R=16, 268,435,456 bf16 per rank, N(0, std 1e-3), seed 3
  cfg5  AllToAllv  R=128 rows of 7168 bf16, counts default_rng(4).integers(0,9) then an
                         independent Bernoulli(1/2) mask forces pairs to zero
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

BF16 = "bf16"
F32 = "f32"
F16 = "f16"
U8 = "u8"

ELEM_SIZE = {BF16: 2, F32: 4, F16: 2, U8: 1}


@dataclass(frozen=True)
class A2AConfig:
    name: str
    R: int
    width: int          # elements per row (token hidden size)
    dtype: str
    seed: int
    rows: np.ndarray    # (R, R) int64 rows sent s -> d

    @property
    def counts(self) -> np.ndarray:
        """C[s][d] in ELEMENTS of dtype (rows x width), the unit the C ABI takes."""
        return (self.rows * self.width).astype(np.int64)


@dataclass(frozen=True)
class ReduceConfig:
    name: str
    kind: str           # "allreduce" | "reducescatter"
    R: int
    count: int          # elements per rank INPUT
    dtype: str
    seed: int
    std: float


def cfg1_rows() -> np.ndarray:
    return np.random.default_rng(0).integers(0, 257, (4, 4)).astype(np.int64)


def cfg3_rows(R: int = 64, tokens: int = 16384, experts: int = 128, s: float = 1.1,
              seed: int = 2) -> np.ndarray:
    p = (np.arange(experts) + 1.0) ** (-s)
    p /= p.sum()
    rng = np.random.default_rng(seed)
    per_expert = np.stack([rng.multinomial(tokens, p) for _ in range(R)])
    per_rank = experts // R
    return per_expert.reshape(R, R, per_rank).sum(-1).astype(np.int64)


def cfg5_rows(R: int = 128, seed: int = 4) -> np.ndarray:
    rng = np.random.default_rng(seed)
    c = rng.integers(0, 9, (R, R))
    mask = rng.random((R, R)) < 0.5
    c[mask] = 0
    return c.astype(np.int64)


def a2a_config(idx: int) -> A2AConfig:
    if idx == 1:
        return A2AConfig("cfg1_a2a_R4", 4, 128, BF16, 0, cfg1_rows())
    if idx == 3:
        return A2AConfig("cfg3_moe_dispatch_R64", 64, 5120, BF16, 2, cfg3_rows())
    if idx == 5:
        return A2AConfig("cfg5_small_msg_R128", 128, 7168, BF16, 4, cfg5_rows())
    raise ValueError(idx)


def reduce_config(idx: int) -> ReduceConfig:
    if idx == 2:
        return ReduceConfig("cfg2_allreduce_R8", "allreduce", 8, 4_194_304, BF16, 1, 1.0)
    if idx == 4:
        return ReduceConfig("cfg4_reducescatter_R16", "reducescatter", 16, 268_435_456, BF16, 3, 1e-3)
    raise ValueError(idx)


def scaled_a2a(cfg: A2AConfig, row_div: int, name: str | None = None) -> A2AConfig:
    """Same count STRUCTURE with every row count divided by row_div (floor): the
    bounded sample the CPU baseline and the mid-size parity tests run."""
    return A2AConfig(name or f"{cfg.name}_div{row_div}", cfg.R, cfg.width, cfg.dtype, cfg.seed,
                     (cfg.rows // row_div).astype(np.int64))


# --------------------------------------------------------------------------- values

def np_values(n: int, dtype: str, seed: int, std: float = 1.0) -> np.ndarray:
    """CPU generator (small cases / CPU-only tests).  bf16/f16 come back as uint16 bit
    patterns, f32 as float32, u8 as uint8."""
    rng = np.random.default_rng(seed)
    if dtype == U8:
        return rng.integers(0, 256, n, dtype=np.uint8)
    x = (rng.standard_normal(n, dtype=np.float32) * np.float32(std)).astype(np.float32)
    if dtype == F32:
        return x
    if dtype == F16:
        return x.astype(np.float16).view(np.uint16)
    if dtype == BF16:
        import torch  # torch's own cast, used only to make input bytes
        return torch.from_numpy(x).to(torch.bfloat16).view(torch.int16).numpy().view(np.uint16).copy()
    raise ValueError(dtype)


def torch_dtype(dtype: str):
    import torch
    return {BF16: torch.bfloat16, F32: torch.float32, F16: torch.float16, U8: torch.uint8}[dtype]


def torch_values(n: int, dtype: str, seed: int, std: float = 1.0, device="cuda", chunk: int = 1 << 28):
    """Device generator for the big configs: fp32 normal * std, cast to dtype, in chunks so
    the fp32 temporary stays small."""
    import torch
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    td = torch_dtype(dtype)
    out = torch.empty(n, dtype=td, device=device)
    for lo in range(0, n, chunk):
        m = min(chunk, n - lo)
        if dtype == U8:
            out[lo:lo + m] = torch.randint(0, 256, (m,), generator=g, device=device, dtype=torch.uint8)
        else:
            t = torch.randn(m, generator=g, device=device, dtype=torch.float32)
            if std != 1.0:
                t.mul_(std)
            out[lo:lo + m] = t.to(td)
    return out


def tagged_payload_u32(s: int, n: int) -> np.ndarray:
    """Self-describing payload: element j of rank s's send buffer is (s << 24) | j
    (SURVEY.md section 8(c.4)).  A label, not arithmetic of the method."""
    assert n < (1 << 24) and s < 256
    return (np.uint32(s) << np.uint32(24)) | np.arange(n, dtype=np.uint32)


def dynamic_moe_metadata(R: int = 64, tokens: int = 256, experts: int = 128, width: int = 5120, s: float = 1.1,
                         seed: int = 5, redundant_hot_expert: bool = True):
    """Metadata of an inference-shaped AllToAllvDynamic call (Table 3: batch
    128/256 tokens per rank): per source rank one multinomial(tokens, Zipf(s)) over the experts gives
    sendSplitLengths (rows x width elements, sorted by expert id, MetaShuffling L699); rank d hosts experts
    [d*E/R, (d+1)*E/R) and, if asked, the last rank also hosts a redundant copy of the hottest expert 0
    (duplicated experts, L437).  -> (split_lengths (R,E), indices (R,maxIndices), block_lens (R,R), maxBlockLen)."""
    p = (np.arange(experts) + 1.0) ** (-s)
    p /= p.sum()
    rng = np.random.default_rng(seed)
    rows = np.stack([rng.multinomial(tokens, p) for _ in range(R)]).astype(np.int64)
    per = experts // R
    J = per + (1 if redundant_hot_expert else 0)
    bl = np.full((R, R), per, np.int64)
    if redundant_hot_expert:
        bl[:, R - 1] = per + 1
    lst = []
    for d in range(R):
        lst += list(range(d * per, (d + 1) * per))
        if redundant_hot_expert and d == R - 1:
            lst.append(0)
    idx = np.tile(np.array(lst, np.int64), (R, 1))
    return rows * width, idx, bl, J


def topk_routing(R: int, T: int, k: int, experts: int, seed: int, s: float = 1.1):
    """Synthetic top-k router + MetaShuffling order: every token of every rank draws k
    DISTINCT experts (Zipf(s) popularity, Gumbel top-k), copies are sorted by (expert id, token id) into the
    virtual send buffer.  -> (pos (R, T, k) int32: row of copy j of token t in rank s's sorted buffer;
    Crows (R, R) int64: rows sent s -> d, expert e living on rank e // (experts // R)).
    A labelling of the input, not arithmetic of the method (no offsets, no sums of payload)."""
    rng = np.random.default_rng(seed)
    logp = -s * np.log(np.arange(experts) + 1.0)
    per = experts // R
    pos = np.empty((R, T, k), np.int32)
    C = np.zeros((R, R), np.int64)
    for r in range(R):
        g = rng.gumbel(size=(T, experts)) + logp
        top = np.argsort(-g, axis=1)[:, :k]                       # router order j = 0..k-1
        flat_e = top.reshape(-1)
        order = np.argsort(flat_e * (T * k) + np.arange(T * k), kind="stable")   # by expert, then (token, j)
        p = np.empty(T * k, np.int64)
        p[order] = np.arange(T * k)
        pos[r] = p.reshape(T, k).astype(np.int32)
        C[r] = np.bincount(flat_e // per, minlength=R)
    return pos, C
