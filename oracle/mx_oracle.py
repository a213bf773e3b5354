"""CPU oracle of the block-scaled MXFP8 linear layer — TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/dit_oracle.py's header
for who may import it).  Plain and slow; shares no code with the CUDA path (it reuses oracle/fp8_oracle.py's E4M3 table and
rounding, which are pinned in tests/test_fp8_oracle.py).

What it is: SURVEY.md §8(f) item 2 ("block-scaled ... mxf8 GEMMs with the same oracle"), reading R43.  The paper does
not describe it; the format is the OCP Microscaling (MX) MXFP8 format, restated from its definition:
  * a block is 32 consecutive elements along K; it stores 32 E4M3 codes and ONE shared scale X in E8M0 (8-bit exponent, no
    sign, no mantissa): X = 2^(code - 127) for code 0..254, code 255 = NaN;  value of element i = X * e4m3(code_i).
  * quantisation of a block v (R43, the MX specification's conversion rule): amax = max |v_i| in fp32;
        shared_exp = floor(log2(amax)) - 8          (8 = exponent of E4M3's largest power of two, 256 <= 448 < 512)
    clamped to [-127, 127] (amax = 0: shared_exp = 0, code 127, X = 1);  X = 2^shared_exp;  code_i = e4m3(v_i / X) with
    round-to-nearest-even, saturating at +-448.  floor(log2(amax)) is the fp32 exponent of amax (subnormal amax: -127), so the
    decision is exact in fp32 on both sides, and v_i / X is an exact scaling by a power of two.  The scaled block maximum
    lies in [256, 512): values in (448, 512) saturate to 448 — a property of the rule, kept.
    linear_mx:  out[m, n] = sum over blocks b of  Xa[m, b] Xw[n, b] sum_{k in b} e4m3(Aq[m, k]) e4m3(Wq[n, k])  + bias[n]   (fp64)

Pins (tests/test_mx_oracle.py): the E8M0 table against torch's float8_e8m0fnu conversion (an independent library routine) and
hand values; the shared exponent on hand-made blocks (powers of two, just below / above a power of two, the saturating
band, zero block, tiny and huge blocks); |dequantised - v| bounds; linear_mx against a hand-computed example and against the
plain fp64 product of the DEQUANTISED operands (an independent formulation).
"""
from __future__ import annotations

import torch

from oracle import fp8_oracle as F8

BLOCK = 32


def e8m0_table() -> torch.Tensor:
    """fp64 [256]: 2^(code - 127); code 255 = NaN."""
    t = torch.tensor([2.0 ** (c - 127) for c in range(255)] + [float("nan")], dtype=torch.float64)
    return t


def shared_exponent(amax: torch.Tensor) -> torch.Tensor:
    """fp32 amax >= 0 -> int64 shared exponent by the rule in the header."""
    a = amax.to(torch.float32)
    bits = a.view(torch.int32).to(torch.int64)
    e = ((bits >> 23) & 0xFF) - 127                 # floor(log2(a)) for normal a; -127 for zero / subnormal
    sh = (e - 8).clamp(-127, 127)
    return torch.where(a > 0, sh, torch.zeros_like(sh))


def quantize_mx(x: torch.Tensor):
    """x [M, K] (K % 32 == 0; used as fp32) -> (codes uint8 [M, K], scales uint8 [M, K / 32] E8M0)."""
    M, K = x.shape
    assert K % BLOCK == 0
    v = x.to(torch.float32).reshape(M, K // BLOCK, BLOCK)
    sh = shared_exponent(v.abs().amax(dim=2))                           # [M, K/32]
    r = v.double() * torch.pow(torch.tensor(2.0, dtype=torch.float64), -sh.double())[:, :, None]   # exact: power of two
    codes = F8.round_to_e4m3(r.reshape(M, K))
    return codes, (sh + 127).to(torch.uint8)


def dequantize_mx(codes: torch.Tensor, scales: torch.Tensor) -> torch.Tensor:
    M, K = codes.shape
    X = e8m0_table()[scales.long()]                                     # [M, K/32]
    return (F8.decode(codes).reshape(M, K // BLOCK, BLOCK) * X[:, :, None]).reshape(M, K)


def linear_mx(Aq, sa, Wq, sw, bias=None) -> torch.Tensor:
    """out [M, N] fp64, block by block as in the header."""
    M, K = Aq.shape
    N = Wq.shape[0]
    a = F8.decode(Aq).reshape(M, K // BLOCK, BLOCK)
    w = F8.decode(Wq).reshape(N, K // BLOCK, BLOCK)
    Xa, Xw = e8m0_table()[sa.long()], e8m0_table()[sw.long()]
    out = torch.zeros(M, N, dtype=torch.float64)
    for b in range(K // BLOCK):
        out += (a[:, b] @ w[:, b].T) * Xa[:, b][:, None] * Xw[:, b][None, :]
    if bias is not None:
        out = out + bias.double()[None, :]
    return out
