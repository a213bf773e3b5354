"""CPU oracle of the fp8 (e4m3) linear layer — TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/dit_oracle.py's header for who
may import it).  Plain and slow; shares no code with the CUDA path.

What it is: SURVEY.md §8(f) item 2 ("fp8 ... GEMMs with the same oracle"), reading R42.  The paper does not
describe an fp8 path; the format is the OCP 8-bit floating point E4M3 ("e4m3fn": 1 sign, 4 exponent bits with bias 7, 3 mantissa
bits, no infinities, S.1111.111 = NaN, largest finite value 448), written out here from its definition:
    value(code) = (-1)^s * 2^(e-7) * (1 + m/8)   for e in 1..15   (e = 15, m = 7 is NaN)
                = (-1)^s * 2^-6   * (m/8)        for e = 0        (subnormals)
Quantisation of a row x (R42): amax = max|x| in fp32; inv = 448 / amax and scale = amax / 448, both fp32 divisions (1 when
amax = 0); r = x * inv, one fp32 multiplication; code = the e4m3 value nearest to r, ties to the even code, saturating at
+-448; `scale` is what the consumer multiplies back.  The decision is taken in fp32 on both sides
(the rule for "floating point decides an integer"); everything after it is exact: decode(code) in fp64.
    linear_fp8:  out[m, n] = a_scale[m] * w_scale[n] * sum_k decode(Aq[m, k]) decode(Wq[n, k]) + bias[n]     (fp64)

Pins (tests/test_fp8_oracle.py): the decode table and the rounding against torch's float8_e4m3fn conversion (an independent
library routine) on every code, on every midpoint between neighbouring values and on random values; hand values (0x38 = 1,
0x7E = 448, 0x01 = 2^-9); the row-scale rule on hand-made rows; linear_fp8 against a hand-computed 2 x 2 example; the
relative-error bound 2^-4 of round-to-nearest with 3 mantissa bits.
"""
from __future__ import annotations

import torch

E4M3_MAX = 448.0


def decode_table() -> torch.Tensor:
    """fp64 [256]: the value of every code (NaN for 0x7F / 0xFF), from the format's definition."""
    out = torch.empty(256, dtype=torch.float64)
    for code in range(256):
        s, e, m = code >> 7, (code >> 3) & 15, code & 7
        if e == 15 and m == 7:
            v = float("nan")
        elif e == 0:
            v = 2.0 ** -6 * (m / 8.0)
        else:
            v = 2.0 ** (e - 7) * (1.0 + m / 8.0)
        out[code] = -v if s else v
    return out


def decode(codes: torch.Tensor) -> torch.Tensor:
    """uint8 codes -> fp64 values."""
    return decode_table()[codes.long()]


def round_to_e4m3(r: torch.Tensor) -> torch.Tensor:
    """fp32 / fp64 values -> uint8 codes: nearest e4m3 value, ties to the even code, |r| > 448 saturates to 448 (code 0x7E)."""
    pos = decode_table()[:127]                      # codes 0..126: 0 .. 448, strictly increasing
    a = r.double().abs().clamp(max=E4M3_MAX)
    hi = torch.searchsorted(pos, a).clamp(max=126)  # first code whose value >= a
    lo = (hi - 1).clamp(min=0)
    d_hi, d_lo = pos[hi] - a, a - pos[lo]
    take_lo = (d_lo < d_hi) | ((d_lo == d_hi) & (lo % 2 == 0))
    code = torch.where(take_lo, lo, hi)
    neg = (r < 0) | ((r == 0) & (torch.signbit(r)))
    return (code + 128 * neg.long()).to(torch.uint8)


def quantize_rows(x: torch.Tensor):
    """x [M, K] (any float dtype; used as fp32) -> (codes uint8 [M, K], scale fp32 [M]) by the rule in the header."""
    xf = x.to(torch.float32)
    amax = xf.abs().amax(dim=1)
    m = torch.tensor(E4M3_MAX, dtype=torch.float32)
    scale = torch.where(amax > 0, amax / m, torch.ones_like(amax))       # fp32 divisions (IEEE, round to nearest)
    inv = torch.where(amax > 0, m / amax, torch.ones_like(amax))
    r = xf * inv[:, None]                                                # one fp32 multiplication per element
    return round_to_e4m3(r), scale


def linear_fp8(Aq, a_scale, Wq, w_scale, bias=None) -> torch.Tensor:
    """out [M, N] fp64 = (decode(Aq) decode(Wq)^T) * a_scale[:, None] * w_scale[None, :] + bias."""
    acc = decode(Aq) @ decode(Wq).T
    out = acc * a_scale.double()[:, None] * w_scale.double()[None, :]
    if bias is not None:
        out = out + bias.double()[None, :]
    return out
