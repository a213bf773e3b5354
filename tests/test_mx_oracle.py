"""Pins of oracle/mx_oracle.py (no GPU): E8M0 against torch's float8_e8m0fnu (an independent library routine), the shared
exponent rule on hand-made blocks, dequantisation error bounds, and the block-scaled product against a hand-computed example
and against the plain product of the dequantised operands."""
import math

import torch

from oracle import fp8_oracle as F8
from oracle import mx_oracle as MX


def test_e8m0_table_hand_values_and_library():
    t = MX.e8m0_table()
    assert t[127] == 1.0 and t[128] == 2.0 and t[126] == 0.5 and t[0] == 2.0 ** -127 and t[254] == 2.0 ** 127
    assert math.isnan(float(t[255]))
    lib = torch.arange(256, dtype=torch.uint8).view(torch.float8_e8m0fnu).to(torch.float32).double()
    assert torch.equal(lib[:255], t[:255]) and bool(torch.isnan(lib[255]))


def _block(vals):
    v = torch.zeros(1, 32)
    v[0, :len(vals)] = torch.tensor(vals)
    return v


def test_shared_exponent_rule_by_hand():
    # amax = 1 -> floor(log2) = 0 -> shared_exp = -8 -> code 119; 1 / 2^-8 = 256 = e4m3 code of 256
    q, s = MX.quantize_mx(_block([1.0, -0.5, 0.75]))
    assert s.tolist() == [[119]]
    assert F8.decode(q[0, :3]).tolist() == [256.0, -128.0, 192.0]
    # just below a power of two: amax = 1.999 -> still exponent 0; 1.999 * 256 = 511.7 saturates to 448 (the rule's band)
    q, s = MX.quantize_mx(_block([1.999, 1.7]))
    assert s.tolist() == [[119]]
    assert F8.decode(q[0, :2]).tolist() == [448.0, 448.0]       # 1.7 * 256 = 435.2 -> nearest of {416, 448} = 448
    # amax = 2 -> exponent 1 -> shared_exp -7 -> code 120; 2 / 2^-7 = 256
    q, s = MX.quantize_mx(_block([2.0, 1.0]))
    assert s.tolist() == [[120]] and F8.decode(q[0, :2]).tolist() == [256.0, 128.0]
    # zero block: X = 1 (code 127), codes 0
    q, s = MX.quantize_mx(torch.zeros(1, 32))
    assert s.tolist() == [[127]] and int(q.sum()) == 0
    # huge block: 2^127 -> shared_exp 119 -> code 246; tiny block: 2^-140 (fp32 subnormal) -> clamped to -127 -> code 0
    q, s = MX.quantize_mx(_block([2.0 ** 127]))
    assert s.tolist() == [[246]] and F8.decode(q[0, :1]).tolist() == [256.0]
    q, s = MX.quantize_mx(_block([2.0 ** -140]))
    assert s.tolist() == [[0]]
    assert F8.decode(q[0, :1]).tolist() == [0.0]     # 2^-140 / 2^-127 = 2^-13, below half of E4M3's smallest subnormal (2^-10)


def test_blocks_are_independent_and_two_blocks_per_row():
    x = torch.cat([_block([1.0, 0.25]), _block([64.0, -3.0])], dim=1)     # one row, two blocks
    q, s = MX.quantize_mx(x)
    assert s.tolist() == [[119, 125]]                                      # 64 -> exponent 6 -> -2 -> 125
    assert F8.decode(q[0, [0, 1, 32, 33]]).tolist() == [256.0, 64.0, 256.0, -12.0]
    back = MX.dequantize_mx(q, s)
    assert torch.equal(back, x.double())                                   # all exactly representable


def test_dequantisation_error_bound():
    g = torch.Generator().manual_seed(4)
    x = (torch.randn(64, 256, generator=g) * torch.exp(torch.randn(64, 1, generator=g) * 3)).to(torch.bfloat16)
    q, s = MX.quantize_mx(x)
    back = MX.dequantize_mx(q, s)
    X = MX.e8m0_table()[s.long()].repeat_interleave(32, dim=1)
    xd = x.double()
    sat = xd.abs() > 448 * X                                               # the saturating band (448, 512) X
    err = (back - xd).abs()
    assert bool((err[~sat] <= xd.abs()[~sat] * 2.0 ** -4 + X[~sat] * 2.0 ** -10).all())
    assert bool((back.abs()[sat] == 448 * X[sat]).all()) and bool((xd.abs()[sat] < 512 * X[sat]).all())
    # the scaled block maximum lies in [256, 512)
    amax = xd.abs().reshape(64, 8, 32).amax(dim=2)
    Xb = MX.e8m0_table()[s.long()]
    assert bool(((amax / Xb >= 256) & (amax / Xb < 512)).all())


def test_linear_mx_by_hand_and_against_dequantised_product():
    # one row of A and one of W, two blocks each, by hand:
    #   A: block 0 X = 2 (code 128), values e4m3 (1, 2, 0...);  block 1 X = 0.5 (code 126), values (4, 0...)
    #   W: block 0 X = 1 (code 127), values (3, -1, 0...);      block 1 X = 4 (code 129), values (0.5, 0...)
    t = F8.decode_table()
    code = {float(v): c for c, v in enumerate(t.tolist()) if not math.isnan(v)}
    Aq = torch.zeros(1, 64, dtype=torch.uint8); Wq = torch.zeros(1, 64, dtype=torch.uint8)
    Aq[0, 0], Aq[0, 1], Aq[0, 32] = code[1.0], code[2.0], code[4.0]
    Wq[0, 0], Wq[0, 1], Wq[0, 32] = code[3.0], code[-1.0], code[0.5]
    sa, sw = torch.tensor([[128, 126]], dtype=torch.uint8), torch.tensor([[127, 129]], dtype=torch.uint8)
    out = MX.linear_mx(Aq, sa, Wq, sw, torch.tensor([0.25]))
    # block 0: 2 * 1 * (1*3 + 2*-1) = 2;  block 1: 0.5 * 4 * (4 * 0.5) = 4;  + 0.25
    assert out.tolist() == [[6.25]]
    g = torch.Generator().manual_seed(8)
    A = torch.randn(24, 128, generator=g).to(torch.bfloat16); W = (torch.randn(40, 128, generator=g) * 0.1).to(torch.bfloat16)
    b = torch.randn(40, generator=g).to(torch.bfloat16)
    qa, sa = MX.quantize_mx(A); qw, sw = MX.quantize_mx(W)
    want = MX.dequantize_mx(qa, sa) @ MX.dequantize_mx(qw, sw).T + b.double()
    assert torch.allclose(MX.linear_mx(qa, sa, qw, sw, b), want, rtol=1e-13, atol=1e-13)
