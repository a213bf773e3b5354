"""Pins of oracle/fp8_oracle.py (no GPU): the e4m3 table and rounding against torch's float8_e4m3fn conversion (an independent
library routine), hand values from the format definition, the row-scale rule, a hand-computed linear layer, the error bound."""
import math

import torch

from oracle import fp8_oracle as F


def test_decode_table_hand_values_and_library():
    t = F.decode_table()
    # hand values from the definition: 1 sign, 4 exponent bits (bias 7), 3 mantissa bits
    assert t[0x00] == 0.0 and t[0x38] == 1.0 and t[0x40] == 2.0 and t[0x3C] == 1.5
    assert t[0x7E] == 448.0 and t[0xFE] == -448.0            # largest finite: 2^8 * 1.75
    assert t[0x01] == 2.0 ** -9 and t[0x07] == 7 * 2.0 ** -9  # subnormals: m/8 * 2^-6
    assert t[0x08] == 2.0 ** -6                               # smallest normal
    assert math.isnan(float(t[0x7F])) and math.isnan(float(t[0xFF]))
    lib = torch.arange(256, dtype=torch.uint8).view(torch.float8_e4m3fn).to(torch.float64)
    ok = torch.isnan(lib) == torch.isnan(t)
    assert bool(ok.all())
    fin = ~torch.isnan(t)
    assert torch.equal(lib[fin], t[fin])
    pos = t[:127]
    assert bool((pos[1:] > pos[:-1]).all())


def _lib_codes(r):
    return r.to(torch.float32).to(torch.float8_e4m3fn).view(torch.uint8)


def test_rounding_matches_library_on_codes_midpoints_and_random():
    t = F.decode_table()
    pos = t[:127]
    exact = torch.cat([pos, -pos[1:]]).to(torch.float32)
    assert torch.equal(F.round_to_e4m3(exact), _lib_codes(exact))
    assert torch.equal(F.decode(F.round_to_e4m3(exact)), exact.double())          # every value is a fixed point
    mid = ((pos[1:] + pos[:-1]) / 2).to(torch.float32)                             # exact in fp32: ties
    mids = torch.cat([mid, -mid])
    got = F.round_to_e4m3(mids)
    assert torch.equal(got, _lib_codes(mids))
    assert bool(((got & 1) == 0).all())                                            # ties go to the even code
    eps = torch.cat([torch.nextafter(mid, torch.tensor(float("inf"))), torch.nextafter(mid, torch.tensor(0.0))])
    assert torch.equal(F.round_to_e4m3(eps), _lib_codes(eps))
    g = torch.Generator().manual_seed(3)
    r = torch.cat([torch.randn(20000, generator=g) * s for s in (1e-3, 0.02, 1.0, 30.0, 150.0)]).clamp(-448, 448)
    assert torch.equal(F.round_to_e4m3(r), _lib_codes(r))
    # saturation is this oracle's rule (the library conversion has no saturating mode): beyond 448 -> +-448
    big = torch.tensor([449.0, 464.0, 1e6, -500.0])
    assert F.round_to_e4m3(big).tolist() == [0x7E, 0x7E, 0x7E, 0xFE]
    # signed zero keeps its sign bit
    assert F.round_to_e4m3(torch.tensor([0.0, -0.0])).tolist() == [0x00, 0x80]


def test_round_to_nearest_error_bound():
    g = torch.Generator().manual_seed(5)
    r = (torch.rand(50000, generator=g) * 2 - 1) * 448
    d = F.decode(F.round_to_e4m3(r))
    normal = r.abs() >= 2.0 ** -6
    assert bool(((d - r.double()).abs()[normal] <= r.double().abs()[normal] * 2.0 ** -4).all())   # half an ulp of 3 mantissa bits
    assert bool(((d - r.double()).abs()[~normal] <= 2.0 ** -10).all())                             # half a subnormal step


def test_quantize_rows_scale_rule():
    x = torch.tensor([[0.5, -2.0, 1.0, 0.0], [0.0, 0.0, 0.0, 0.0], [3.0, 448.0, -7.0, 1e-4]])
    q, s = F.quantize_rows(x)
    assert s.dtype == torch.float32 and q.dtype == torch.uint8
    assert s.tolist() == [float(torch.tensor(2.0) / torch.tensor(448.0)), 1.0, 1.0]
    # row 0: inv = 448 / 2 = 224 exactly; x * inv = 112, -448, 224, 0 -> all representable
    assert torch.equal(F.decode(q[0]), torch.tensor([112.0, -448.0, 224.0, 0.0], dtype=torch.float64))
    assert q[1].tolist() == [0, 0, 0, 0]
    # row 2 (amax = 448: inv = scale = 1): 3 -> 3, 448 -> 448, -7 -> -7, 1e-4 -> 0 (below half the smallest subnormal 2^-10)
    assert torch.equal(F.decode(q[2]), torch.tensor([3.0, 448.0, -7.0, 0.0], dtype=torch.float64))
    # a row whose scale is not a power of two: inv = fp32(448 / 3), codes of x * inv by hand
    q3, s3 = F.quantize_rows(torch.tensor([[3.0, 1.0, -0.01, 2.0]]))
    inv3 = float(torch.tensor(448.0) / torch.tensor(3.0))                       # 149.33333...
    assert s3.tolist() == [float(torch.tensor(3.0) / torch.tensor(448.0))]
    # 3 * inv = 448 -> 448; 1 * inv = 149.33 -> between 144 and 160: 144; -0.01 * inv = -1.4933 -> between 1.375 and 1.5: -1.5;
    # 2 * inv = 298.67 -> between 288 and 320: 288
    assert 447.9 < 3 * inv3 < 448.1
    assert F.decode(q3[0]).tolist() == [448.0, 144.0, -1.5, 288.0]
    # the row maximum always lands on +-448
    g = torch.Generator().manual_seed(9)
    y = torch.randn(64, 96, generator=g).to(torch.bfloat16)
    qy, sy = F.quantize_rows(y)
    assert bool((F.decode(qy).abs().amax(dim=1) == 448.0).all())
    back = F.decode(qy) * sy.double()[:, None]
    err = (back - y.double()).abs()
    assert bool((err <= y.double().abs() * 2.0 ** -4 + sy.double()[:, None] * 2.0 ** -10 + 1e-12).all())


def test_linear_fp8_by_hand():
    # A = [[1, 2], [-0.5, 4]] with row scales (2, 0.5); W = [[1.5, -1], [0.25, 8]] with row scales (4, 1); bias (10, -1)
    t = F.decode_table()
    code = {float(v): c for c, v in enumerate(t.tolist()) if not math.isnan(v)}
    Aq = torch.tensor([[code[1.0], code[2.0]], [code[-0.5], code[4.0]]], dtype=torch.uint8)
    Wq = torch.tensor([[code[1.5], code[-1.0]], [code[0.25], code[8.0]]], dtype=torch.uint8)
    out = F.linear_fp8(Aq, torch.tensor([2.0, 0.5]), Wq, torch.tensor([4.0, 1.0]), torch.tensor([10.0, -1.0]))
    # row 0: dots (1*1.5 + 2*-1, 1*0.25 + 2*8) = (-0.5, 16.25) -> * 2 * (4, 1) = (-4, 32.5) + bias = (6, 31.5)
    # row 1: dots (-0.75 - 4, -0.125 + 32) = (-4.75, 31.875) -> * 0.5 * (4, 1) = (-9.5, 15.9375) + bias = (0.5, 14.9375)
    assert out.tolist() == [[6.0, 31.5], [0.5, 14.9375]]
    assert out.dtype == torch.float64
