"""GPU parity of the block-scaled MXFP8 linear layer (R43) against oracle/mx_oracle.py: codes
and E8M0 block scales bit for bit (byte work), the block-scaled GEMM element by element on the same codes."""
import math

import pytest
import torch

from oracle import dit_oracle as O
from oracle import mx_oracle as MX
from paper_2606_13501_b200 import binding as B
from paper_2606_13501_b200 import synth
from util import check, check_rounding, errors

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def rnd(name, shape, dtype, std=1.0, seed=23):
    return synth.normal(seed, name, shape, std=std, dtype=dtype, device=DEV)


def _wide_range(x, seed_name):
    """Rows and blocks of very different magnitude (the case block scaling exists for)."""
    M, K = x.shape
    g = synth.normal(29, seed_name, (M, K // 32), dtype=torch.float32, device=DEV)
    return (x.float() * torch.exp2(torch.round(g * 6)).repeat_interleave(32, dim=1)).to(x.dtype)


@pytest.mark.parametrize("dtype", [torch.bfloat16, torch.float32])
@pytest.mark.parametrize("M,K", [(1, 32), (37, 224), (300, 3072), (1000, 4096 + 128)])
def test_quantize_mx_codes_and_scales_are_bit_exact(lib, dtype, M, K):
    x = _wide_range(rnd("x", (M, K), dtype, std=2.0), "g")
    if M > 2:
        x[1].zero_()                                  # zero blocks: scale code 127, codes 0
        x[2, :4] = torch.tensor([1.999, -2.0, 447.0, 3.0e38], dtype=dtype, device=DEV)      # saturating band, huge block
        x[0, 32:36] = torch.tensor([1e-40, -1e-42, 0.0, -0.0], dtype=dtype, device=DEV)     # subnormals, signed zeros
        x[0, 36:64] = 0
    q, s = B.dit_quantize_mxfp8(x)
    torch.cuda.synchronize()
    q_ref, s_ref = MX.quantize_mx(x.cpu())
    assert torch.equal(s.cpu(), s_ref), f"{int((s.cpu() != s_ref).sum())} block scales differ"
    assert torch.equal(q.cpu(), q_ref), f"{int((q.cpu() != q_ref).sum())} codes differ"


GEMM_SHAPES = [(128, 128, 128), (300, 520, 256), (77, 1032, 4096), (1000, 256, 1152), (513, 3072, 3072)]


@pytest.mark.parametrize("M,N,K", GEMM_SHAPES)
@pytest.mark.parametrize("epi", [B.EPI_BIAS_F32, B.EPI_BIAS, B.EPI_BIAS_GELU])
def test_linear_mx_against_oracle_on_the_same_codes(lib, M, N, K, epi):
    A = _wide_range(rnd("A", (M, K), torch.bfloat16), "ga")
    W = _wide_range(rnd("W", (N, K), torch.bfloat16, std=1.0 / math.sqrt(K)), "gw")
    b = rnd("b", (N,), torch.bfloat16, std=0.5)
    Aq, sa = B.dit_quantize_mxfp8(A)
    Wq, sw = B.dit_quantize_mxfp8(W)
    got = B.dit_linear_mxfp8(Aq, sa, Wq, sw, b, epi)
    torch.cuda.synchronize()
    Aq_r, sa_r = MX.quantize_mx(A.cpu())
    Wq_r, sw_r = MX.quantize_mx(W.cpu())
    assert torch.equal(Aq.cpu(), Aq_r) and torch.equal(sa.cpu(), sa_r) and torch.equal(Wq.cpu(), Wq_r) and torch.equal(sw.cpu(), sw_r)
    ref = MX.linear_mx(Aq_r, sa_r, Wq_r, sw_r, b.cpu())
    if epi == B.EPI_BIAS_GELU:
        ref = O.gelu_tanh(ref)
    if epi == B.EPI_BIAS_F32:
        check(got, ref, torch.float32, f"linear_mx f32 {M}x{N}x{K}", rel=1e-5, maxabs=1e-4)
    else:
        check(got, ref, torch.bfloat16, f"linear_mx {M}x{N}x{K}", rel=3e-3, maxabs=float("inf"))   # heavy-tailed output: the element-wise bound below replaces max-abs / RMS
        check_rounding(got, ref, f"linear_mx {M}x{N}x{K}")


@pytest.mark.parametrize("M,N,K", [(256, 256, 512), (300, 520, 384), (600, 456, 1024)])   # K % 512 == 0: the CTA-pair kernel
def test_linear_mx_scales_are_applied_per_block_and_per_row(lib, M, N, K):
    """A wrong scale layout in tensor memory (row group, K slice or operand swapped) cannot pass: every (row, block) of A and of
    W gets its own power-of-two scale while all codes are the SAME constant, so out[m, n] = c^2 32 sum_b Xa[m, b] Xw[n, b]."""
    code_one = 0x38                                                      # e4m3 1.0
    Aq = torch.full((M, K), code_one, dtype=torch.uint8, device=DEV)
    Wq = torch.full((N, K), code_one, dtype=torch.uint8, device=DEV)
    ea = (torch.arange(M, device=DEV)[:, None] % 7) + (torch.arange(K // 32, device=DEV)[None, :] % 5) - 5
    ew = (torch.arange(N, device=DEV)[:, None] % 3) * 2 - (torch.arange(K // 32, device=DEV)[None, :] % 4)
    sa, sw = (ea + 127).to(torch.uint8), (ew + 127).to(torch.uint8)
    got = B.dit_linear_mxfp8(Aq, sa, Wq, sw, None, B.EPI_BIAS_F32)
    torch.cuda.synchronize()
    want = 32.0 * (torch.exp2(ea.double()) @ torch.exp2(ew.double()).T)
    assert torch.equal(got.double().cpu(), want.cpu())                   # sums of few powers of two: exact in fp32
    ref = MX.linear_mx(Aq.cpu(), sa.cpu(), Wq.cpu(), sw.cpu())
    assert torch.equal(ref, want.cpu())


def test_linear_mx_bad_arguments(lib):
    A, W = rnd("A2", (64, 256), torch.bfloat16), rnd("W2", (128, 256), torch.bfloat16)
    Aq, sa = B.dit_quantize_mxfp8(A)
    Wq, sw = B.dit_quantize_mxfp8(W)
    out = B.dit_linear_mxfp8(Aq[:0], sa[:0], Wq, sw)                     # M = 0
    assert out.shape == (0, 128)
    with pytest.raises(B.DitError):                                      # K not a multiple of 128
        B.dit_linear_mxfp8(Aq[:, :224].contiguous(), sa[:, :7].contiguous(), Wq[:, :224].contiguous(), sw[:, :7].contiguous())
    with pytest.raises(B.DitError):
        B.dit_linear_mxfp8(Aq, None, Wq, sw)
    with pytest.raises(B.DitError):                                      # K not a multiple of 32
        B.dit_quantize_mxfp8(A[:, :40].contiguous())


def test_mx_layer_error_against_the_unquantised_product(lib):
    """Block scaling keeps the e4m3 element error (~2^-4 relative per element) but removes the dynamic-range problem: on
    operands whose blocks differ by 2^+-18 in magnitude the MX layer stays at a few 1e-2 rel-L2 of the exact product where
    one scale per row (dit_linear_fp8, R42) loses the small blocks entirely."""
    M, N, K = 256, 512, 2048
    A = _wide_range(rnd("A3", (M, K), torch.bfloat16), "ga3")
    W = rnd("W3", (N, K), torch.bfloat16, std=1.0 / math.sqrt(K))
    exact = A.double().cpu() @ W.double().cpu().T
    got = B.dit_linear_mxfp8(*B.dit_quantize_mxfp8(A), *B.dit_quantize_mxfp8(W), None, B.EPI_BIAS_F32)
    e_mx, _ = errors(got, exact)
    assert 1e-2 < e_mx < 6e-2, e_mx
