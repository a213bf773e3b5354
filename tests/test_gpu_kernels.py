"""GPU parity, kernel level: each C-ABI building block of the step against the CPU oracle on the same
seeded inputs, element by element (sizes span several tiles and a ragged tail; edge cases included)."""
import math

import pytest
import torch

from oracle import dit_oracle as O
from paper_2606_13501_b200 import binding as B
from paper_2606_13501_b200 import synth
from util import check, check_rounding, errors

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
DTYPES = [torch.float32, torch.bfloat16]


def rnd(name, shape, dtype, std=1.0, mean=0.0, seed=3):
    return synth.normal(seed, name, shape, std=std, mean=mean, dtype=dtype, device=DEV)


# ------------------------------------------------------------------------------ GEMV (t-MLP, modulation)
@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("R,N,K,silu", [(1, 256, 256, False), (1, 1030, 3072, True), (3, 517, 512, True),
                                         (6, 96, 1024, True), (8, 40, 256, False)])
def test_gemv(lib, dtype, R, N, K, silu):
    x = rnd("in", (R, K), torch.float32)
    W, b = rnd("W", (N, K), dtype, std=0.05), rnd("b", (N,), dtype, std=0.05)
    got = B.dit_gemv(x, W, b, silu_input=silu)
    xin = x.double().cpu()
    ref = O.linear(O.silu(xin) if silu else xin, W.cpu(), b.cpu())
    check(got, ref, torch.float32, f"gemv {dtype}", rel=2e-6, maxabs=2e-5)


# ------------------------------------------------------------------------------ adaLN
@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("T,D", [(1, 256), (37, 256), (301, 3072), (130, 5120), (66, 1024)])
@pytest.mark.parametrize("fused", [False, True])
def test_adaln(lib, dtype, T, D, fused):
    x = rnd("x", (T, D), torch.float32, std=2.0, mean=0.3)
    mod = rnd("mod", (1, 3 * D), torch.float32, std=0.3)
    h = rnd("h", (T, D), dtype) if fused else None
    xg = x.clone()
    y = B.dit_adaln(xg, dtype, h=h, gate=mod[:, 2 * D:] if fused else None, shift=mod[:, :D], scale=mod[:, D:2 * D],
                    mod_stride=3 * D)
    xr = x.double().cpu()
    m = mod.double().cpu()[0]
    if fused:
        xr = xr + m[2 * D:] * h.double().cpu()
        check(xg, xr, torch.float32, "adaln x update", rel=1e-6, maxabs=1e-5)
    else:
        assert torch.equal(xg, x)
    ref = O.modulate(xr, m[:D], m[D:2 * D], 1e-6)
    if dtype == torch.float32:
        check(y, ref, dtype, "adaln y", rel=2e-6, maxabs=2e-5)
    else:   # the only bf16 error is the output rounding: bound it element-wise (outliers of |y| ~ 8 RMS exist)
        check(y, ref, dtype, "adaln y", rel=3e-3, maxabs=6e-2)
        check_rounding(y, ref, "adaln y")


@pytest.mark.parametrize("dtype", DTYPES)
def test_adaln_varlen_requests_and_null_modulation(lib, dtype):
    T, D, R = 75, 512, 3
    cu = torch.tensor([0, 20, 21, 75], dtype=torch.int32, device=DEV)
    x = rnd("x", (T, D), torch.float32)
    mod = rnd("mod", (R, 2 * D), torch.float32, std=0.3)
    y = B.dit_adaln(x, dtype, shift=mod[:, :D], scale=mod[:, D:], mod_stride=2 * D, cu_seqlens=cu, n_requests=R)
    m = mod.double().cpu()
    req = torch.tensor([0] * 20 + [1] + [2] * 54)
    ref = O.layer_norm(x.double().cpu(), 1e-6) * (1 + m[req][:, D:]) + m[req][:, :D]
    tol = dict(rel=2e-6, maxabs=2e-5) if dtype == torch.float32 else dict(rel=3e-3, maxabs=2e-2)
    check(y, ref, dtype, "adaln varlen", **tol)
    # NULL shift/scale = plain LN; NULL gate = 1
    h = rnd("h", (T, D), dtype)
    x2 = x.clone()
    y2 = B.dit_adaln(x2, dtype, h=h)
    xr = x.double().cpu() + h.double().cpu()
    check(x2, xr, torch.float32, "ungated residual", rel=1e-6, maxabs=1e-5)
    check(y2, O.layer_norm(xr, 1e-6), dtype, "plain LN", **tol)
    # constant rows => y = shift (degenerate variance)
    xc = torch.full((4, D), 3.25, device=DEV)
    yc = B.dit_adaln(xc, dtype, shift=mod[:1, :D], scale=mod[:1, D:], mod_stride=2 * D)
    check(yc, m[0, :D].expand(4, D), dtype, "constant row", **tol)


@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("T,D,R", [(592, 1024, 1), (1000, 3072, 3), (4352, 3072, 1), (777, 5120, 2), (2000, 2048, 5), (650, 6144, 1)])
def test_adaln_persistent_rows_kernel(lib, dtype, T, D, R):
    """T >= 592 rows without the residual take the persistent bulk-copy kernel (CTAs walk rows with a stride, modulation
    rows held in registers and reloaded when the request changes): ragged request boundaries, every D / 1024."""
    bounds = sorted({0, T} | {(T * (2 * r + 1)) // (2 * R) + r for r in range(R - 1)})
    assert len(bounds) == R + 1
    cu = torch.tensor(bounds, dtype=torch.int32, device=DEV)
    x = rnd("xp", (T, D), torch.float32, std=2.0, mean=-0.2)
    mod = rnd("modp", (R, 2 * D), torch.float32, std=0.3)
    y = B.dit_adaln(x, dtype, shift=mod[:, :D], scale=mod[:, D:], mod_stride=2 * D, cu_seqlens=cu if R > 1 else None, n_requests=R)
    m = mod.double().cpu()
    req = torch.repeat_interleave(torch.arange(R), torch.tensor([bounds[r + 1] - bounds[r] for r in range(R)]))
    ref = O.layer_norm(x.double().cpu(), 1e-6) * (1 + m[req][:, D:]) + m[req][:, :D]
    if dtype == torch.float32:
        check(y, ref, dtype, "adaln persistent", rel=2e-6, maxabs=2e-5)
    else:
        check(y, ref, dtype, "adaln persistent", rel=3e-3, maxabs=6e-2)
        check_rounding(y, ref, "adaln persistent")
    # plain LN (no modulation) on the same kernel
    y0 = B.dit_adaln(x, dtype)
    check(y0, O.layer_norm(x.double().cpu(), 1e-6), dtype, "adaln persistent, plain LN",
          **(dict(rel=2e-6, maxabs=2e-5) if dtype == torch.float32 else dict(rel=3e-3, maxabs=6e-2)))


# ------------------------------------------------------------------------------ QK-RMSNorm + RoPE
@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("T,H,d", [(33, 4, 64), (130, 24, 128), (7, 3, 128)])
@pytest.mark.parametrize("norm,rope", [(True, True), (True, False), (False, True)])
def test_qknorm_rope(lib, dtype, T, H, d, norm, rope):
    D = H * d
    qkv = rnd("qkv", (T, 3 * D), dtype)
    gq, gk = rnd("gq", (d,), dtype, std=0.1, mean=1.0), rnd("gk", (d,), dtype, std=0.1, mean=1.0)
    pos = torch.stack([torch.arange(T) % 3, torch.arange(T) % 5, torch.arange(T) // 5], 1)
    dims = (d // 4, d // 4, d // 2)
    ang = O.rope_angles(pos, dims, 10000.0)
    rc, rs = torch.cos(ang).float().to(DEV), torch.sin(ang).float().to(DEV)
    ref = qkv.double().cpu().reshape(T, 3, H, d)
    q, k = ref[:, 0], ref[:, 1]
    if norm:
        q, k = O.rms_norm_heads(q, gq.double().cpu(), 1e-6), O.rms_norm_heads(k, gk.double().cpu(), 1e-6)
    if rope:
        a = torch.atan2(rs.double().cpu(), rc.double().cpu())  # the fp32 table the kernel is given
        q, k = O.apply_rope(q, a), O.apply_rope(k, a)
    ref = torch.stack([q, k, ref[:, 2]], 1).reshape(T, 3 * D)
    got = qkv.clone()
    B.dit_qknorm_rope(got, H, d, 2, gq if norm else None, gk if norm else None, 1e-6, rc if rope else None,
                      rs if rope else None)
    tol = dict(rel=2e-6, maxabs=2e-5) if dtype == torch.float32 else dict(rel=3e-3, maxabs=2e-2)
    check(got, ref, dtype, "qknorm_rope", **tol)
    assert torch.equal(got[:, 2 * D:], qkv[:, 2 * D:])          # v untouched


# ------------------------------------------------------------------------------ Linear (GEMM + epilogues)
# the last two pick the 240-wide tile (34 x 13 tiles = 2.99 waves of 148 SMs; ragged last N tile) and, with 20000
# rows, several persistent rounds per CTA of the 256-wide one
GEMM_SHAPES = [(1, 64, 64), (100, 72, 16), (288, 768, 256), (257, 1024, 320), (130, 3072, 64), (515, 200, 1032),
               (1000, 256, 4096), (4352, 3072, 128), (20000, 512, 64)]


@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("M,N,K", [(128, 128, 64), (300, 520, 200), (1000, 1096, 512), (4352, 1992, 3072), (77, 8, 4096)])
def test_linear_swiglu(lib, dtype, M, N, K):
    """Gated-MLP up-projection (R40): SiLU(A W1^T + b1) (.) (A W3^T + b3).  bf16: one tcgen05 kernel, W1 | W3 halves of a
    256-column accumulator tile (N = 520 / 1096 / 1992 / 8: ragged last 128-column tile); fp32: two GEMMs + product."""
    A = rnd("A", (M, K), dtype)
    W1, W3 = rnd("W1", (N, K), dtype, std=1.0 / math.sqrt(K)), rnd("W3", (N, K), dtype, std=1.0 / math.sqrt(K))
    b1, b3 = rnd("b1", (N,), dtype, std=0.5), rnd("b3", (N,), dtype, std=0.5)
    got = B.dit_linear_swiglu(A, W1, b1, W3, b3)
    Ad = A.double().cpu()
    ref = O.silu(O.linear(Ad, W1.cpu(), b1.cpu())) * O.linear(Ad, W3.cpu(), b3.cpu())
    if dtype == torch.float32:
        check(got, ref, dtype, f"swiglu {M}x{N}x{K}", rel=2e-6, maxabs=1e-4)
    else:
        # heavy-tailed product (max ~ 40 RMS): the bf16 rounding of the largest elements alone exceeds any bar relative to
        # the RMS, so the element-wise bound below (2^-8 |ref| + 2e-3 RMS) replaces max-abs / RMS
        check(got, ref, dtype, f"swiglu {M}x{N}x{K}", rel=3e-3, maxabs=1.0)
        check_rounding(got, ref, f"swiglu {M}x{N}x{K}")
    got0 = B.dit_linear_swiglu(A, W1, None, W3, None)                            # no biases
    ref0 = O.silu(O.linear(Ad, W1.cpu(), None)) * O.linear(Ad, W3.cpu(), None)
    check(got0, ref0, dtype, "swiglu no bias", **(dict(rel=2e-6, maxabs=1e-4) if dtype == torch.float32 else dict(rel=3e-3, maxabs=1.0)))
    if dtype != torch.float32:
        check_rounding(got0, ref0, "swiglu no bias")


@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("M,N,K", GEMM_SHAPES)
@pytest.mark.parametrize("epi", [B.EPI_BIAS, B.EPI_BIAS_GELU, B.EPI_BIAS_F32])
def test_linear(lib, dtype, M, N, K, epi):
    if dtype == torch.float32 and epi == B.EPI_BIAS_F32:
        pytest.skip("fp32 output is the fp32 path's only output type")
    A = rnd("A", (M, K), dtype)
    W, b = rnd("W", (N, K), dtype, std=1.0 / math.sqrt(K)), rnd("b", (N,), dtype, std=0.5)
    got = B.dit_linear(A, W, b, epi)
    ref = O.linear(A.double().cpu(), W.cpu(), b.cpu())
    if epi == B.EPI_BIAS_GELU:
        ref = O.gelu_tanh(ref)
    odt = torch.float32 if (epi == B.EPI_BIAS_F32 or dtype == torch.float32) else torch.bfloat16
    assert got.dtype == odt
    if dtype == torch.float32:
        tol = dict(rel=2e-6, maxabs=3e-5)
    elif odt == torch.float32:  # tcgen05 accumulates in fp32 but aligns addends by truncation: ~sqrt(K) 2^-24 growth
        tol = dict(rel=1e-5, maxabs=1e-4)  # (measured 4.0e-6 at K = 4096; DESIGN.md §7 tolerances)
    else:
        tol = dict(rel=3e-3, maxabs=3e-2)
    check(got, ref, odt, f"linear {M}x{N}x{K} epi{epi}", **tol)
    if odt == torch.bfloat16:       # fp32 accumulation: the only bf16 error is the output rounding
        check_rounding(got, ref, f"linear {M}x{N}x{K} epi{epi}")


@pytest.mark.parametrize("M,H,K", [(1, 1, 64), (300, 3, 256), (515, 2, 1032), (129, 5, 128)])
@pytest.mark.parametrize("norm,rope", [(True, True), (True, False), (False, True)])
def test_linear_qkv_fused_norm_rope_epilogue(lib, M, H, K, norm, rope):
    """QKV projection with QK-RMSNorm + RoPE in the GEMM epilogue against the definition written out with the
    oracle's pieces: linear -> per-head RMSNorm of q, k (gains g_q, g_k) -> RoPE on interleaved pairs; v untouched.
    H odd: the last 256-column tile holds one head of v only; M spans several row tiles with a ragged tail."""
    dt, d = torch.bfloat16, 128
    D = H * d
    A = rnd("A", (M, K), dt)
    W, b = rnd("W", (3 * D, K), dt, std=1.0 / math.sqrt(K)), rnd("b", (3 * D,), dt, std=0.5)
    gq, gk = rnd("gq", (d,), dt, std=0.1, mean=1.0), rnd("gk", (d,), dt, std=0.1, mean=1.0)
    ang = rnd("ang", (M, d // 2), torch.float32, std=2.0).double().cpu()
    rc, rs = torch.cos(ang).float().to(DEV), torch.sin(ang).float().to(DEV)
    got = B.dit_linear_qkv(A, W, b, D, gq if norm else None, gk if norm else None, 1e-6, rc if rope else None,
                           rs if rope else None)
    qkv = O.linear(A.double().cpu(), W.cpu(), b.cpu())
    q, k, v = (qkv[:, i * D:(i + 1) * D].reshape(M, H, d) for i in range(3))
    if norm:
        q, k = O.rms_norm_heads(q, gq.double().cpu(), 1e-6), O.rms_norm_heads(k, gk.double().cpu(), 1e-6)
    if rope:   # the tables the kernel consumes are fp32: rotate with exactly those values
        a32 = (rc.double().cpu(), rs.double().cpu())
        def rot(x):
            x2 = x.reshape(M, H, d // 2, 2)
            c_, s_ = a32[0][:, None, :], a32[1][:, None, :]
            return torch.stack([x2[..., 0] * c_ - x2[..., 1] * s_, x2[..., 0] * s_ + x2[..., 1] * c_], dim=-1).reshape(M, H, d)
        q, k = rot(q), rot(k)
    ref = torch.cat([q.reshape(M, D), k.reshape(M, D), v.reshape(M, D)], dim=1)
    check(got, ref, dt, f"linear_qkv {M}x{H}x{K}", rel=3e-3, maxabs=3e-2)
    check_rounding(got, ref, f"linear_qkv {M}x{H}x{K}")       # fp32 up to the single bf16 rounding


@pytest.mark.parametrize("dtype", DTYPES)
def test_linear_strided_views_and_no_bias(lib, dtype):
    """A and out are column slices of wider buffers (the step's qkv / packed layouts)."""
    M, N, K = 300, 384, 512
    big = rnd("A", (M, 3 * K), dtype)
    A = big[:, K:2 * K]
    W = rnd("W", (N, K), dtype, std=1.0 / math.sqrt(K))
    outbig = torch.zeros((M, 2 * N), dtype=dtype, device=DEV)
    B.dit_linear(A, W, None, B.EPI_BIAS, out=outbig[:, N:])
    ref = O.linear(A.double().cpu(), W.cpu())
    tol = dict(rel=2e-6, maxabs=3e-5) if dtype == torch.float32 else dict(rel=3e-3, maxabs=2e-2)
    check(outbig[:, N:], ref, dtype, "strided linear", **tol)
    assert (outbig[:, :N] == 0).all()
    assert B.dit_linear(A[:0], W, None).shape == (0, N)


@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("M,N,K,R", [(288, 256, 256, 1), (515, 768, 1032, 3), (130, 3072, 512, 1), (1000, 264, 4096, 4),
                                     (4352, 3072, 64, 2)])   # the last one takes the 240-wide tile
@pytest.mark.parametrize("gated", [True, False])
def test_linear_residual_gate_epilogue(lib, dtype, M, N, K, R, gated):
    """x <- x + gate[req(row)] (.) (A W^T + b) in the GEMM epilogue (the out-projection / fc2 of every block).
    Request boundaries fall inside 128-row tiles; N is not a multiple of the 256-column tile."""
    A = rnd("A", (M, K), dtype)
    W, b = rnd("W", (N, K), dtype, std=1.0 / math.sqrt(K)), rnd("b", (N,), dtype, std=0.5)
    x0 = rnd("x", (M, N), torch.float32, std=2.0)
    gate = rnd("gate", (R, 2 * N), torch.float32, std=0.5)[:, N:] if gated else None   # a slice: stride 2N
    bounds = [0] + sorted(int(v) for v in (synth.uniform01(5, "cu", R - 1) * M)) + [M] if R > 1 else [0, M]
    cu = torch.tensor(bounds, dtype=torch.int32, device=DEV)
    x = x0.clone()
    B.dit_linear_residual(A, W, x, b, gate, 2 * N if gated else 0, cu if R > 1 else None, R)
    branch = O.linear(A.double().cpu(), W.cpu(), b.cpu())
    if gated:
        req = torch.bucketize(torch.arange(M), torch.tensor(bounds[1:-1]), right=True) if R > 1 else torch.zeros(M, dtype=torch.long)
        branch = gate.double().cpu()[req] * branch
    ref = x0.double().cpu() + branch
    tol = dict(rel=2e-6, maxabs=3e-5) if dtype == torch.float32 else dict(rel=1e-5, maxabs=1e-4)
    check(x, ref, torch.float32, f"linear_residual {M}x{N}x{K} R={R}", **tol)
    # zero gate: x is returned bit-exact (adaLN-Zero identity, BASELINE.json north_star)
    if gated:
        x = x0.clone()
        B.dit_linear_residual(A, W, x, b, torch.zeros_like(gate), N, cu if R > 1 else None, R)
        assert torch.equal(x, x0)


# ------------------------------------------------------------------------------ attention partial + merge
def _attn_tol(dtype):
    return dict(rel=2e-6, maxabs=3e-5) if dtype == torch.float32 else dict(rel=4e-3, maxabs=2.5e-2)


@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("nq,nk,H,d", [(1, 1, 1, 64), (77, 133, 3, 64), (288, 288, 4, 64), (300, 515, 2, 128),
                                        (128, 1024, 2, 128), (640, 257, 3, 128), (5, 64, 1, 128), (129, 65, 1, 128),
                                        (256, 192, 2, 128), (100, 1, 2, 128)])
def test_attn_partial(lib, dtype, nq, nk, H, d):
    q, k, v = synth.make_attention_qkv(11, nq, nk, H, d, dtype=dtype, device=DEV)
    o, lse = B.dit_attn_partial(q, k, v)
    ro, rl = O.attention(q.cpu(), k.cpu(), v.cpu())
    check(o, ro, dtype, f"attn o {nq}x{nk}", **_attn_tol(dtype))
    assert float((lse.double().cpu() - rl).abs().max()) < (1e-5 if dtype == torch.float32 else 2e-2)


@pytest.mark.parametrize("dtype", DTYPES)
def test_attn_peaky_and_identical_keys(lib, dtype):
    """x4 logits (peaky softmax, R7/§8(c) sensitivity warning) and the 'identical keys => mean of V' invariant."""
    nq, nk, H, d = 200, 333, 2, 128
    q, k, v = synth.make_attention_qkv(11, nq, nk, H, d, dtype=dtype, device=DEV, logit_gain=4.0)
    o, lse = B.dit_attn_partial(q, k, v)
    ro, rl = O.attention(q.cpu(), k.cpu(), v.cpu())
    check(o, ro, dtype, "peaky attention", **_attn_tol(dtype))
    k1 = k[:1].expand(nk, H, d).contiguous()
    o1, _ = B.dit_attn_partial(q, k1, v)
    mean_v = v.double().cpu().mean(0, keepdim=True).expand(nq, H, d)
    check(o1, mean_v, dtype, "identical keys", **_attn_tol(dtype))
    ones = torch.ones_like(v)
    o2, _ = B.dit_attn_partial(q, k, ones)                      # softmax rows sum to 1
    assert float((o2.double().cpu() - 1).abs().max()) < (1e-5 if dtype == torch.float32 else 8e-3)


@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("nq,nk", [(130, 700), (257, 1100)])
def test_attn_growing_row_maxima_force_rescale(lib, dtype, nq, nk):
    """Keys whose norm ramps up 6x along the sequence: the running row max grows by far more than the lazy-rescale
    threshold (2^8) from key tile to key tile, so the O / row-sum rescale path (R25; taken jointly by the
    leader and follower softmax warps of a row) runs several times per row."""
    H, d = 2, 128
    q, k, v = synth.make_attention_qkv(11, nq, nk, H, d, dtype=dtype, device=DEV, logit_gain=3.0)
    ramp = (1.0 + 5.0 * torch.arange(nk, device=DEV, dtype=torch.float32) / nk).view(nk, 1, 1)
    k = (k.float() * ramp).to(dtype)
    o, lse = B.dit_attn_partial(q, k, v)
    ro, rl = O.attention(q.cpu(), k.cpu(), v.cpu())
    check(o, ro, dtype, f"rescale attention {nq}x{nk}", **_attn_tol(dtype))
    assert float((lse.double().cpu() - rl).abs().max()) < (1e-4 if dtype == torch.float32 else 5e-2)


@pytest.mark.parametrize("nq,nk,jump_at", [(300, 1000, 700), (130, 300, 140), (512, 8192, 5000)])
def test_attn_score_jump_repeats_the_pass_exactly(lib, nq, nk, jump_at):
    """One key far down the sequence is 12 x a query row: that row's score jumps ~190 log2 units above everything seen
    before, inside one key tile.  The optimistic pass of the tensor-core kernel (no row max after the first key tile,
    DESIGN.md R33) overflows there, raises the CTA's panic flag and the CTA (for n_k >= 8192: the CTA pair) repeats the
    keys with the exact per-tile row max; rows of other CTAs keep their optimistic result.  Both must match the oracle."""
    H, d = 2, 128
    q, k, v = synth.make_attention_qkv(11, nq, nk, H, d, dtype=torch.bfloat16, device=DEV)
    k[jump_at] = (12.0 * q[5].float()).to(torch.bfloat16)
    o, lse = B.dit_attn_partial(q, k, v)
    torch.cuda.synchronize()
    assert torch.isfinite(o.float()).all() and torch.isfinite(lse).all()
    ro, rl = O.attention(q.cpu(), k.cpu(), v.cpu())
    # row 5 returns v[jump_at] itself (|v| up to ~4 against RMS(o) ~ 0.1): its bf16 output rounding alone exceeds the
    # max-abs / RMS bar, so the element-wise rounding bound is used next to the rel-L2 bar
    assert errors(o, ro)[0] <= 4e-3
    check_rounding(o, ro, f"score jump {nq}x{nk}", ulps=1.0, atol_rms=2.5e-2)
    assert float((lse.double().cpu() - rl).abs().max()) < 5e-2
    assert float((o[5].float().cpu() - v[jump_at].float().cpu()).abs().max()) < 2e-2       # row 5 sees only that key
    # the repeated pass is deterministic, and the split-KV form (the jump sits in one of P = 2 shards; the other shard's
    # partial keeps its optimistic result) merges to the same answer
    o2, lse2 = B.dit_attn_partial(q, k, v)
    assert torch.equal(o, o2) and torch.equal(lse, lse2)
    half = (nk + 1) // 2
    parts = [B.dit_attn_partial(q, k[a:b], v[a:b]) for a, b in ((0, half), (half, nk))]
    om, lm = B.dit_attn_merge([x[0] for x in parts], [x[1] for x in parts])
    torch.cuda.synchronize()
    assert errors(om, ro)[0] <= 5e-3 and float((lm.double().cpu() - rl).abs().max()) < 5e-2


def test_attn_cta_pair_multicast_path(lib):
    """n_k >= 8192 and an even number of 256-row query blocks: the kernel runs as CTA pairs that share every K / V
    tile by TMA multicast.  Sampled query rows (both CTAs of a pair, ragged last key tile) against the oracle, and
    the whole output against the same call made with an odd block count (single-CTA path) on the common rows."""
    H, d, nk = 2, 128, 8192 + 77
    q, k, v = synth.make_attention_qkv(11, 1024, nk, H, d, dtype=torch.bfloat16, device=DEV)
    o, lse = B.dit_attn_partial(q, k, v)                       # 4 query blocks -> 2 pairs
    rows = torch.tensor([0, 255, 256, 300, 511, 512, 767, 768, 1023])
    ro, rl = O.attention(q[rows.to(DEV)].cpu(), k.cpu(), v.cpu())
    check(o[rows.to(DEV)], ro, torch.bfloat16, "pair attention sampled rows", **_attn_tol(torch.bfloat16))
    assert float((lse[rows.to(DEV)].double().cpu() - rl).abs().max()) < 2e-2
    o1, lse1 = B.dit_attn_partial(q[:768], k, v)               # 3 query blocks -> single-CTA kernel
    assert torch.equal(o[:768], o1) and torch.equal(lse[:768], lse1)


@pytest.mark.parametrize("dtype", DTYPES)
def test_attn_strided_qkv_buffer_and_empty(lib, dtype):
    T, H, d = 150, 3, 64
    D = H * d
    qkv = rnd("qkv", (T, 3 * D), dtype)
    q, k, v = (qkv[:, i * D:(i + 1) * D].view(T, H, d) for i in range(3))
    o, lse = B.dit_attn_partial(q, k, v)
    ro, rl = O.attention(q.cpu(), k.cpu(), v.cpu())
    check(o, ro, dtype, "strided attention", **_attn_tol(dtype))
    o0, l0 = B.dit_attn_partial(q, k[:0], v[:0])                # n_k = 0: o = 0, lse = -inf (R18)
    assert (o0 == 0).all() and torch.isinf(l0).all() and (l0 < 0).all()
    oe, le = B.dit_attn_partial(q[:0], k, v)
    assert oe.shape == (0, H, d)


@pytest.mark.parametrize("dtype", DTYPES)
@pytest.mark.parametrize("P", [1, 2, 3, 4, 8])
def test_split_kv_merge_reproduces_unsplit(lib, dtype, P):
    nq, nk, H, d = 260, 1000, 2, 128
    q, k, v = synth.make_attention_qkv(11, nq, nk, H, d, dtype=dtype, device=DEV)
    parts = [B.dit_attn_partial(q, k[a:b], v[a:b]) for a, b in O.shard_bounds(nk, P)]
    o, lse = B.dit_attn_merge([p[0] for p in parts], [p[1] for p in parts])
    ro, rl = O.attention(q.cpu(), k.cpu(), v.cpu())
    check(o, ro, dtype, f"split P={P}", **_attn_tol(dtype))
    assert float((lse.double().cpu() - rl).abs().max()) < (1e-5 if dtype == torch.float32 else 2e-2)
    # the merge kernel alone against the oracle's merge of the SAME partials (isolates the merge)
    mo, ml = O.merge_partials([p[0].cpu() for p in parts], [p[1].cpu() for p in parts])
    tol = dict(rel=1e-6, maxabs=1e-5) if dtype == torch.float32 else dict(rel=3e-3, maxabs=1.6e-2)
    check(o, mo, dtype, "merge kernel", **tol)
    o1, _ = B.dit_attn_partial(q, k, v)
    e_rel, _ = errors(o, o1)
    # P-invariance on the GPU itself.  bf16: both sides carry independent roundings (P and O to bf16; the split side
    # also its bf16 partials), each ~2^-9/sqrt(3) = 1.1e-3 rel-L2 on these noise-like outputs => ~3e-3 between them
    assert e_rel < (2e-6 if dtype == torch.float32 else 4.5e-3)


@pytest.mark.parametrize("dtype", DTYPES)
def test_merge_closed_forms_and_empty_shards(lib, dtype):
    nq, H, d = 70, 2, 64
    o = rnd("o", (nq, H, d), dtype)
    lse = rnd("lse", (nq, H), torch.float32, std=3.0)
    mo, ml = B.dit_attn_merge([o] * 4, [lse] * 4)               # P copies => O, LSE + ln P
    tol = dict(rel=1e-6, maxabs=1e-5) if dtype == torch.float32 else dict(rel=3e-3, maxabs=1.6e-2)
    check(mo, o, dtype, "merge of copies", **tol)
    assert float((ml - (lse + math.log(4))).abs().max()) < 1e-5
    ninf = torch.full_like(lse, -math.inf)
    z = torch.zeros_like(o)
    mo, ml = B.dit_attn_merge([z, o], [ninf, lse])
    assert torch.equal(mo, o) and torch.equal(ml, lse)
    mo, ml = B.dit_attn_merge([z, z], [ninf, ninf])
    assert (mo == 0).all() and torch.isinf(ml).all()
    lse2 = lse.clone(); lse2[::2] = -math.inf                   # mixed: some rows have an empty shard
    o2 = rnd("o2", (nq, H, d), dtype)
    mo, ml = B.dit_attn_merge([o, o2], [lse, lse2])
    ro, rl = O.merge_partials([o.cpu(), o2.cpu()], [lse.cpu(), lse2.cpu()])
    check(mo, ro, dtype, "merge mixed -inf", **tol)
