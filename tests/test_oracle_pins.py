"""Pins for the CPU oracle (oracle/dit_oracle.py) against things OTHER than itself: brute force in pure
Python, closed forms, invariants, torch library routines as special cases, stored hand-computed fixtures.
SURVEY.md §8(c) "What pins the oracle"; BASELINE.json north_star invariants.  CPU only."""
import math
import os

import pytest
import torch

from oracle import dit_oracle as O
from paper_2606_13501_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden")
F64 = torch.float64


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [[float(t) for t in ln.split()] for ln in f if not ln.startswith("#")]


def rnd(*shape, seed=0, name="x"):
    return synth.normal(seed, name, shape, dtype=F64)


# ---------------------------------------------------------------- attention
def brute_attention(q, k, v, scale):
    """triple loop, direct exp with NO max subtraction (pure Python floats)."""
    Nq, H, d = q.shape
    Nk = k.shape[0]
    o = torch.zeros(Nq, H, d, dtype=F64)
    lse = torch.zeros(Nq, H, dtype=F64)
    for i in range(Nq):
        for h in range(H):
            e = []
            for j in range(Nk):
                s = 0.0
                for c in range(d):
                    s += float(q[i, h, c]) * float(k[j, h, c])
                e.append(math.exp(s * scale))
            z = sum(e)
            lse[i, h] = math.log(z)
            for c in range(d):
                o[i, h, c] = sum(e[j] * float(v[j, h, c]) for j in range(Nk)) / z
    return o, lse


def test_attention_brute_force_tiny():
    q, k, v = rnd(5, 2, 4, name="q"), rnd(7, 2, 4, name="k"), rnd(7, 2, 4, name="v")
    o, lse = O.attention(q, k, v)
    ob, lb = brute_attention(q, k, v, 1 / math.sqrt(4))
    assert torch.allclose(o, ob, rtol=1e-12, atol=1e-13)
    assert torch.allclose(lse, lb, rtol=1e-12, atol=1e-13)


def test_attention_closed_form_fixture():
    r = _rows("attention_2x2_closed_form.txt")[0]
    q = torch.tensor(r[0:2], dtype=F64).reshape(2, 1, 1)
    k = torch.tensor(r[2:4], dtype=F64).reshape(2, 1, 1)
    v = torch.tensor(r[4:6], dtype=F64).reshape(2, 1, 1)
    o, lse = O.attention(q, k, v, scale=1.0)
    assert torch.allclose(o.reshape(-1), torch.tensor(r[6:8], dtype=F64), rtol=1e-13)
    assert torch.allclose(lse.reshape(-1), torch.tensor(r[8:10], dtype=F64), rtol=1e-13)


def test_attention_matches_torch_sdpa():
    q, k, v = rnd(33, 3, 16, name="q"), rnd(50, 3, 16, name="k"), rnd(50, 3, 16, name="v")
    o, _ = O.attention(q, k, v)
    ref = torch.nn.functional.scaled_dot_product_attention(q.permute(1, 0, 2), k.permute(1, 0, 2), v.permute(1, 0, 2))
    assert torch.allclose(o, ref.permute(1, 0, 2), rtol=1e-10, atol=1e-12)


def test_softmax_rows_sum_to_one_via_ones_value():
    # V = all ones  =>  O = sum_j p_ij = 1 exactly the row sum of the softmax
    q, k = rnd(9, 2, 8, name="q") * 3, rnd(11, 2, 8, name="k") * 3
    o, _ = O.attention(q, k, torch.ones(11, 2, 8, dtype=F64))
    assert torch.allclose(o, torch.ones_like(o), rtol=0, atol=1e-14)


def test_identical_keys_give_mean_of_v():
    q, v = rnd(6, 2, 8, name="q"), rnd(10, 2, 8, name="v")
    k = rnd(1, 2, 8, name="k").expand(10, 2, 8).contiguous()
    o, lse = O.attention(q, k, v)
    assert torch.allclose(o, v.mean(0, keepdim=True).expand_as(o), rtol=1e-13, atol=1e-14)
    s = torch.einsum("qhd,hd->qh", q, k[0]) / math.sqrt(8)
    assert torch.allclose(lse, s + math.log(10), rtol=1e-13)
    o0, _ = O.attention(torch.zeros_like(q), rnd(10, 2, 8, name="k2"), v)           # q = 0 => mean of V
    assert torch.allclose(o0, v.mean(0, keepdim=True).expand_as(o0), rtol=1e-13, atol=1e-14)


def test_single_key_permutation_linearity_shift_peaky():
    q, k, v = rnd(6, 2, 8, name="q"), rnd(10, 2, 8, name="k"), rnd(10, 2, 8, name="v")
    o, lse = O.attention(q, k, v)
    o1, _ = O.attention(q, k[:1], v[:1])
    assert torch.allclose(o1, v[:1].expand_as(o1))                                    # Nk = 1 => v0
    perm = torch.tensor([3, 1, 4, 0, 9, 2, 6, 5, 8, 7])
    op, lp = O.attention(q, k[perm], v[perm])
    assert torch.allclose(op, o, rtol=1e-12, atol=1e-14) and torch.allclose(lp, lse, rtol=1e-12)
    o2, _ = O.attention(q, k, 2 * v)
    assert torch.allclose(o2, 2 * o, rtol=1e-13)                                      # linear in V
    u = rnd(1, 2, 8, name="u")
    os_, _ = O.attention(q, k + u, v)
    assert torch.allclose(os_, o, rtol=1e-10, atol=1e-12)                             # softmax shift invariance
    kp = k.clone(); kp[4] = q[2] * 60.0 / (q[2] ** 2).sum(-1, keepdim=True) * math.sqrt(8)   # logit +60 for row 2
    opk, _ = O.attention(q[2:3], kp, v)
    assert torch.allclose(opk, v[4:5], atol=1e-9)                                     # peaky: max subtraction works
    big = O.attention(q * 1e3, k, v)[0]
    assert torch.isfinite(big).all()


# ---------------------------------------------------------------- partial + merge
@pytest.mark.parametrize("P", [1, 2, 3, 4, 8])
def test_split_p_invariance(P):
    q, k, v = rnd(12, 2, 8, name="q"), rnd(37, 2, 8, name="k"), rnd(37, 2, 8, name="v")
    o, lse = O.attention(q, k, v)
    op, lp = O.attention_split(q, k, v, P)
    assert torch.allclose(op, o, rtol=1e-12, atol=1e-14) and torch.allclose(lp, lse, rtol=1e-12)


def test_merge_closed_forms():
    q, k, v = rnd(5, 2, 8, name="q"), rnd(9, 2, 8, name="k"), rnd(9, 2, 8, name="v")
    o, lse = O.attention(q, k, v)
    om, lm = O.merge_partials([o] * 4, [lse] * 4)                                     # P copies => O, LSE + ln P
    assert torch.allclose(om, o, rtol=1e-13) and torch.allclose(lm, lse + math.log(4), rtol=1e-13)
    oe, le = O.attention(q, k[:0], v[:0])                                             # empty shard: 0, -inf
    assert (oe == 0).all() and torch.isinf(le).all() and (le < 0).all()
    om, lm = O.merge_partials([oe, o], [le, lse])
    assert torch.equal(om, o) and torch.equal(lm, lse)
    om, lm = O.merge_partials([oe, oe], [le, le])
    assert (om == 0).all() and torch.isinf(lm).all()
    assert O.shard_bounds(10, 4) == [(0, 3), (3, 6), (6, 9), (9, 10)]
    assert O.shard_bounds(5, 8)[-1] == (5, 5)
    # P larger than Nk (empty tail shards) still reproduces the unsplit result
    o8, l8 = O.attention_split(q, k[:5], v[:5], 8)
    o1, l1 = O.attention(q, k[:5], v[:5])
    assert torch.allclose(o8, o1, rtol=1e-12) and torch.allclose(l8, l1, rtol=1e-12)


# ---------------------------------------------------------------- norms, activations, rope
def test_layer_norm_properties_and_library():
    x = rnd(7, 48, name="x") * 3 + 1.5
    y = O.layer_norm(x, 1e-6)
    assert torch.allclose(y.mean(-1), torch.zeros(7, dtype=F64), atol=1e-14)
    var = x.var(-1, unbiased=False)
    assert torch.allclose(y.var(-1, unbiased=False), var / (var + 1e-6), rtol=1e-12)
    assert torch.allclose(y, torch.nn.functional.layer_norm(x, (48,), eps=1e-6), rtol=1e-11, atol=1e-13)
    const = torch.full((2, 48), 3.25, dtype=F64)
    sh, sc = rnd(48, name="sh"), rnd(48, name="sc")
    assert torch.allclose(O.modulate(const, sh, sc, 1e-6), sh.expand(2, 48))          # constant row => y = shift
    z = torch.zeros(48, dtype=F64)
    assert torch.equal(O.modulate(x, z, z, 1e-6), y)                                  # zero shift/scale => plain LN
    assert torch.allclose(O.modulate(x, sh, sc, 1e-6), y * (1 + sc) + sh)             # '1 + scale' (R3)


def test_rms_norm_properties():
    x = rnd(5, 3, 16, name="x") * 2
    one = torch.ones(16, dtype=F64)
    y = O.rms_norm_heads(x, one, 1e-6)
    ms = (x ** 2).mean(-1)
    assert torch.allclose((y ** 2).mean(-1).sqrt(), 1 / torch.sqrt(1 + 1e-6 / ms), rtol=1e-12)
    assert torch.allclose(O.rms_norm_heads(7.0 * x, one, 0.0), O.rms_norm_heads(x, one, 0.0), rtol=1e-13)
    g = rnd(16, name="g")
    assert torch.allclose(O.rms_norm_heads(x, g, 1e-6), y * g, rtol=1e-13)
    manual = x[2, 1] / math.sqrt(sum(float(t) ** 2 for t in x[2, 1]) / 16 + 1e-6) * g
    assert torch.allclose(O.rms_norm_heads(x, g, 1e-6)[2, 1], manual, rtol=1e-13)


def test_gelu_silu():
    for z, g in _rows("gelu_tanh_points.txt"):
        assert abs(float(O.gelu_tanh(torch.tensor(z, dtype=F64))) - g) <= 1e-15 * max(1, abs(g))
    z = torch.linspace(-6, 6, 101, dtype=F64)
    assert torch.allclose(O.gelu_tanh(z) - O.gelu_tanh(-z), z, atol=1e-14)            # odd-part identity
    assert (O.gelu_tanh(z) - torch.nn.functional.gelu(z)).abs().max() < 1e-3          # close to the erf form
    assert torch.allclose(O.gelu_tanh(z), torch.nn.functional.gelu(z, approximate="tanh"), atol=1e-14)
    assert torch.allclose(O.silu(z), torch.nn.functional.silu(z), atol=1e-14)
    assert float(O.silu(torch.tensor(0.0, dtype=F64))) == 0.0


def test_rope_fixture_identity_norm_relative():
    rows = _rows("rope_points.txt")
    pos = torch.tensor([[0, 3, 0]])
    ang = O.rope_angles(pos, (0, 8, 0), 10000.0)
    x = torch.zeros(1, 1, 8, dtype=F64); x[..., 0::2] = 1.0                            # pairs (1, 0)
    y = O.apply_rope(x, ang)
    for j, c, s in rows:
        assert abs(float(y[0, 0, 2 * int(j)]) - c) < 1e-15 and abs(float(y[0, 0, 2 * int(j) + 1]) - s) < 1e-15
    # segments are laid out in axis order (f, h, w): with dims (4, 2, 2) the h axis owns elements 4..5
    a3 = O.rope_angles(torch.tensor([[5, 7, 11]]), (4, 2, 2), 10000.0)
    assert torch.allclose(a3, torch.tensor([[5.0, 5.0 * 10000 ** -0.5, 7.0, 11.0]], dtype=F64))
    q = rnd(6, 2, 8, name="q"); k = rnd(6, 2, 8, name="k")
    p0 = torch.zeros(6, 3, dtype=torch.int64)
    assert torch.equal(O.apply_rope(q, O.rope_angles(p0, (0, 4, 4), 1e4)), q)          # pos 0 => identity
    pos = torch.stack([torch.zeros(6, dtype=torch.int64), torch.arange(6) % 3, torch.arange(6) // 3], 1)
    a = O.rope_angles(pos, (0, 4, 4), 1e4)
    qr, kr = O.apply_rope(q, a), O.apply_rope(k, a)
    assert torch.allclose((qr ** 2).sum(-1), (q ** 2).sum(-1), rtol=1e-13)            # norm preserving
    pos2 = pos + torch.tensor([0, 5, 9])
    a2 = O.rope_angles(pos2, (0, 4, 4), 1e4)
    s1 = torch.einsum("qhd,khd->hqk", qr, kr)
    s2 = torch.einsum("qhd,khd->hqk", O.apply_rope(q, a2), O.apply_rope(k, a2))
    assert torch.allclose(s1, s2, rtol=1e-10, atol=1e-12)                             # relative-position property


def test_token_positions_and_patchify():
    pos = O.token_positions((2, 3, 4))
    assert pos.shape == (24, 3) and pos[0].tolist() == [0, 0, 0] and pos[5].tolist() == [0, 1, 1]
    assert pos[(1 * 3 + 2) * 4 + 3].tolist() == [1, 2, 3]
    lat = rnd(3, 2, 4, 6, name="lat")
    tok = O.patchify(lat, (1, 2, 2))
    assert tok.shape == (2 * 2 * 3, 3 * 4)
    # token (f'=1, h'=1, w'=2), feature (c=2, i=0, j=1, k=0)  ==  lat[2, 1, 2*1+1, 2*2+0]
    assert tok[(1 * 2 + 1) * 3 + 2, ((2 * 1 + 0) * 2 + 1) * 2 + 0] == lat[2, 1, 3, 4]
    assert torch.equal(O.unpatchify(tok, (1, 2, 2), lat.shape), lat)                  # round trip
    lat3 = rnd(2, 4, 4, 4, name="lat3")
    t3 = O.patchify(lat3, (2, 2, 2))
    assert t3[(1 * 2 + 0) * 2 + 1, ((1 * 2 + 1) * 2 + 0) * 2 + 1] == lat3[1, 3, 0, 3]
    assert torch.equal(O.unpatchify(t3, (2, 2, 2), lat3.shape), lat3)


def test_timestep_embedding_closed_forms():
    e0 = synth.timestep_embedding([0.0], 256)
    assert torch.equal(e0[0, :128], torch.ones(128)) and torch.equal(e0[0, 128:], torch.zeros(128))
    e = synth.timestep_embedding([500.0], 256)
    assert abs(float(e[0, 0]) - math.cos(500.0)) < 1e-6 and abs(float(e[0, 128]) - math.sin(500.0)) < 1e-6
    w5 = math.exp(-math.log(1e4) * 5 / 128)
    assert abs(float(e[0, 5]) - math.cos(500 * w5)) < 1e-6


# ---------------------------------------------------------------- step composition
def _tiny(**kw):
    d = dict(n_blocks=2, hidden=32, n_heads=2, head_dim=16, mlp_dim=64, latent_channels=2, temb_dim=16, cond_dim=24,
             latent_grid=(1, 8, 8), n_cond=5, dtype="f32")
    d.update(kw)
    return synth.cfg1(**d)


def _run(s, W=None, I=None, **kw):
    W = synth.make_weights(s) if W is None else W
    I = synth.make_inputs(s) if I is None else I
    return O.dit_step(O.cfg_from_shape(s), W, I["latents"], I["temb"], I["cond"], **kw), W, I


def test_zero_gates_make_blocks_identity_bit_exact():
    s = _tiny()
    W = synth.make_weights(s)
    for l in range(s.n_blocks):
        D = s.hidden
        for lo in (2 * D, 5 * D):                                                     # gate1, gate2 chunks
            W[f"blocks.{l}.mod.w"][lo:lo + D] = 0
            W[f"blocks.{l}.mod.b"][lo:lo + D] = 0
    taps = {}
    out, _, _ = _run(s, W, taps=taps)
    assert torch.equal(taps["b1.x_mlp"], taps["x0"])                                  # bit exact identity
    s0 = _tiny(n_blocks=0)
    W0 = {k: v for k, v in W.items() if not k.startswith("blocks.")}
    out0, I, _ = _run(s0, W0)[0], synth.make_inputs(s0), None
    assert torch.equal(out, out0)
    # joint mode, identity blocks: the final layer reads the IMAGE rows x[Lc:] only (step 6), so the output neither depends
    # on the cond tokens nor differs from the same model without conditioning
    other = dict(I, cond=I["cond"] * -3.0 + 1.0)
    assert torch.equal(_run(s0, W0, other)[0], out0)
    sn = _tiny(n_blocks=0, cond_mode="none")
    assert torch.equal(O.dit_step(O.cfg_from_shape(sn), W0, I["latents"], I["temb"], None), out0)


def test_step_split_p_invariance_and_modes():
    for mode, rope, qkn in (("joint", (0, 0, 0), False), ("joint", (0, 8, 8), True), ("cross", (4, 6, 6), True),
                            ("none", (0, 8, 8), False)):
        s = _tiny(cond_mode=mode, rope_dims=rope, qk_rmsnorm=qkn)
        out, W, I = _run(s)
        assert out.shape == (2, 1, 8, 8) and torch.isfinite(out).all()
        for P in (2, 4):
            o2, _, _ = _run(s, W, I, split_p=P)
            assert (o2 - out).norm() / out.norm() < 1e-13


def test_joint_with_no_cond_tokens_equals_none_mode():
    s = _tiny(cond_mode="joint", rope_dims=(0, 8, 8), qk_rmsnorm=True)
    W, I = synth.make_weights(s), synth.make_inputs(s)
    a = O.dit_step(O.cfg_from_shape(s), W, I["latents"], I["temb"], I["cond"][:0])
    sn = _tiny(cond_mode="none", rope_dims=(0, 8, 8), qk_rmsnorm=True)
    b = O.dit_step(O.cfg_from_shape(sn), W, I["latents"], I["temb"], None)
    assert torch.allclose(a, b, rtol=1e-13, atol=1e-15)


def test_permutation_equivariance_without_rope():
    """patch 1x1x1, no RoPE, no cond: permuting latent pixels permutes the output identically."""
    s = _tiny(cond_mode="none", patch=(1, 1, 1), latent_grid=(1, 4, 4))
    out, W, I = _run(s)
    perm = torch.randperm(16, generator=torch.Generator().manual_seed(1))
    lat = I["latents"].reshape(2, 16)[:, perm].reshape(2, 1, 4, 4)
    outp = O.dit_step(O.cfg_from_shape(s), W, lat, I["temb"], None)
    assert torch.allclose(outp.reshape(2, 16), out.reshape(2, 16)[:, perm], rtol=1e-11, atol=1e-13)


def test_patch_embed_selector_and_final_layer():
    """With W_pe a selector and no blocks, x0 rows are raw patches (pins patch order + bias add)."""
    s = _tiny(n_blocks=0, cond_mode="none", hidden=8, n_heads=1, head_dim=8, latent_channels=2)
    W = synth.make_weights(s)
    W["patch_embed.w"] = torch.eye(8); W["patch_embed.b"] = torch.zeros(8)
    I = synth.make_inputs(s)
    taps = {}
    O.dit_step(O.cfg_from_shape(s), W, I["latents"], I["temb"], None, taps=taps)
    assert torch.equal(taps["x0"], O.patchify(I["latents"].double(), (1, 2, 2)))
    # final layer: tok = Wf (LN(x)(1 + scale_f) + shift_f) + bf, checked with torch's layer_norm
    yf = torch.nn.functional.layer_norm(taps["x0"], (8,), eps=1e-6)
    sc = O.silu(taps["c"])
    modf = (W["final.mod.w"].double() @ sc + W["final.mod.b"].double()).reshape(2, 8)
    tok = (yf * (1 + modf[1]) + modf[0]) @ W["final.w"].double().t() + W["final.b"].double()
    assert torch.allclose(taps["tok"], tok, rtol=1e-11, atol=1e-13)


def test_block_by_hand_one_block():
    """One block re-derived with torch library routines (layer_norm, sdpa, gelu, silu) — an independent
    transcription of SURVEY 8(c) step 5 that a dropped term / wrong chunk order in the oracle would fail."""
    s = _tiny(n_blocks=1, cond_mode="none", rope_dims=(0, 0, 0), qk_rmsnorm=False)
    W, I = synth.make_weights(s), synth.make_inputs(s)
    taps = {}
    O.dit_step(O.cfg_from_shape(s), W, I["latents"], I["temb"], None, taps=taps)
    Fn = torch.nn.functional
    Wd = {k: v.double() for k, v in W.items()}
    D, H, d = 32, 2, 16
    c = Fn.linear(Fn.silu(Fn.linear(I["temb"].double(), Wd["t_mlp.w1"], Wd["t_mlp.b1"])), Wd["t_mlp.w2"], Wd["t_mlp.b2"])
    m = Fn.linear(Fn.silu(c), Wd["blocks.0.mod.w"], Wd["blocks.0.mod.b"]).reshape(6, D)
    x = taps["x0"]
    y = Fn.layer_norm(x, (D,), eps=1e-6) * (1 + m[1]) + m[0]
    qkv = Fn.linear(y, Wd["blocks.0.attn.wqkv"], Wd["blocks.0.attn.bqkv"])
    q, k, v = [t.reshape(-1, H, d).permute(1, 0, 2) for t in qkv.split(D, dim=1)]
    o = Fn.scaled_dot_product_attention(q, k, v).permute(1, 0, 2).reshape(-1, D)
    x = x + m[2] * Fn.linear(o, Wd["blocks.0.attn.wo"], Wd["blocks.0.attn.bo"])
    y = Fn.layer_norm(x, (D,), eps=1e-6) * (1 + m[4]) + m[3]
    x = x + m[5] * Fn.linear(Fn.gelu(Fn.linear(y, Wd["blocks.0.mlp.w1"], Wd["blocks.0.mlp.b1"]), approximate="tanh"),
                             Wd["blocks.0.mlp.w2"], Wd["blocks.0.mlp.b2"])
    assert torch.allclose(taps["b0.x_mlp"], x, rtol=1e-10, atol=1e-12)


def _hand_rope(t, pos, rope_dims, theta):
    """Interleaved-pair RoPE written out element by element (R6), independent of O.rope_angles / O.apply_rope:
    head dim cut into per-axis segments (f, h, w); pair j of a d_a-wide segment = elements (2j, 2j+1) of the segment,
    angle pos_a * theta^(-2j/d_a); (a, b) -> (a cos - b sin, a sin + b cos).  t: [T, H, d]."""
    out = t.clone()
    T, H, d = t.shape
    for n in range(T):
        base = 0
        for a, d_a in enumerate(rope_dims):
            for j in range(d_a // 2):
                th = float(pos[n][a]) * theta ** (-2.0 * j / d_a)
                c, s_ = math.cos(th), math.sin(th)
                e, o = t[n, :, base + 2 * j], t[n, :, base + 2 * j + 1]
                out[n, :, base + 2 * j] = e * c - o * s_
                out[n, :, base + 2 * j + 1] = e * s_ + o * c
            base += d_a
    return out


def _wide_gains(W, s):
    """QK-norm gains with std 0.3 (not the near-one gains of R14) so that norm-then-RoPE and RoPE-then-norm differ
    by far more than rounding: a gain is per ELEMENT, RoPE mixes the two elements of a pair."""
    for name in list(W):
        if name.endswith(".gq") or name.endswith(".gk"):
            W[name] = (1.0 + 0.3 * synth.normal(5, "wide:" + name, W[name].shape, dtype=F64)).to(W[name].dtype)
    return W


def test_joint_block_by_hand_rmsnorm_then_rope():
    """One JOINT block with QK-RMSNorm and 2D RoPE, re-derived with torch library routines and a by-hand rotation:
    sequence [ctx ; x] (R9), cond tokens at position 0 (R6), per-head RMSNorm FIRST, RoPE SECOND (R5), then SDPA.
    Fails if the oracle rotates before normalising, swaps cos/sin, uses half-split instead of interleaved pairs,
    puts ctx after x, or gives cond tokens a non-zero position."""
    s = _tiny(n_blocks=1, cond_mode="joint", rope_dims=(0, 8, 8), qk_rmsnorm=True)
    W, I = _wide_gains(synth.make_weights(s), s), synth.make_inputs(s)
    taps = {}
    O.dit_step(O.cfg_from_shape(s), W, I["latents"], I["temb"], I["cond"], taps=taps)
    Fn = torch.nn.functional
    Wd = {k: v.double() for k, v in W.items()}
    D, H, d, Lc = 32, 2, 16, 5
    c = Fn.linear(Fn.silu(Fn.linear(I["temb"].double(), Wd["t_mlp.w1"], Wd["t_mlp.b1"])), Wd["t_mlp.w2"], Wd["t_mlp.b2"])
    m = Fn.linear(Fn.silu(c), Wd["blocks.0.mod.w"], Wd["blocks.0.mod.b"]).reshape(6, D)
    lat = I["latents"].double()                                            # [2, 1, 8, 8], patch (1, 2, 2) -> 4 x 4 tokens
    patches = torch.stack([lat[:, 0, 2 * hh:2 * hh + 2, 2 * ww:2 * ww + 2].reshape(-1) for hh in range(4) for ww in range(4)])
    ximg = Fn.linear(patches, Wd["patch_embed.w"], Wd["patch_embed.b"])
    ctx = Fn.linear(I["cond"].double(), Wd["cond_proj.w"], Wd["cond_proj.b"])
    x = torch.cat([ctx, ximg], 0)
    assert torch.allclose(taps["x0"], x, rtol=1e-12, atol=1e-14)
    pos = [(0, 0, 0)] * Lc + [(0, hh, ww) for hh in range(4) for ww in range(4)]
    y = Fn.layer_norm(x, (D,), eps=1e-6) * (1 + m[1]) + m[0]
    qkv = Fn.linear(y, Wd["blocks.0.attn.wqkv"], Wd["blocks.0.attn.bqkv"])
    q, k, v = [t.reshape(-1, H, d) for t in qkv.split(D, dim=1)]
    q = Fn.rms_norm(q, (d,), weight=Wd["blocks.0.attn.gq"], eps=1e-6)
    k = Fn.rms_norm(k, (d,), weight=Wd["blocks.0.attn.gk"], eps=1e-6)
    q, k = _hand_rope(q, pos, (0, 8, 8), 10000.0), _hand_rope(k, pos, (0, 8, 8), 10000.0)
    assert torch.allclose(taps["b0.q"], q.reshape(-1, D), rtol=1e-11, atol=1e-13)
    assert torch.allclose(taps["b0.k"], k.reshape(-1, D), rtol=1e-11, atol=1e-13)
    o = Fn.scaled_dot_product_attention(q.permute(1, 0, 2), k.permute(1, 0, 2), v.permute(1, 0, 2)).permute(1, 0, 2)
    x = x + m[2] * Fn.linear(o.reshape(-1, D), Wd["blocks.0.attn.wo"], Wd["blocks.0.attn.bo"])
    y = Fn.layer_norm(x, (D,), eps=1e-6) * (1 + m[4]) + m[3]
    x = x + m[5] * Fn.linear(Fn.gelu(Fn.linear(y, Wd["blocks.0.mlp.w1"], Wd["blocks.0.mlp.b1"]), approximate="tanh"),
                             Wd["blocks.0.mlp.w2"], Wd["blocks.0.mlp.b2"])
    assert torch.allclose(taps["b0.x_mlp"], x, rtol=1e-10, atol=1e-12)
    # the order matters at these gains: rotating first and normalising second is a different function
    q2 = Fn.rms_norm(_hand_rope(qkv[:, :D].reshape(-1, H, d), pos, (0, 8, 8), 10000.0), (d,),
                     weight=Wd["blocks.0.attn.gq"], eps=1e-6)
    assert float((q2 - q).abs().max()) > 1e-2


def _cross_block_by_hand(s, W, I, x_in, m, pos):
    """R10 transcribed with torch library routines: self-attention (norm -> RoPE), gated residual, then the cross
    sub-layer x += Wo_c SDPA(RMS(Wq_c LN(x) + bq), RMS(Wk ctx + bk), Wv ctx + bv) + bo_c with wkv rows [k | v], NO
    gate, NO modulation, NO RoPE; then the MLP.  Returns (x after cross, x after MLP)."""
    Fn = torch.nn.functional
    Wd = {k: v.double() for k, v in W.items()}
    D, H, d = s.hidden, s.n_heads, s.head_dim
    ctx = Fn.linear(I["cond"].double(), Wd["cond_proj.w"], Wd["cond_proj.b"])
    y = Fn.layer_norm(x_in, (D,), eps=1e-6) * (1 + m[1]) + m[0]
    qkv = Fn.linear(y, Wd["blocks.0.attn.wqkv"], Wd["blocks.0.attn.bqkv"])
    q, k, v = [t.reshape(-1, H, d) for t in qkv.split(D, dim=1)]
    q = _hand_rope(Fn.rms_norm(q, (d,), weight=Wd["blocks.0.attn.gq"], eps=1e-6), pos, s.rope_dims, 10000.0)
    k = _hand_rope(Fn.rms_norm(k, (d,), weight=Wd["blocks.0.attn.gk"], eps=1e-6), pos, s.rope_dims, 10000.0)
    o = Fn.scaled_dot_product_attention(q.permute(1, 0, 2), k.permute(1, 0, 2), v.permute(1, 0, 2)).permute(1, 0, 2)
    x = x_in + m[2] * Fn.linear(o.reshape(-1, D), Wd["blocks.0.attn.wo"], Wd["blocks.0.attn.bo"])
    qc = Fn.linear(Fn.layer_norm(x, (D,), eps=1e-6), Wd["blocks.0.cross.wq"], Wd["blocks.0.cross.bq"]).reshape(-1, H, d)
    kc = Fn.linear(ctx, Wd["blocks.0.cross.wkv"][:D], Wd["blocks.0.cross.bkv"][:D]).reshape(-1, H, d)   # K = first half
    vc = Fn.linear(ctx, Wd["blocks.0.cross.wkv"][D:], Wd["blocks.0.cross.bkv"][D:]).reshape(-1, H, d)   # V = second half
    qc = Fn.rms_norm(qc, (d,), weight=Wd["blocks.0.cross.gq"], eps=1e-6)
    kc = Fn.rms_norm(kc, (d,), weight=Wd["blocks.0.cross.gk"], eps=1e-6)
    oc = Fn.scaled_dot_product_attention(qc.permute(1, 0, 2), kc.permute(1, 0, 2), vc.permute(1, 0, 2)).permute(1, 0, 2)
    xc = x + Fn.linear(oc.reshape(-1, D), Wd["blocks.0.cross.wo"], Wd["blocks.0.cross.bo"])
    y = Fn.layer_norm(xc, (D,), eps=1e-6) * (1 + m[4]) + m[3]
    xm = xc + m[5] * Fn.linear(Fn.gelu(Fn.linear(y, Wd["blocks.0.mlp.w1"], Wd["blocks.0.mlp.b1"]), approximate="tanh"),
                               Wd["blocks.0.mlp.w2"], Wd["blocks.0.mlp.b2"])
    return xc, xm


def test_cross_block_by_hand():
    """One CROSS block (cfg 3's topology, R10) against an independent torch-library transcription; also pins
    block_rows in cross mode (the whole oracle side of the full-size cfg 3 test) to the same transcription.
    Fails if the K / V halves of wkv are swapped, the cross branch is gated or modulated, RoPE is applied to the
    cross q / k, the cross sub-layer is placed after the MLP, or its RMSNorm gains are dropped."""
    s = _tiny(n_blocks=1, cond_mode="cross", rope_dims=(4, 6, 6), qk_rmsnorm=True, latent_grid=(2, 8, 8), n_cond=7)
    W, I = _wide_gains(synth.make_weights(s), s), synth.make_inputs(s)
    cfg = O.cfg_from_shape(s)
    taps = {}
    O.dit_step(cfg, W, I["latents"], I["temb"], I["cond"], taps=taps)
    Fn = torch.nn.functional
    Wd = {k: v.double() for k, v in W.items()}
    c = Fn.linear(Fn.silu(Fn.linear(I["temb"].double(), Wd["t_mlp.w1"], Wd["t_mlp.b1"])), Wd["t_mlp.w2"], Wd["t_mlp.b2"])
    m = Fn.linear(Fn.silu(c), Wd["blocks.0.mod.w"], Wd["blocks.0.mod.b"]).reshape(6, s.hidden)
    pos = [(f, hh, ww) for f in range(2) for hh in range(4) for ww in range(4)]        # token n = (f H' + h) W' + w
    assert taps["x0"].shape[0] == len(pos)                                             # cross mode: sequence = x only
    xc, xm = _cross_block_by_hand(s, W, I, taps["x0"], m, pos)
    assert torch.allclose(taps["b0.x_cross"], xc, rtol=1e-10, atol=1e-12)
    assert torch.allclose(taps["b0.x_mlp"], xm, rtol=1e-10, atol=1e-12)
    # the cross branch is not negligible here, so the comparison really sees it
    assert float((taps["b0.x_cross"] - taps["b0.x_attn"]).norm() / taps["b0.x_attn"].norm()) > 1e-3
    # block_rows, cross mode, against the hand transcription (not against dit_step)
    ang = O.rope_angles(torch.tensor(pos), cfg["rope_dims"], cfg["rope_theta"])
    ctx = Fn.linear(I["cond"].double(), Wd["cond_proj.w"], Wd["cond_proj.b"])
    rows = torch.tensor([0, 3, 17, 31])
    got = O.block_rows(cfg, W, 0, taps["x0"], taps["mod"][0], ang, rows, ctx=ctx)
    assert torch.allclose(got, xm[rows], rtol=1e-10, atol=1e-12)


def test_block_rows_cross_equals_step_rows():
    """block_rows(..., ctx) in cross mode == the same rows of dit_step's second block (teacher forcing changes nothing
    when the forced input is the oracle's own)."""
    s = _tiny(n_blocks=2, cond_mode="cross", rope_dims=(4, 6, 6), qk_rmsnorm=True, latent_grid=(2, 8, 8), n_cond=7)
    W, I = _wide_gains(synth.make_weights(s), s), synth.make_inputs(s)
    cfg = O.cfg_from_shape(s)
    taps = {}
    O.dit_step(cfg, W, I["latents"], I["temb"], I["cond"], taps=taps)
    ang = O.rope_angles(O.token_positions((2, 4, 4)), cfg["rope_dims"], cfg["rope_theta"])
    ctx = O.linear(I["cond"].double(), W["cond_proj.w"], W["cond_proj.b"])
    rows = torch.tensor([1, 2, 16, 30])
    got = O.block_rows(cfg, W, 1, taps["b0.x_mlp"], taps["mod"][1], ang, rows, ctx=ctx)
    assert torch.allclose(got, taps["b1.x_mlp"][rows], rtol=1e-12, atol=1e-14)


def test_dual_stream_equals_single_stream_when_both_streams_share_weights():
    """Dual-stream joint blocks (R37) with the text stream's tensors set equal to the image stream's ARE the single-stream
    joint blocks (R9): same rows, same order, one attention over [ctx ; x]."""
    s2 = _tiny(cond_mode="joint2", rope_dims=(0, 8, 8), qk_rmsnorm=True)
    s1 = _tiny(cond_mode="joint", rope_dims=(0, 8, 8), qk_rmsnorm=True)
    W1 = _wide_gains(synth.make_weights(s1), s1)
    W2 = dict(W1)
    for k, v in W1.items():
        if k.startswith("blocks."):
            l, rest = k.split(".", 2)[1:]
            W2[f"blocks.{l}.txt.{rest}"] = v
    assert set(W2) == set(synth.weight_shapes(s2))
    I = synth.make_inputs(s1)
    a = O.dit_step(O.cfg_from_shape(s1), W1, I["latents"], I["temb"], I["cond"])
    b = O.dit_step(O.cfg_from_shape(s2), W2, I["latents"], I["temb"], I["cond"])
    assert torch.allclose(a, b, rtol=1e-12, atol=1e-14)
    b4 = O.dit_step(O.cfg_from_shape(s2), W2, I["latents"], I["temb"], I["cond"], split_p=4)
    assert torch.allclose(a, b4, rtol=1e-11, atol=1e-13)


def test_dual_stream_block_by_hand():
    """One dual-stream block with DIFFERENT weights per stream, re-derived with torch library routines: per-stream adaLN
    (own modulation), QKV, QK-RMSNorm (own gains), by-hand RoPE, ONE SDPA over [txt ; img], per-stream gated out-projection
    and MLP.  Fails if the streams' weights are swapped, the text rows do not attend to the image rows, the text stream
    takes the image stream's modulation / gains, or the text rows are placed after the image rows."""
    s = _tiny(n_blocks=1, cond_mode="joint2", rope_dims=(0, 8, 8), qk_rmsnorm=True)
    W, I = _wide_gains(synth.make_weights(s), s), synth.make_inputs(s)
    taps = {}
    O.dit_step(O.cfg_from_shape(s), W, I["latents"], I["temb"], I["cond"], taps=taps)
    Fn = torch.nn.functional
    Wd = {k: v.double() for k, v in W.items()}
    D, H, d, Lc = 32, 2, 16, 5
    c = Fn.linear(Fn.silu(Fn.linear(I["temb"].double(), Wd["t_mlp.w1"], Wd["t_mlp.b1"])), Wd["t_mlp.w2"], Wd["t_mlp.b2"])
    x = taps["x0"]
    pos = [(0, 0, 0)] * Lc + [(0, hh, ww) for hh in range(4) for ww in range(4)]
    streams = (("blocks.0.txt.", slice(0, Lc)), ("blocks.0.", slice(Lc, None)))
    mods, qkvs = {}, {}
    for pre, rows in streams:
        m = Fn.linear(Fn.silu(c), Wd[pre + "mod.w"], Wd[pre + "mod.b"]).reshape(6, D)
        y = Fn.layer_norm(x[rows], (D,), eps=1e-6) * (1 + m[1]) + m[0]
        q, k, v = [t.reshape(-1, H, d) for t in Fn.linear(y, Wd[pre + "attn.wqkv"], Wd[pre + "attn.bqkv"]).split(D, dim=1)]
        q = Fn.rms_norm(q, (d,), weight=Wd[pre + "attn.gq"], eps=1e-6)
        k = Fn.rms_norm(k, (d,), weight=Wd[pre + "attn.gk"], eps=1e-6)
        mods[pre], qkvs[pre] = m, (q, k, v)
    q, k, v = [torch.cat([qkvs["blocks.0.txt."][i], qkvs["blocks.0."][i]], 0) for i in range(3)]
    q, k = _hand_rope(q, pos, (0, 8, 8), 10000.0), _hand_rope(k, pos, (0, 8, 8), 10000.0)
    o = Fn.scaled_dot_product_attention(q.permute(1, 0, 2), k.permute(1, 0, 2), v.permute(1, 0, 2)).permute(1, 0, 2).reshape(-1, D)
    outs = []
    for pre, rows in streams:
        m = mods[pre]
        xa = x[rows] + m[2] * Fn.linear(o[rows], Wd[pre + "attn.wo"], Wd[pre + "attn.bo"])
        y = Fn.layer_norm(xa, (D,), eps=1e-6) * (1 + m[4]) + m[3]
        outs.append(xa + m[5] * Fn.linear(Fn.gelu(Fn.linear(y, Wd[pre + "mlp.w1"], Wd[pre + "mlp.b1"]), approximate="tanh"),
                                          Wd[pre + "mlp.w2"], Wd[pre + "mlp.b2"]))
    want = torch.cat(outs, 0)
    assert torch.allclose(taps["b0.x_mlp"], want, rtol=1e-10, atol=1e-12)
    # the streams really differ: giving the text rows the image stream's weights changes the text rows
    Wsw = dict(W)
    for kk in list(W):
        if kk.startswith("blocks.0.txt."):
            Wsw[kk] = W["blocks.0." + kk[len("blocks.0.txt."):]]
    t2 = {}
    O.dit_step(O.cfg_from_shape(s), Wsw, I["latents"], I["temb"], I["cond"], taps=t2)
    assert float((t2["b0.x_mlp"][:Lc] - want[:Lc]).abs().max()) > 1e-3


def test_gated_mlp_block_by_hand_and_special_case():
    """Gated MLP (R40): x += gate2 (.) (W2 (SiLU(W1 y + b1) (.) (W3 y + b3)) + b2), against torch library routines; with
    W3 = 0, b3 = 1 the second factor is 1 and the branch is W2 SiLU(W1 y + b1) + b2."""
    s = _tiny(n_blocks=1, cond_mode="none", extras={"mlp_gated": True})
    W, I = synth.make_weights(s), synth.make_inputs(s)
    assert "blocks.0.mlp.w3" in W and O.cfg_from_shape(s)["mlp_gated"]
    taps = {}
    O.dit_step(O.cfg_from_shape(s), W, I["latents"], I["temb"], None, taps=taps)
    Fn = torch.nn.functional
    Wd = {k: v.double() for k, v in W.items()}
    D = 32
    c = Fn.linear(Fn.silu(Fn.linear(I["temb"].double(), Wd["t_mlp.w1"], Wd["t_mlp.b1"])), Wd["t_mlp.w2"], Wd["t_mlp.b2"])
    m = Fn.linear(Fn.silu(c), Wd["blocks.0.mod.w"], Wd["blocks.0.mod.b"]).reshape(6, D)
    xa = taps["b0.x_attn"]
    y = Fn.layer_norm(xa, (D,), eps=1e-6) * (1 + m[4]) + m[3]
    u = Fn.silu(Fn.linear(y, Wd["blocks.0.mlp.w1"], Wd["blocks.0.mlp.b1"])) * Fn.linear(y, Wd["blocks.0.mlp.w3"], Wd["blocks.0.mlp.b3"])
    want = xa + m[5] * Fn.linear(u, Wd["blocks.0.mlp.w2"], Wd["blocks.0.mlp.b2"])
    assert torch.allclose(taps["b0.u"], u, rtol=1e-11, atol=1e-13)
    assert torch.allclose(taps["b0.x_mlp"], want, rtol=1e-10, atol=1e-12)
    W1 = dict(W)
    W1["blocks.0.mlp.w3"] = torch.zeros_like(W["blocks.0.mlp.w3"]); W1["blocks.0.mlp.b3"] = torch.ones_like(W["blocks.0.mlp.b3"])
    t1 = {}
    O.dit_step(O.cfg_from_shape(s), W1, I["latents"], I["temb"], None, taps=t1)
    assert torch.allclose(t1["b0.u"], Fn.silu(Fn.linear(t1["b0.y2"], Wd["blocks.0.mlp.w1"], Wd["blocks.0.mlp.b1"])), rtol=1e-12, atol=1e-14)
    # and it is not the GELU block
    s0 = _tiny(n_blocks=1, cond_mode="none")
    t0 = {}
    O.dit_step(O.cfg_from_shape(s0), {k: v for k, v in W.items() if "w3" not in k and "b3" not in k}, I["latents"], I["temb"], None, taps=t0)
    assert float((t0["b0.u"] - taps["b0.u"]).abs().max()) > 1e-3


def test_varlen_is_per_request_and_block_rows():
    s = _tiny(cond_mode="joint", rope_dims=(0, 8, 8), qk_rmsnorm=True)
    W = synth.make_weights(s)
    Is = [synth.make_inputs(s, tag=f"r{i}", t=100.0 * (i + 1)) for i in range(3)]
    outs = O.dit_step_varlen(O.cfg_from_shape(s), W, [i["latents"] for i in Is], [i["temb"] for i in Is],
                             [i["cond"] for i in Is])
    for o, i in zip(outs, Is):
        assert torch.equal(o, O.dit_step(O.cfg_from_shape(s), W, i["latents"], i["temb"], i["cond"]))
    # teacher-forced block on sampled rows == the same rows of the full block
    cfg = O.cfg_from_shape(s)
    taps = {}
    O.dit_step(cfg, W, Is[0]["latents"], Is[0]["temb"], Is[0]["cond"], taps=taps)
    pos = torch.cat([torch.zeros(5, 3, dtype=torch.int64), O.token_positions((1, 4, 4))])
    ang = O.rope_angles(pos, cfg["rope_dims"], cfg["rope_theta"])
    rows = torch.tensor([0, 4, 5, 20])
    got = O.block_rows(cfg, W, 1, taps["b0.x_mlp"], taps["mod"][1], ang, rows)
    assert torch.allclose(got, taps["b1.x_mlp"][rows], rtol=1e-12, atol=1e-14)


# ---------------------------------------------------------------- trajectory (dit_sample)
def _traj_inputs(s, n_steps, seed_tag=""):
    I = synth.make_inputs(s)
    ts = [900.0 - 250.0 * i for i in range(n_steps)]
    tembs = synth.timestep_embedding(ts, s.temb_dim)
    sigmas = [1.0 - (i / n_steps) ** 1.5 for i in range(n_steps + 1)]      # uneven spacing, decreasing to 0
    unc = synth.normal(s.seed, "uncond" + seed_tag, (3, s.cond_dim), dtype=s.torch_dtype)
    return I, tembs, sigmas, unc


def test_sample_constant_velocity_closed_form():
    """final.w = 0 makes v = unpatchify(final.b) whatever x and t are: x_n = x_0 + (sigma_n - sigma_0) v exactly
    (wrong sign of the step, a dropped step or an accumulated-vs-overwritten state all fail this)."""
    s = _tiny()
    W = synth.make_weights(s)
    W["final.w"] = torch.zeros_like(W["final.w"])
    I, tembs, sigmas, _ = _traj_inputs(s, 3)
    cfg = O.cfg_from_shape(s)
    C_, (F_, H_, W_) = s.latent_channels, s.latent_grid
    n_tok = (F_ // s.patch[0]) * (H_ // s.patch[1]) * (W_ // s.patch[2])
    v = O.unpatchify(W["final.b"].double().repeat(n_tok, 1), s.patch, (C_, F_, H_, W_))
    out = O.dit_sample(cfg, W, I["latents"], tembs, sigmas, I["cond"])
    want = I["latents"].double() + (sigmas[-1] - sigmas[0]) * v
    assert torch.allclose(out, want, rtol=0, atol=1e-12)
    assert sigmas[-1] - sigmas[0] == -1.0 and float((out - I["latents"].double() + v).abs().max()) < 1e-12


def test_sample_semigroup_and_single_step():
    """A 3-step trajectory equals three chained 1-step trajectories with the sliced tembs / sigmas (catches a wrong
    temb or sigma index), and one step equals x + dsigma * dit_step."""
    s = _tiny(rope_dims=(0, 8, 8), qk_rmsnorm=True)
    W = synth.make_weights(s)
    I, tembs, sigmas, _ = _traj_inputs(s, 3)
    cfg = O.cfg_from_shape(s)
    full = O.dit_sample(cfg, W, I["latents"], tembs, sigmas, I["cond"])
    x = I["latents"].double()
    for i in range(3):
        x1 = O.dit_sample(cfg, W, x, tembs[i:i + 1], sigmas[i:i + 2], I["cond"])
        v = O.dit_step(cfg, W, x, tembs[i:i + 1], I["cond"])
        assert torch.allclose(x1, x + (sigmas[i + 1] - sigmas[i]) * v, rtol=0, atol=1e-13)
        x = x1
    assert torch.equal(full, x)
    # the steps really differ (tembs and sigmas are not interchangeable): permuting tembs changes the result
    perm = O.dit_sample(cfg, W, I["latents"], tembs.flip(0), sigmas, I["cond"])
    assert float((perm - full).abs().max()) > 1e-6


def test_sample_guidance_special_cases():
    s = _tiny()
    W = synth.make_weights(s)
    I, tembs, sigmas, unc = _traj_inputs(s, 2)
    cfg = O.cfg_from_shape(s)
    lat, cond = I["latents"], I["cond"]
    only_c = O.dit_sample(cfg, W, lat, tembs, sigmas, cond)
    only_u = O.dit_sample(cfg, W, lat, tembs, sigmas, unc)
    assert torch.allclose(O.dit_sample(cfg, W, lat, tembs, sigmas, cond, unc, 1.0), only_c, rtol=0, atol=1e-13)
    assert torch.allclose(O.dit_sample(cfg, W, lat, tembs, sigmas, cond, unc, 0.0), only_u, rtol=0, atol=1e-13)
    assert torch.allclose(O.dit_sample(cfg, W, lat, tembs, sigmas, cond, cond, 7.5), only_c, rtol=0, atol=1e-12)
    # one step: the guided update is affine in the scale, x(g) = x(0) + g (x(1) - x(0))
    g1 = O.dit_sample(cfg, W, lat, tembs[:1], sigmas[:2], cond, unc, 3.0)
    c1 = O.dit_sample(cfg, W, lat, tembs[:1], sigmas[:2], cond)
    u1 = O.dit_sample(cfg, W, lat, tembs[:1], sigmas[:2], unc)
    assert torch.allclose(g1, u1 + 3.0 * (c1 - u1), rtol=0, atol=1e-13)
    assert float((only_c - only_u).abs().max()) > 1e-6


def test_cfg1_shape_facts():
    s = synth.cfg1()
    assert s.n_tokens == 256 and s.n_cond == 32 and s.token_grid == (1, 16, 16)
    assert synth.cfg2().n_tokens == 4096 and synth.cfg3().n_tokens == 32760
    assert [r.n_tokens for r in synth.cfg4_requests()] == list(synth.CFG4_TOKENS)
    I = synth.make_inputs(s)
    assert I["t"] == 500.0 and I["latents"].shape == (4, 1, 32, 32)
    # generator is order independent and deterministic
    a = synth.normal(3, "z", (1000,)); b = synth.normal(3, "z", (1000,), chunk=64)
    assert torch.equal(a, b) and abs(float(a.mean())) < 0.15 and abs(float(a.std()) - 1) < 0.1
