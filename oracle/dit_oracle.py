"""CPU oracle for one DiT denoising step — TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s cpu_baseline / `--impl reference` legs may
import this module.  It shares no code with the CUDA path (`paper_2606_13501_b200/csrc`, `binding.py`)
and imports nothing from the package.

What it is: the *plain definition* of the computation, written with PyTorch CPU ops in float64
(SURVEY.md §8(c)); a library matmul / exp / sum serves as a step, nothing is tiled, fused, made "online"
or re-ordered.  Attention materialises the full score matrix of a head and applies the textbook
softmax; the split-P form computes P independent partials and merges them with the log-sum-exp rule.

Authority: PAPER.md says of the step only that it is a "compute-intensive denoising stage" that
"dominates execution time" (§1) and "performs bidirectional computation over the entire
latent sequence" (§2.1), run under sequence parallelism with all-gather/all-to-all
(§4.1).  The DiT mathematics is fixed by BASELINE.json `north_star` / `configs` and the
readings R1-R23 of SURVEY.md §8(c), restated in DESIGN.md §3; each function cites the reading it follows.

Pins (tests/test_oracle_pins.py, `-m "not gpu"`): brute-force attention in pure Python on tiny inputs;
softmax rows sum to 1; identical keys -> mean of V; zero gates -> identity (bit exact); split-P
invariance; merge closed forms; LN / RMSNorm / RoPE / GELU / patchify invariants; torch library routines
(layer_norm, scaled_dot_product_attention, gelu(tanh), silu) as special cases; stored hand-computed
fixtures under tests/golden/; the trajectory (`dit_sample`): constant-velocity closed form, guidance special cases,
semigroup property; the block in all three modes re-derived with torch library routines and a by-hand RoPE
(`test_dual_stream_*`: the dual-stream block against a torch-library transcription and against the single-stream block
with the same weights in both streams; `test_block_by_hand_one_block`, `test_joint_block_by_hand_rmsnorm_then_rope`: [ctx ; x] order, cond position 0,
RMSNorm BEFORE RoPE, interleaved pairs; `test_cross_block_by_hand`: wkv rows [k | v], ungated / unmodulated / un-roped
cross branch, also for `block_rows` in cross mode).  Mutants of each of those lines fail the CPU suite.
PARITY UNPINNED: the *composition order* of the block (R1, R9, R10, R12: which sub-layer follows which,
single-stream joint attention, cross-attention placement, final layer) is a definition this repo makes
— the paper prints nothing it could be checked against; the transcriptions above pin the oracle to DESIGN.md §3's
sentences, not to the paper.
"""
from __future__ import annotations

import math

import torch

F64 = torch.float64


def _d(x):
    return x.to(F64) if x is not None else None


# ------------------------------------------------------------------------------------------------
# primitives
# ------------------------------------------------------------------------------------------------
def silu(z):
    """SiLU(z) = z / (1 + e^-z)."""
    return z / (1.0 + torch.exp(-z))


def gelu_tanh(z):
    """GELU_tanh(z) = 0.5 z (1 + tanh(0.7978845608028654 (z + 0.044715 z^3)))  (§8(c) step 5)."""
    return 0.5 * z * (1.0 + torch.tanh(0.7978845608028654 * (z + 0.044715 * z ** 3)))


def mlp(cfg, W, pre, y):
    """The block's MLP branch before the gated residual (§8(c) step 5).  Default: W2 GELU_tanh(W1 y + b1) + b2.
    `mlp_gated` (SURVEY.md §8(f) item 2 "gated-MLP variants", reading R40): the SwiGLU form
    W2 (SiLU(W1 y + b1) (.) (W3 y + b3)) + b2.  Returns (u, W2 u + b2)."""
    if cfg.get("mlp_gated"):
        u = silu(linear(y, W[pre + "mlp.w1"], W[pre + "mlp.b1"])) * linear(y, W[pre + "mlp.w3"], W[pre + "mlp.b3"])
    else:
        u = gelu_tanh(linear(y, W[pre + "mlp.w1"], W[pre + "mlp.b1"]))
    return u, linear(u, W[pre + "mlp.w2"], W[pre + "mlp.b2"])


def layer_norm(x, eps):
    """LN(x) = (x - mu) / sqrt(var + eps), biased variance over the last dim, no affine (R4)."""
    mu = x.mean(dim=-1, keepdim=True)
    var = ((x - mu) ** 2).mean(dim=-1, keepdim=True)
    return (x - mu) / torch.sqrt(var + eps)


def modulate(x, shift, scale, eps):
    """adaLN: y = LN(x) * (1 + scale) + shift  (R3: '1 + scale')."""
    return layer_norm(x, eps) * (1.0 + scale) + shift


def rms_norm_heads(x, g, eps):
    """QK-RMSNorm per token per head over d (R5): x / sqrt(mean_d(x^2) + eps) * g.  x: [T, H, d], g: [d]."""
    ms = (x ** 2).mean(dim=-1, keepdim=True)
    return x / torch.sqrt(ms + eps) * g


def linear(x, w, b=None):
    """y = x W^T + b; W is [out, in]."""
    y = x @ _d(w).t()
    return y + _d(b) if b is not None else y


def rope_angles(pos, rope_dims, theta):
    """R6. pos: [T, 3] integer (f, h, w) coordinates.  Returns angle[T, d/2] (float64).
    The head dim is cut into contiguous per-axis segments of rope_dims[a] dims in order (f, h, w);
    inside a segment of d_a dims pair j covers elements (2j, 2j+1) and rotates by pos_a * theta^(-2j/d_a)."""
    cols = []
    for a, d_a in enumerate(rope_dims):
        if d_a == 0:
            continue
        j = torch.arange(d_a // 2, dtype=F64)
        omega = theta ** (-2.0 * j / d_a)
        cols.append(pos[:, a].to(F64)[:, None] * omega[None, :])
    return torch.cat(cols, dim=1)


def apply_rope(x, ang):
    """(a, b) -> (a cos - b sin, a sin + b cos) on interleaved pairs.  x: [T, H, d], ang: [T, d/2]."""
    a, b = x[..., 0::2], x[..., 1::2]
    c, s = torch.cos(ang)[:, None, :], torch.sin(ang)[:, None, :]
    out = torch.empty_like(x)
    out[..., 0::2] = a * c - b * s
    out[..., 1::2] = a * s + b * c
    return out


def token_positions(token_grid):
    """Patch-grid coordinates of token n = (f' H' + h') W' + w'  (§8(c) step 3) -> [N, 3]."""
    Fp, Hp, Wp = token_grid
    f, h, w = torch.meshgrid(torch.arange(Fp), torch.arange(Hp), torch.arange(Wp), indexing="ij")
    return torch.stack([f.reshape(-1), h.reshape(-1), w.reshape(-1)], dim=1)


# ------------------------------------------------------------------------------------------------
# attention: plain definition, partials, merge
# ------------------------------------------------------------------------------------------------
def attention(q, k, v, scale=None):
    """Non-causal full attention, plain definition (§8(c) step 5, R7, R18).
    q: [Nq, H, d], k, v: [Nk, H, d]  ->  o [Nq, H, d], lse [Nq, H]  (all float64).
    s_ij = q_i.k_j * scale; p = softmax_j(s); o_i = sum_j p_ij v_j; lse_i = ln sum_j e^{s_ij}.
    Nk = 0 gives o = 0, lse = -inf (R18)."""
    q, k, v = _d(q), _d(k), _d(v)
    Nq, H, d = q.shape
    if scale is None:
        scale = 1.0 / math.sqrt(d)
    if k.shape[0] == 0:
        return torch.zeros(Nq, H, v.shape[-1], dtype=F64), torch.full((Nq, H), -math.inf, dtype=F64)
    o = torch.empty(Nq, H, v.shape[-1], dtype=F64)
    lse = torch.empty(Nq, H, dtype=F64)
    for h in range(H):                                             # one head at a time (memory only)
        s = (q[:, h, :] @ k[:, h, :].t()) * scale                  # [Nq, Nk] full score matrix of the head
        m = s.max(dim=-1, keepdim=True).values
        e = torch.exp(s - m)
        z = e.sum(dim=-1, keepdim=True)
        p = e / z
        o[:, h, :] = p @ v[:, h, :]
        lse[:, h] = (m + torch.log(z)).squeeze(-1)
    return o, lse


def merge_partials(o_parts, lse_parts):
    """LSE merge (§8(c) step 7, R18): lse = ln sum_p e^{lse_p};  o = sum_p e^{lse_p - lse} o_p.
    Shards with lse_p = -inf contribute nothing; if every shard is -inf the result is o = 0, lse = -inf."""
    L = torch.stack([_d(l) for l in lse_parts], dim=0)             # [P, Nq, H]
    O = torch.stack([_d(o) for o in o_parts], dim=0)               # [P, Nq, H, d]
    m = L.max(dim=0).values
    m_safe = torch.where(torch.isinf(m), torch.zeros_like(m), m)
    w = torch.exp(L - m_safe)                                      # e^{-inf} = 0
    z = w.sum(dim=0)
    lse = m_safe + torch.log(z)                                    # log(0) = -inf when all shards are empty
    wn = torch.where(z > 0, w / torch.where(z > 0, z, torch.ones_like(z)), torch.zeros_like(w))
    o = (wn[..., None] * O).sum(dim=0)
    return o, lse


def shard_bounds(n, P):
    """R20: P contiguous shards of size ceil(n / P), the last one shorter (possibly empty)."""
    sz = -(-n // P)
    return [(min(p * sz, n), min((p + 1) * sz, n)) for p in range(P)]


def relayout(shards, p_dst):
    """Re-layout of a row-sharded artifact between split degrees (§5.3): the P
    source shards are the R20 row ranges of ONE logical tensor, the result is its P' R20 row ranges — the plain
    definition: put the rows back together, cut them again."""
    full = torch.cat(list(shards), dim=0)
    return [full[a:b] for a, b in shard_bounds(full.shape[0], p_dst)]


def attention_split(q, k, v, P, scale=None):
    """§8(c) step 7: P independent partials over contiguous KV shards, then merge.  P = 1 == attention()."""
    parts = [attention(q, k[a:b], v[a:b], scale) for a, b in shard_bounds(k.shape[0], P)]
    return merge_partials([p[0] for p in parts], [p[1] for p in parts])


# ------------------------------------------------------------------------------------------------
# patchify / unpatchify
# ------------------------------------------------------------------------------------------------
def patchify(lat, patch):
    """§8(c) step 3 / R11.  lat: [C, F, H, W] -> [N, C*pf*ph*pw]; token n = (f' H' + h') W' + w',
    feature ((c pf + i) ph + j) pw + k  (conv-weight flatten order)."""
    C, F_, H_, W_ = lat.shape
    pf, ph, pw = patch
    x = lat.reshape(C, F_ // pf, pf, H_ // ph, ph, W_ // pw, pw)
    x = x.permute(1, 3, 5, 0, 2, 4, 6)                             # f' h' w' c i j k
    return x.reshape((F_ // pf) * (H_ // ph) * (W_ // pw), C * pf * ph * pw)


def unpatchify(tok, patch, latent_shape):
    """Inverse of patchify: [N, C*pv] -> [C, F, H, W]."""
    C, F_, H_, W_ = latent_shape
    pf, ph, pw = patch
    x = tok.reshape(F_ // pf, H_ // ph, W_ // pw, C, pf, ph, pw)
    x = x.permute(3, 0, 4, 1, 5, 2, 6)                             # c f' i h' j w' k
    return x.reshape(C, F_, H_, W_)


# ------------------------------------------------------------------------------------------------
# the step
# ------------------------------------------------------------------------------------------------
def conditioning(cfg, W, temb):
    """§8(c) steps 1-2 (R2): c = W2 SiLU(W1 temb + b1) + b2;  mod_l = Wmod_l SiLU(c) + bmod_l."""
    c = linear(silu(linear(_d(temb).reshape(1, -1), W["t_mlp.w1"], W["t_mlp.b1"])), W["t_mlp.w2"], W["t_mlp.b2"])
    sc = silu(c)
    mods = [linear(sc, W[f"blocks.{l}.mod.w"], W[f"blocks.{l}.mod.b"]).reshape(6, -1) for l in range(cfg["n_blocks"])]
    modf = linear(sc, W["final.mod.w"], W["final.mod.b"]).reshape(2, -1)
    return c.reshape(-1), mods, modf


def conditioning_txt(cfg, W, c):
    """Dual-stream blocks (R37): the text stream's own modulation, mod_txt_l = Wmod_txt_l SiLU(c) + bmod_txt_l (6 chunks
    in the same order as the image stream's)."""
    sc = silu(_d(c).reshape(1, -1))
    return [linear(sc, W[f"blocks.{l}.txt.mod.w"], W[f"blocks.{l}.txt.mod.b"]).reshape(6, -1) for l in range(cfg["n_blocks"])]


def dual_stream_block(cfg, W, l, x, Lc, m_img, m_txt, ang, split_p, taps):
    """One DUAL-STREAM joint block (reading R37 — the MMDiT form of the models the paper
    serves): the text rows x[:Lc] and the image rows x[Lc:] each have their OWN modulation, QKV projection
    (and QK-RMSNorm gains), out-projection and MLP (`blocks.l.txt.*` / `blocks.l.*`); ONE attention runs over the joint
    sequence [txt ; img] (RoPE as in the single-stream block: text rows at position 0).  Everything else is step 5."""
    D, H, d, eps = cfg["hidden"], cfg["n_heads"], cfg["head_dim"], cfg["ln_eps"]
    parts = (("txt", f"blocks.{l}.txt.", x[:Lc], m_txt), ("img", f"blocks.{l}.", x[Lc:], m_img))
    qs, ks, vs = [], [], []
    for name, pre, xs, m in parts:
        y1 = modulate(xs, m[0], m[1], eps)
        qkv = linear(y1, W[pre + "attn.wqkv"], W[pre + "attn.bqkv"])
        q, k, v = (qkv[:, i * D:(i + 1) * D].reshape(-1, H, d) for i in range(3))
        if cfg["qk_rmsnorm"]:
            q = rms_norm_heads(q, _d(W[pre + "attn.gq"]), cfg["rms_eps"])
            k = rms_norm_heads(k, _d(W[pre + "attn.gk"]), cfg["rms_eps"])
        qs.append(q); ks.append(k); vs.append(v)
        if taps is not None:
            taps[f"b{l}.{name}.y1"] = y1
    q, k, v = torch.cat(qs, 0), torch.cat(ks, 0), torch.cat(vs, 0)               # [txt ; img]
    if ang is not None:
        q, k = apply_rope(q, ang), apply_rope(k, ang)
    o, _ = attention_split(q, k, v, split_p)
    o = o.reshape(-1, D)
    if taps is not None:
        taps[f"b{l}.q"], taps[f"b{l}.k"], taps[f"b{l}.v"], taps[f"b{l}.o"] = q.reshape(-1, D), k.reshape(-1, D), v.reshape(-1, D), o
    outs = []
    for (name, pre, xs, m), os_ in zip(parts, (o[:Lc], o[Lc:])):
        xa = xs + m[2] * linear(os_, W[pre + "attn.wo"], W[pre + "attn.bo"])
        y2 = modulate(xa, m[3], m[4], eps)
        u, hm = mlp(cfg, W, pre, y2)
        outs.append(xa + m[5] * hm)
        if taps is not None:
            taps[f"b{l}.{name}.x_attn"], taps[f"b{l}.{name}.y2"], taps[f"b{l}.{name}.u"] = xa, y2, u
    x = torch.cat(outs, 0)
    if taps is not None:
        taps[f"b{l}.x_mlp"] = x.clone()
    return x


def self_attention_block(cfg, W, l, y, ang, split_p, taps, rows=None):
    """§8(c) step 5, attention half: q,k,v = split(Wqkv y + b); QK-RMSNorm (R5); RoPE (R6); softmax(QK^T/sqrt d)V.
    `rows` (optional index tensor) restricts the QUERY rows (sampled-row checks at large sizes);
    keys/values always cover the whole sequence."""
    D, H, d = cfg["hidden"], cfg["n_heads"], cfg["head_dim"]
    p = f"blocks.{l}.attn."
    qkv = linear(y, W[p + "wqkv"], W[p + "bqkv"])
    T = y.shape[0]
    q, k, v = (qkv[:, i * D:(i + 1) * D].reshape(T, H, d) for i in range(3))
    if cfg["qk_rmsnorm"]:
        q = rms_norm_heads(q, _d(W[p + "gq"]), cfg["rms_eps"])
        k = rms_norm_heads(k, _d(W[p + "gk"]), cfg["rms_eps"])
    if ang is not None:
        q, k = apply_rope(q, ang), apply_rope(k, ang)
    if taps is not None:
        taps[f"b{l}.q"], taps[f"b{l}.k"], taps[f"b{l}.v"] = q.reshape(T, D), k.reshape(T, D), v.reshape(T, D)
    if rows is not None:
        q = q[rows]
    o, lse = attention_split(q, k, v, split_p)
    return o.reshape(-1, D), lse


def dit_step(cfg, W, latents, temb, cond=None, split_p=1, taps=None):
    """One denoising step for one request (§8(c) steps 1-7).  cfg: dict with keys
    n_blocks, hidden, n_heads, head_dim, mlp_dim, patch, cond_mode, rope_dims, rope_theta, ln_eps,
    rms_eps, qk_rmsnorm.  W: name -> tensor ([out, in] Linear weights).  latents: [C, F, H, W].
    Returns `out` with the latent's shape (float64).  If `taps` is a dict it receives intermediates."""
    D = cfg["hidden"]
    eps = cfg["ln_eps"]
    lat = _d(latents)
    C, F_, H_, W_ = lat.shape
    pf, ph, pw = cfg["patch"]
    grid = (F_ // pf, H_ // ph, W_ // pw)
    c, mods, modf = conditioning(cfg, W, temb)
    x = linear(patchify(lat, cfg["patch"]), W["patch_embed.w"], W["patch_embed.b"])            # step 3
    N = x.shape[0]
    mode = cfg["cond_mode"]
    ctx = None
    Lc = 0
    if mode != "none":
        ctx = linear(_d(cond), W["cond_proj.w"], W["cond_proj.b"])                               # step 4
    if mode in ("joint", "joint2"):
        Lc = ctx.shape[0]
        x = torch.cat([ctx, x], dim=0)                                                            # [ctx ; x] (R9)
    mods_txt = conditioning_txt(cfg, W, c) if mode == "joint2" else None
    ang = None
    if sum(cfg["rope_dims"]) > 0:
        pos = token_positions(grid)
        if Lc:
            pos = torch.cat([torch.zeros(Lc, 3, dtype=pos.dtype), pos], dim=0)                    # cond pos = 0 (R6)
        ang = rope_angles(pos, cfg["rope_dims"], cfg["rope_theta"])
    if taps is not None:
        taps["c"], taps["x0"] = c, x.clone()
        taps["mod"] = torch.stack(mods, 0) if mods else torch.zeros(0, 6, D, dtype=F64)
        taps["modf"] = modf
    for l in range(cfg["n_blocks"]):
        if mode == "joint2":                                                                      # dual-stream block (R37)
            x = dual_stream_block(cfg, W, l, x, Lc, mods[l], mods_txt[l], ang, split_p, taps)
            continue
        sh1, sc1, g1, sh2, sc2, g2 = mods[l]                                                      # step 2 order
        y1 = modulate(x, sh1, sc1, eps)
        o, _ = self_attention_block(cfg, W, l, y1, ang, split_p, taps)
        x = x + g1 * linear(o, W[f"blocks.{l}.attn.wo"], W[f"blocks.{l}.attn.bo"])
        if taps is not None:
            taps[f"b{l}.y1"], taps[f"b{l}.o"], taps[f"b{l}.x_attn"] = y1, o, x.clone()
        if mode == "cross":                                                                       # R10
            p = f"blocks.{l}.cross."
            H, d = cfg["n_heads"], cfg["head_dim"]
            qc = linear(layer_norm(x, eps), W[p + "wq"], W[p + "bq"]).reshape(-1, H, d)
            kv = linear(ctx, W[p + "wkv"], W[p + "bkv"])
            kc, vc = kv[:, :D].reshape(-1, H, d), kv[:, D:].reshape(-1, H, d)
            qc = rms_norm_heads(qc, _d(W[p + "gq"]), cfg["rms_eps"])
            kc = rms_norm_heads(kc, _d(W[p + "gk"]), cfg["rms_eps"])
            oc, _ = attention(qc, kc, vc)
            x = x + linear(oc.reshape(-1, D), W[p + "wo"], W[p + "bo"])
            if taps is not None:
                taps[f"b{l}.oc"], taps[f"b{l}.x_cross"] = oc.reshape(-1, D), x.clone()
        y2 = modulate(x, sh2, sc2, eps)
        u, hm = mlp(cfg, W, f"blocks.{l}.", y2)
        x = x + g2 * hm
        if taps is not None:
            taps[f"b{l}.y2"], taps[f"b{l}.u"], taps[f"b{l}.x_mlp"] = y2, u, x.clone()
    xi = x[Lc:]                                                                                   # image tokens only
    yf = modulate(xi, modf[0], modf[1], eps)
    tok = linear(yf, W["final.w"], W["final.b"])                                                  # step 6
    if taps is not None:
        taps["yf"], taps["tok"] = yf, tok
    return unpatchify(tok, cfg["patch"], (C, F_, H_, W_))


def dit_step_varlen(cfg, W, latents_list, temb_list, cond_list, split_p=1):
    """§8(c) step 8: packing is DEFINED as running every request on its own."""
    return [dit_step(cfg, W, lat, te, co, split_p) for lat, te, co in zip(latents_list, temb_list, cond_list)]


def dit_sample(cfg, W, latents, tembs, sigmas, cond=None, uncond=None, guidance_scale=1.0, split_p=1):
    """One request's denoising trajectory (§3.1: a request is a chain of trajectory tasks, one per
    denoising step; DESIGN.md §3 step 9, readings R30-R32).  tembs [n_steps, temb_dim],
    sigmas n_steps + 1 numbers.  Step i:  v = dit_step(x_i, tembs[i], cond); with `uncond` given (classifier-free
    guidance)  v = v_u + guidance_scale (v - v_u),  v_u = dit_step(x_i, tembs[i], uncond);  flow-matching Euler update
    x_{i+1} = x_i + (sigmas[i+1] - sigmas[i]) v.  Returns x_{n_steps} (float64).
    Pins: closed form for a constant velocity field, guidance special cases (scale 0 / 1, cond == uncond), the
    semigroup property (a trajectory equals the chained single-step trajectories)."""
    x = _d(latents).clone()
    n_steps = len(sigmas) - 1
    assert tembs.shape[0] == n_steps
    for i in range(n_steps):
        te = tembs[i:i + 1]
        v = dit_step(cfg, W, x, te, cond, split_p)
        if uncond is not None:
            vu = dit_step(cfg, W, x, te, uncond, split_p)
            v = vu + float(guidance_scale) * (v - vu)
        x = x + (float(sigmas[i + 1]) - float(sigmas[i])) * v
    return x


def block_rows(cfg, W, l, x_in, mods_l, ang, rows, ctx=None):
    """Teacher-forced check of one block at full size on sampled rows (SURVEY §8(d) plan (b)):
    given the block input x_in [T, D] (all rows: K and V need them), return the block output for `rows`."""
    D, eps = cfg["hidden"], cfg["ln_eps"]
    x_in = _d(x_in)
    sh1, sc1, g1, sh2, sc2, g2 = mods_l
    y1 = modulate(x_in, sh1, sc1, eps)
    o, _ = self_attention_block(cfg, W, l, y1, ang, 1, None, rows=rows)
    x = x_in[rows] + g1 * linear(o, W[f"blocks.{l}.attn.wo"], W[f"blocks.{l}.attn.bo"])
    if cfg["cond_mode"] == "cross":
        p = f"blocks.{l}.cross."
        H, d = cfg["n_heads"], cfg["head_dim"]
        qc = linear(layer_norm(x, eps), W[p + "wq"], W[p + "bq"]).reshape(-1, H, d)
        kv = linear(_d(ctx), W[p + "wkv"], W[p + "bkv"])
        kc, vc = kv[:, :D].reshape(-1, H, d), kv[:, D:].reshape(-1, H, d)
        qc = rms_norm_heads(qc, _d(W[p + "gq"]), cfg["rms_eps"])
        kc = rms_norm_heads(kc, _d(W[p + "gk"]), cfg["rms_eps"])
        oc, _ = attention(qc, kc, vc)
        x = x + linear(oc.reshape(-1, D), W[p + "wo"], W[p + "bo"])
    y2 = modulate(x, sh2, sc2, eps)
    return x + g2 * mlp(cfg, W, f"blocks.{l}.", y2)[1]


def cfg_from_shape(s):
    """Plain dict view of a synth.DiTShape (duck-typed; the oracle does not import the package)."""
    return dict(n_blocks=s.n_blocks, hidden=s.hidden, n_heads=s.n_heads, head_dim=s.head_dim, mlp_dim=s.mlp_dim,
                patch=tuple(s.patch), cond_mode=s.cond_mode, rope_dims=tuple(s.rope_dims), rope_theta=s.rope_theta,
                ln_eps=s.ln_eps, rms_eps=s.rms_eps, qk_rmsnorm=bool(s.qk_rmsnorm), mlp_gated=bool(s.extras.get("mlp_gated", False)))
