"""Seeded synthetic inputs for the DiT denoising-step path (test / bench infrastructure).

This module holds NONE of the method's arithmetic: it only manufactures the tensors that
BASELINE.json's configs describe (weights N(0, 0.02), latents / cond tokens N(0, 1), timesteps,
the sinusoidal timestep embedding that `dit_step` takes as an INPUT, cu_seqlens) and hands the very
same tensors to both the CPU oracle (`oracle/`) and the CUDA path.  It imports neither.

Generator: counter based, order independent.  Element `i` of the tensor
called `name` under `seed` is Box-Muller of two uniforms hashed (splitmix64 finaliser) from
(seed, crc32(name), i).  Implemented with torch int64 ops so the same code fills a tensor on the
CPU (tests, small) or directly in HBM (bench, GB-sized weights).  The integer hash is bit exact on
every device; the log/cos of Box-Muller may differ by an ulp between devices, which is irrelevant
because a tensor is generated once and then shared by both sides.
"""
from __future__ import annotations

import math
import zlib
from dataclasses import dataclass, field

import torch

_M64 = (1 << 64) - 1


def _i64(v: int) -> int:
    v &= _M64
    return v - (1 << 64) if v >= (1 << 63) else v


_C1 = _i64(0xBF58476D1CE4E5B9)
_C2 = _i64(0x94D049BB133111EB)
_GOLD = _i64(0x9E3779B97F4A7C15)


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """logical shift right on int64 tensors (torch's >> is arithmetic)."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def _mix(z: torch.Tensor) -> torch.Tensor:
    z = (z ^ _lsr(z, 30)) * _C1
    z = (z ^ _lsr(z, 27)) * _C2
    return z ^ _lsr(z, 31)


def _mix_int(z: int) -> int:
    z &= _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def stream_key(seed: int, name: str) -> int:
    return _mix_int(_mix_int(seed + 0x1234567) ^ (zlib.crc32(name.encode()) * 0x9E3779B97F4A7C15))


def uniform01(seed: int, name: str, n: int, device="cpu", lane: int = 0, start: int = 0) -> torch.Tensor:
    """n doubles in (0, 1), elements start .. start+n-1 of stream (seed, name, lane)."""
    key = _i64(stream_key(seed, name) + lane * 0x632BE59BD9B4E019)
    idx = torch.arange(start, start + n, dtype=torch.int64, device=device)
    h = _mix(idx * _GOLD + key)
    return (_lsr(h, 11).to(torch.float64) + 0.5) * (1.0 / (1 << 53))


def normal(seed: int, name: str, shape, std: float = 1.0, mean: float = 0.0,
           dtype=torch.float32, device="cpu", chunk: int = 1 << 26) -> torch.Tensor:
    n = int(math.prod(shape))
    out = torch.empty(n, dtype=dtype, device=device)
    for s in range(0, n, chunk):
        m = min(chunk, n - s)
        u1 = uniform01(seed, name, m, device, 0, s)
        u2 = uniform01(seed, name, m, device, 1, s)
        z = torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)
        out[s:s + m] = (z * std + mean).to(torch.float32).to(dtype)
    return out.reshape(*shape)


# ----------------------------------------------------------------------------------------------
# Workload descriptions (BASELINE.json configs[0..4] = SURVEY cfg 1..5)
# ----------------------------------------------------------------------------------------------
@dataclass
class DiTShape:
    name: str
    dtype: str                  # "f32" | "bf16"
    n_blocks: int
    hidden: int
    n_heads: int
    head_dim: int
    mlp_dim: int
    latent_channels: int
    patch: tuple                # (pf, ph, pw)
    temb_dim: int
    cond_dim: int
    cond_mode: str              # "none" | "joint" | "cross" | "joint2" (dual-stream joint blocks)
    rope_dims: tuple            # per axis (f, h, w); all zero = no RoPE
    qk_rmsnorm: bool
    latent_grid: tuple          # (F, H, W) of the latent (before patching)
    n_cond: int
    seed: int = 0
    rope_theta: float = 10000.0
    ln_eps: float = 1e-6
    rms_eps: float = 1e-6
    extras: dict = field(default_factory=dict)

    @property
    def torch_dtype(self):
        return torch.float32 if self.dtype == "f32" else torch.bfloat16

    @property
    def patch_volume(self):
        return self.patch[0] * self.patch[1] * self.patch[2]

    @property
    def token_grid(self):
        return tuple(g // p for g, p in zip(self.latent_grid, self.patch))

    @property
    def n_tokens(self):
        f, h, w = self.token_grid
        return f * h * w


def cfg1(**kw) -> DiTShape:
    """BASELINE.json configs[0]: tiny fp32 DiT (2 blocks, D=256, 4x64), 256 + 32 tokens, t=500."""
    d = dict(name="cfg1_tiny_f32", dtype="f32", n_blocks=2, hidden=256, n_heads=4, head_dim=64,
             mlp_dim=1024, latent_channels=4, patch=(1, 2, 2), temb_dim=256, cond_dim=256,
             cond_mode="joint", rope_dims=(0, 0, 0), qk_rmsnorm=False, latent_grid=(1, 32, 32),
             n_cond=32, seed=0, extras={"t": 500.0})
    d.update(kw)
    return DiTShape(**d)


def cfg2(**kw) -> DiTShape:
    """configs[1]: image DiT bf16, 8 blocks, D=3072, 24x128, 4096 + 256 joint tokens."""
    d = dict(name="cfg2_image_bf16", dtype="bf16", n_blocks=8, hidden=3072, n_heads=24, head_dim=128,
             mlp_dim=12288, latent_channels=16, patch=(1, 2, 2), temb_dim=256, cond_dim=3072,
             cond_mode="joint", rope_dims=(0, 64, 64), qk_rmsnorm=True, latent_grid=(1, 128, 128),
             n_cond=256, seed=0)
    d.update(kw)
    return DiTShape(**d)


def cfg3(**kw) -> DiTShape:
    """configs[2]: video DiT bf16, 4 blocks, D=5120, 40x128, ffn 13824, 32760 tokens, cross-attn 512."""
    d = dict(name="cfg3_video_bf16", dtype="bf16", n_blocks=4, hidden=5120, n_heads=40, head_dim=128,
             mlp_dim=13824, latent_channels=16, patch=(1, 2, 2), temb_dim=256, cond_dim=5120,
             cond_mode="cross", rope_dims=(44, 42, 42), qk_rmsnorm=True, latent_grid=(21, 60, 104),
             n_cond=512, seed=0)
    d.update(kw)
    return DiTShape(**d)


CFG4_TOKENS = (1024, 1024, 4096, 4096, 9216, 16384)      # configs[3]; grids 32^2 .. 128^2, patch 2


def cfg4_requests(tokens=CFG4_TOKENS, **kw):
    """configs[3]: six heterogeneous requests, cfg2 block shape, seed 7, 256 cond tokens each (R15)."""
    reqs = []
    for n in tokens:
        side = int(round(math.sqrt(n)))
        assert side * side == n
        reqs.append(cfg2(name=f"cfg4_req{len(reqs)}_{n}", latent_grid=(1, 2 * side, 2 * side), seed=7, **kw))
    return reqs


# ----------------------------------------------------------------------------------------------
# Weights / inputs
# ----------------------------------------------------------------------------------------------
def weight_shapes(s: DiTShape) -> dict:
    """name -> shape.  Linear weights are [out, in] row-major (K-major for both GEMM operands)."""
    D, F, d, pvC = s.hidden, s.mlp_dim, s.head_dim, s.patch_volume * s.latent_channels
    w = {"t_mlp.w1": (D, s.temb_dim), "t_mlp.b1": (D,), "t_mlp.w2": (D, D), "t_mlp.b2": (D,),
         "patch_embed.w": (D, pvC), "patch_embed.b": (D,)}
    if s.cond_mode != "none":
        w["cond_proj.w"] = (D, s.cond_dim)
        w["cond_proj.b"] = (D,)
    for l in range(s.n_blocks):
        p = f"blocks.{l}."
        w[p + "mod.w"] = (6 * D, D); w[p + "mod.b"] = (6 * D,)
        w[p + "attn.wqkv"] = (3 * D, D); w[p + "attn.bqkv"] = (3 * D,)
        if s.qk_rmsnorm:
            w[p + "attn.gq"] = (d,); w[p + "attn.gk"] = (d,)
        w[p + "attn.wo"] = (D, D); w[p + "attn.bo"] = (D,)
        if s.cond_mode == "cross":
            w[p + "cross.wq"] = (D, D); w[p + "cross.bq"] = (D,)
            w[p + "cross.wkv"] = (2 * D, D); w[p + "cross.bkv"] = (2 * D,)
            w[p + "cross.gq"] = (d,); w[p + "cross.gk"] = (d,)
            w[p + "cross.wo"] = (D, D); w[p + "cross.bo"] = (D,)
        w[p + "mlp.w1"] = (F, D); w[p + "mlp.b1"] = (F,)
        w[p + "mlp.w2"] = (D, F); w[p + "mlp.b2"] = (D,)
        if s.extras.get("mlp_gated"):    # gated MLP (SwiGLU): the second up-projection
            w[p + "mlp.w3"] = (F, D); w[p + "mlp.b3"] = (F,)
        if s.cond_mode == "joint2":      # dual-stream blocks: the text stream's own copy of every per-block tensor
            for k in [k for k in w if k.startswith(p) and not k.startswith(p + "txt.")]:
                w[p + "txt." + k[len(p):]] = w[k]
    w["final.mod.w"] = (2 * D, D); w["final.mod.b"] = (2 * D,)
    w["final.w"] = (pvC, D); w["final.b"] = (pvC,)
    return w


def make_weights(s: DiTShape, device="cpu", std: float = 0.02, seed=None) -> dict:
    """Every Linear weight AND bias ~ N(0, 0.02) (R14); norm gains g = 1 + N(0, 0.02); config dtype."""
    seed = s.seed if seed is None else seed
    out = {}
    for name, shape in weight_shapes(s).items():
        is_gain = name.endswith(".gq") or name.endswith(".gk")
        out[name] = normal(seed, "w:" + name, shape, std=std, mean=1.0 if is_gain else 0.0,
                           dtype=s.torch_dtype, device=device)
    return out


def timestep_embedding(t, dim: int, device="cpu") -> torch.Tensor:
    """[R, dim] fp32 = concat(cos(t w_i), sin(t w_i)), w_i = exp(-ln(1e4) i / (dim/2)) (R16).
    An INPUT of dit_step (BASELINE.json: dit_step(latents, timestep_emb, cond_tokens, out))."""
    t = torch.as_tensor(t, dtype=torch.float64, device=device).reshape(-1, 1)
    half = dim // 2
    w = torch.exp(-math.log(10000.0) * torch.arange(half, dtype=torch.float64, device=device) / half)
    a = t * w
    return torch.cat([torch.cos(a), torch.sin(a)], dim=1).to(torch.float32)


def make_inputs(s: DiTShape, device="cpu", t=None, tag: str = "") -> dict:
    F_, H_, W_ = s.latent_grid
    lat = normal(s.seed, f"latents{tag}", (s.latent_channels, F_, H_, W_), dtype=s.torch_dtype, device=device)
    cond = None
    if s.cond_mode != "none":
        cond = normal(s.seed, f"cond{tag}", (s.n_cond, s.cond_dim), dtype=s.torch_dtype, device=device)
    if t is None:
        t = s.extras.get("t")
    if t is None:
        t = float(uniform01(s.seed, f"t{tag}", 1)[0]) * 1000.0
    return {"latents": lat, "cond": cond, "t": float(t),
            "temb": timestep_embedding([t], s.temb_dim, device=device)}


def make_attention_qkv(seed: int, n_q: int, n_k: int, n_heads: int, head_dim: int, dtype=torch.bfloat16,
                       device="cpu", logit_gain: float = 1.0):
    """cfg 5 tensors: q, k, v ~ N(0, 1), [N, H, d]; logit_gain > 1 gives the 'peaky' variant."""
    q = normal(seed, "attn.q", (n_q, n_heads, head_dim), std=logit_gain, dtype=dtype, device=device)
    k = normal(seed, "attn.k", (n_k, n_heads, head_dim), dtype=dtype, device=device)
    v = normal(seed, "attn.v", (n_k, n_heads, head_dim), dtype=dtype, device=device)
    return q, k, v
