"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (same dit_config, same
weights recipe, whole 8- / 4-block model resident), END TO END against the oracle:
  cfg 2  the whole 8-block step against O.dit_step (whole tensors: `out`, and the residual stream after every block —
         the accumulation curve of the error across blocks);
  cfg 3  the whole 4-block step against sampled rows of ONE full oracle step stored in tests/golden/cfg3_oracle_rows.pt
         (written by tests/golden/make_fullsize_oracle.py from oracle/ only: 168 TFLOP of fp64 do not fit in a test run),
         plus every block teacher-forced on sampled rows (oracle.block_rows: the block's input is read back from the
         GPU, keys / values cover the whole sequence, queries and everything after attention only the sampled rows);
  cfg 4  requests 0-3 of the PACKED step against O.dit_step of each request, the 16384-token request's blocks
         teacher-forced on sampled rows, and packing invariance for all six;
  cfg 5  sampled query rows against the plain definition over all keys up to N = 131072, split-KV P = 2 / 4 / 8.
Measured errors are printed (pytest -s) and, when DIT_PARITY_LOG names a file, appended to it as JSON lines."""
import json
import os
import time

import pytest
import torch

from oracle import dit_oracle as O
from paper_2606_13501_b200 import binding as B
from paper_2606_13501_b200 import synth
from util import check, errors

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _host_gb():
    try:
        import psutil
        return psutil.virtual_memory().available / 2 ** 30
    except Exception:
        return 0.0


def _log(**kw):
    print(json.dumps(kw))
    path = os.environ.get("DIT_PARITY_LOG")
    if path:
        with open(path, "a") as f:
            f.write(json.dumps(kw) + "\n")


class KeepTaps(dict):
    """taps dict that keeps only the named oracle intermediates (the others are 0.1-4 GB each at these sizes)."""

    def __init__(self, keep):
        super().__init__()
        self.keep = set(keep)

    def __setitem__(self, k, v):
        if k in self.keep:
            super().__setitem__(k, v)


def _assert_same_generator_on_both_devices(s):
    """The stored oracle rows were computed from CPU-generated tensors, the GPU test generates in HBM: the integer hash
    is bit exact and the fp64 log / cos may differ by an ulp of fp64, which does not survive the rounding to fp32 /
    bf16 — checked here on a slice instead of assumed."""
    for name, shape in (("w:blocks.0.attn.wqkv", (1 << 20,)), ("latents", (1 << 18,)), ("w:blocks.1.cross.gk", (128,))):
        a = synth.normal(s.seed, name, shape, std=0.02, dtype=s.torch_dtype)
        b = synth.normal(s.seed, name, shape, std=0.02, dtype=s.torch_dtype, device=DEV).cpu()
        assert torch.equal(a, b), f"generator differs between CPU and GPU for {name}"


def _block_weights_cpu(W, l):
    """Only block l's tensors travel to the host (the full cfg 3 model is 8 GB)."""
    return {k: v.cpu() for k, v in W.items() if k.startswith(f"blocks.{l}.")}


def _x_taps(m, step, T, D, L, stage):
    """The residual stream [T, D] after `stage` of every block (one debug-stopped step per block)."""
    xs = []
    for l in range(L):
        m.dit_debug_stop_after(l, stage)
        step()
        xs.append(m.dit_get_tap("x", (T, D), torch.float32))
    m.dit_debug_stop_after(-1, 0)
    torch.cuda.synchronize()
    return xs


def _teacher_forced_blocks(s, m, W, I, step, blocks, rows, what, T, row0=0, mod_row=0, n_req=1):
    """Blocks `blocks` of a resident model, each teacher-forced: block input x_l (all rows of the request: K and V need
    them) is read back from the GPU, the oracle computes the block output for `rows`, compared with the GPU's x_{l+1}.
    row0 / T select the request inside a packed sequence (T_total rows), mod_row its modulation row."""
    D, L = s.hidden, s.n_blocks
    joint = s.cond_mode == "joint"
    Tr = s.n_tokens + (s.n_cond if joint else 0)
    cfg = O.cfg_from_shape(s)
    mod_len = L * 6 * D + 2 * D
    Wc = {k: v.cpu() for k, v in W.items() if k.startswith("t_mlp.") or ".mod." in k}
    _, mods, modf = O.conditioning(cfg, Wc, I["temb"].cpu())
    ref_mod = torch.cat([mm.reshape(-1) for mm in mods] + [modf.reshape(-1)])
    pos = O.token_positions(s.token_grid)
    if joint:
        pos = torch.cat([torch.zeros(s.n_cond, 3, dtype=torch.int64), pos])
    ang = O.rope_angles(pos, cfg["rope_dims"], cfg["rope_theta"])
    ctx = None
    if s.cond_mode == "cross":
        ctx = O.linear(I["cond"].cpu().double(), W["cond_proj.w"].cpu(), W["cond_proj.b"].cpu())
    worst = (0.0, 0.0)
    for l in blocks:
        m.dit_debug_stop_after(l, "y1")
        step()
        x_in = m.dit_get_tap("x", (T, D), torch.float32)[row0:row0 + Tr]
        if l == blocks[0]:
            mod = m.dit_get_tap("mod", (n_req, mod_len), torch.float32)[mod_row]
            check(mod, ref_mod, torch.float32, f"{what}: modulation", rel=2e-5, maxabs=2e-4)
        m.dit_debug_stop_after(l, "fc2")
        step()
        x_out = m.dit_get_tap("x", (T, D), torch.float32)[row0:row0 + Tr]
        torch.cuda.synchronize()
        t0 = time.time()
        ref = O.block_rows(cfg, _block_weights_cpu(W, l), l, x_in.cpu(), mods[l], ang, rows, ctx=ctx)
        e = errors(x_out[rows.to(DEV)], ref)
        # the block's own contribution (x_out - x_in), where the residual does not mask the error
        xin_rows = x_in[rows.to(DEV)].double().cpu()
        d_rel, _ = errors(x_out[rows.to(DEV)].double().cpu() - xin_rows, ref - xin_rows)
        _log(test=what, block=l, rows=len(rows), rel_l2=e[0], max_abs_over_rms=e[1], branch_rel_l2=d_rel,
             branch_over_x=float((ref - xin_rows).norm() / ref.norm()), oracle_s=round(time.time() - t0, 1))
        assert e[0] <= 5e-3, f"{what}, block {l}: rel-L2 {e[0]:.3e}"
        assert d_rel < 3e-2, f"{what}, block {l}: branch-only rel-L2 {d_rel:.2e}"
        worst = (max(worst[0], e[0]), max(worst[1], e[1]))
    m.dit_debug_stop_after(-1, 0)
    return worst


def _rows(seed, name, n_total, n):
    """n distinct seeded rows of [0, n_total) incl. the first / last row and a tile boundary."""
    fixed = [r for r in (0, 127, 128, 255, 256, n_total - 1) if 0 <= r < n_total]
    picked = list(dict.fromkeys(fixed + [int(x * n_total) for x in synth.uniform01(seed, name, 4 * n).tolist()]))
    return torch.tensor(sorted(picked[:n]), dtype=torch.int64)


def test_cfg2_full_size_end_to_end(lib):
    """configs[1], the workload bench.py times: the WHOLE 8-block step against the oracle's whole step — `out`, the
    final-layer tokens, and the residual stream after every block (error accumulation across blocks, which per-block
    teacher forcing cannot see)."""
    if _host_gb() < 24:
        pytest.skip("the oracle's fp64 intermediates of a whole cfg 2 step need ~16 GB of host memory")
    s = synth.cfg2()
    W = synth.make_weights(s, device=DEV)
    I = synth.make_inputs(s, device=DEV)
    m = B.Dit(B.make_config(s), W, DEV)
    lat, temb, cond = I["latents"], I["temb"][0].contiguous(), I["cond"]
    D, L, T = s.hidden, s.n_blocks, s.n_tokens + s.n_cond
    n0 = B.dit_fallback_launches()
    out = m.dit_step(lat, temb, cond)
    tok = m.dit_get_tap("tok", (T, 64), torch.float32)[s.n_cond:]
    xs = _x_taps(m, lambda: m.dit_step(lat, temb, cond), T, D, L, "fc2")
    assert B.dit_fallback_launches() == n0
    taps = KeepTaps(["tok"] + [f"b{l}.x_mlp" for l in range(L)])
    t0 = time.time()
    ref = O.dit_step(O.cfg_from_shape(s), {k: v.cpu() for k, v in W.items()}, lat.cpu(), I["temb"].cpu(), cond.cpu(), taps=taps)
    t_or = time.time() - t0
    curve = []
    for l in range(L):
        e = check(xs[l], taps[f"b{l}.x_mlp"], torch.bfloat16, f"cfg2 end to end: x after block {l}")
        curve.append(e)
    e_tok = check(tok, taps["tok"], torch.bfloat16, "cfg2 end to end: final-layer tokens (fp32, before the bf16 rounding of out)")
    e_out = check(out, ref, torch.bfloat16, "cfg2 end to end: out")
    _log(test="cfg2 end to end (8 blocks, whole tensors)", out_rel_l2=e_out[0], out_max_abs_over_rms=e_out[1],
         tok_rel_l2=e_tok[0], tok_max_abs_over_rms=e_tok[1], x_after_block_rel_l2=[c[0] for c in curve],
         x_after_block_max_abs_over_rms=[c[1] for c in curve], oracle_s=round(t_or, 1))


def test_cfg2_shape_dual_stream_gated_end_to_end(lib):
    """The block variants bench.py times as cfg2_dual_gated, at the cfg 2 SHAPE (4096 + 256 rows, D = 3072, F = 12288) with two
    blocks: dual-stream joint blocks (one segmented tcgen05 launch per projection over the text and image segments, 17 row-tile
    pairs, 240- / 256-wide tiles) with the gated MLP — whole tensors against the oracle's whole step: `out` and the residual
    stream after each block."""
    if _host_gb() < 24:
        pytest.skip("the oracle's fp64 intermediates need ~16 GB of host memory")
    s = synth.cfg2(name="cfg2_dual_gated_2", cond_mode="joint2", n_blocks=2, extras={"mlp_gated": True})
    W = synth.make_weights(s, device=DEV)
    I = synth.make_inputs(s, device=DEV)
    m = B.Dit(B.make_config(s), W, DEV)
    lat, temb, cond = I["latents"], I["temb"][0].contiguous(), I["cond"]
    D, L, T = s.hidden, s.n_blocks, s.n_tokens + s.n_cond
    n0 = B.dit_fallback_launches()
    out = m.dit_step(lat, temb, cond)
    xs = _x_taps(m, lambda: m.dit_step(lat, temb, cond), T, D, L, "fc2")
    assert B.dit_fallback_launches() == n0
    taps = KeepTaps([f"b{l}.x_mlp" for l in range(L)])
    t0 = time.time()
    ref = O.dit_step(O.cfg_from_shape(s), {k: v.cpu() for k, v in W.items()}, lat.cpu(), I["temb"].cpu(), cond.cpu(), taps=taps)
    t_or = time.time() - t0
    curve = [check(xs[l], taps[f"b{l}.x_mlp"], torch.bfloat16, f"cfg2 dual + gated: x after block {l}") for l in range(L)]
    e_out = check(out, ref, torch.bfloat16, "cfg2 dual + gated: out")
    _log(test="cfg2 shape, dual-stream + gated MLP, 2 blocks, end to end", out_rel_l2=e_out[0], out_max_abs_over_rms=e_out[1],
         x_after_block_rel_l2=[c[0] for c in curve], oracle_s=round(t_or, 1))


def test_cfg2_full_size_blocks_teacher_forced(lib):
    s = synth.cfg2()
    W = synth.make_weights(s, device=DEV)
    I = synth.make_inputs(s, device=DEV)
    m = B.Dit(B.make_config(s), W, DEV)
    lat, temb, cond = I["latents"], I["temb"][0].contiguous(), I["cond"]
    T = s.n_tokens + s.n_cond
    rows = _rows(2, "cfg2.rows", T, 64)
    _teacher_forced_blocks(s, m, W, I, lambda: m.dit_step(lat, temb, cond), [0, 3, 7], rows,
                           "cfg2 full size, teacher forced, 64 sampled rows", T)


def _cfg3_model():
    s = synth.cfg3()
    W = synth.make_weights(s, device=DEV)
    I = synth.make_inputs(s, device=DEV)
    m = B.Dit(B.make_config(s), W, DEV)
    return s, W, I, m


def test_cfg3_full_size_every_block_teacher_forced(lib):
    """configs[2]: ALL four blocks, 64 sampled rows each (self-attention over 32760 keys with 3D RoPE, the cross-attention
    sub-layer, the MLP)."""
    if _host_gb() < 48:
        pytest.skip("the oracle's fp64 K/V of 32760 x 15360 need ~40 GB of host memory")
    s, W, I, m = _cfg3_model()
    lat, temb, cond = I["latents"], I["temb"][0].contiguous(), I["cond"]
    rows = _rows(3, "cfg3.rows", s.n_tokens, 64)
    n0 = B.dit_fallback_launches()
    _teacher_forced_blocks(s, m, W, I, lambda: m.dit_step(lat, temb, cond), list(range(s.n_blocks)), rows,
                           "cfg3 full size, teacher forced, 64 sampled rows", s.n_tokens)
    assert B.dit_fallback_launches() == n0


def test_cfg3_full_size_end_to_end_vs_stored_oracle_rows(lib):
    """configs[2] END TO END: the whole 4-block step on the GPU against sampled rows of one full oracle step
    (tests/golden/cfg3_oracle_rows.pt, written by tests/golden/make_fullsize_oracle.py from oracle/ only)."""
    path = os.path.join(os.path.dirname(__file__), "golden", "cfg3_oracle_rows.pt")
    assert os.path.exists(path), "tests/golden/cfg3_oracle_rows.pt is missing: run tests/golden/make_fullsize_oracle.py"
    g = torch.load(path)
    s, W, I, m = _cfg3_model()
    assert g["meta"]["config"] == s.name and abs(g["meta"]["t"] - I["t"]) < 1e-9
    _assert_same_generator_on_both_devices(s)
    lat, temb, cond = I["latents"], I["temb"][0].contiguous(), I["cond"]
    D, L, T = s.hidden, s.n_blocks, s.n_tokens
    out = m.dit_step(lat, temb, cond)
    tok = m.dit_get_tap("tok", (T, 64), torch.float32)
    xs = _x_taps(m, lambda: m.dit_step(lat, temb, cond), T, D, L, "fc2")
    rt, rx = g["rows_tok"].to(DEV), g["rows_x"].to(DEV)
    curve = [errors(xs[l][rx], g["x_blocks"][l]) for l in range(L)]
    e_tok = errors(tok[rt], g["tok"])
    # `out` (bf16, latent layout): its patchify is the token matrix again (memory plumbing, no arithmetic)
    out_tok = O.patchify(out.cpu().double(), s.patch)[g["rows_tok"]]
    e_out = errors(out_tok, g["tok"])
    # the max-abs bar is relative to the RMS of the WHOLE oracle output, stored with the rows
    mx = float((out_tok - g["tok"].double()).abs().max()) / g["out_rms"]
    _log(test="cfg3 end to end (4 blocks) vs stored oracle rows", rows_tok=len(g["rows_tok"]), rows_x=len(g["rows_x"]),
         out_rel_l2=e_out[0], out_max_abs_over_rms=mx, tok_rel_l2=e_tok[0], tok_max_abs_over_rms=e_tok[1],
         x_after_block_rel_l2=[c[0] for c in curve], x_after_block_max_abs_over_rms=[c[1] for c in curve],
         oracle_wall_s=g["meta"]["oracle_wall_s"])
    assert e_out[0] <= 5e-3 and mx <= 3e-2, f"cfg3 end to end: out rel-L2 {e_out[0]:.3e}, max-abs / RMS(out) {mx:.3e}"
    assert e_tok[0] <= 5e-3 and e_tok[1] <= 3e-2, f"cfg3 end to end: final-layer tokens rel-L2 {e_tok[0]:.3e} max {e_tok[1]:.3e}"
    for l in range(L):
        assert curve[l][0] <= 5e-3, f"cfg3 end to end: x after block {l}: rel-L2 {curve[l][0]:.3e}"


def _cfg4_model():
    shapes = synth.cfg4_requests()
    W = synth.make_weights(shapes[0], device=DEV)
    R = len(shapes)
    ts = [float(synth.uniform01(7, f"t{r}", 1)[0]) * 1000 for r in range(R)]
    Is = [synth.make_inputs(sh, device=DEV, tag=f".r{r}", t=ts[r]) for r, sh in enumerate(shapes)]
    T_total = sum(sh.n_tokens + sh.n_cond for sh in shapes)
    assert T_total == 37376
    cfg = B.make_config(shapes[-1], max_tokens=T_total, max_requests=R, max_cond_tokens=sum(sh.n_cond for sh in shapes))
    return shapes, W, Is, B.Dit(cfg, W, DEV), T_total


def test_cfg4_full_size_packed_batch(lib):
    """configs[3]: six requests {1024, 1024, 4096, 4096, 9216, 16384} + 256 text tokens each, packed with cu_seqlens,
    per-request timesteps (seed 7).  (i) requests 0-3 of the PACKED result against the oracle's dit_step of each request,
    whole tensors; (ii) the 16384-token request: first, middle and last block teacher-forced on sampled rows of the packed
    residual stream; (iii) packing invariance for all six: request r of the packed step == dit_step on request r alone."""
    if _host_gb() < 24:
        pytest.skip("the oracle's fp64 intermediates need ~16 GB of host memory")
    shapes, W, Is, m, T_total = _cfg4_model()
    R = len(shapes)
    lats = [i["latents"] for i in Is]
    temb = torch.cat([i["temb"] for i in Is])
    conds = [i["cond"] for i in Is]
    n0 = B.dit_fallback_launches()
    outs = m.dit_step_varlen(lats, temb, conds)
    torch.cuda.synchronize()
    Wc = {k: v.cpu() for k, v in W.items()}
    for r in range(4):
        t0 = time.time()
        ref = O.dit_step(O.cfg_from_shape(shapes[r]), Wc, lats[r].cpu(), Is[r]["temb"].cpu(), conds[r].cpu())
        e = check(outs[r], ref, torch.bfloat16, f"cfg4 packed, request {r} ({shapes[r].n_tokens} tokens) vs oracle")
        _log(test="cfg4 packed request vs oracle dit_step (8 blocks, whole tensor)", request=r, tokens=shapes[r].n_tokens,
             out_rel_l2=e[0], out_max_abs_over_rms=e[1], oracle_s=round(time.time() - t0, 1))
    cu = [0]
    for sh in shapes:
        cu.append(cu[-1] + sh.n_tokens + sh.n_cond)
    r = 5
    rows = _rows(7, "cfg4.rows", shapes[r].n_tokens + shapes[r].n_cond, 48)
    _teacher_forced_blocks(shapes[r], m, W, Is[r], lambda: m.dit_step_varlen(lats, temb, conds), [0, 4, 7], rows,
                           "cfg4 packed, 16384-token request, teacher forced, 48 sampled rows", T_total, row0=cu[r], mod_row=r,
                           n_req=R)
    for r in range(R):
        single = m.dit_step(lats[r], temb[r].contiguous(), conds[r])
        torch.cuda.synchronize()
        e_rel, e_max = errors(outs[r], single)
        assert torch.isfinite(outs[r].float()).all()
        # The packed launch (longest request: 16640 keys) runs the CTA-pair attention kernel, a short request alone the
        # two-tile kernel: both are exact re-associations with different bf16 rounding points (reference of P), so the two
        # GPU results are independent bf16 realisations of the same step — each within the oracle bar above (requests 0-3),
        # their difference within sqrt(2) of it.  Requests 4, 5 alone take the pair kernel too and agree more closely.
        assert e_rel < 5e-3 and e_max < 4.5e-2, f"packing changed request {r}: rel {e_rel:.2e} max {e_max:.2e}"
        _log(test="cfg4 packing invariance (packed vs alone, GPU vs GPU)", request=r, rel_l2=e_rel, max_abs_over_rms=e_max)
    assert B.dit_fallback_launches() == n0


CFG5_ROWS = lambda N: torch.tensor([0, 127, 128, 255, 256, 1000, N // 2 + 3, N - 129, N - 1])


@pytest.mark.parametrize("H,N", [(24, 32768), (40, 16384), (24, 65536), (40, 65536), (24, 131072), (40, 131072)])
def test_cfg5_full_size_attention_sampled_rows_and_split(lib, H, N):
    """configs[4]: q, k, v ~ N(0,1), seed 11, up to the top of the sweep.  Sampled query rows against the plain definition
    over ALL keys; split-KV P = 2 / 4 / 8 partials + LSE merge against the unsplit GPU result (P-invariance) and, on the
    sampled rows, against the oracle."""
    if N * H * 128 * 8 * 3 / 2 ** 30 > _host_gb() - 8:
        pytest.skip("the oracle's fp64 K / V do not fit in host memory")
    q, k, v = synth.make_attention_qkv(11, N, N, H, 128, device=DEV)
    n0 = B.dit_fallback_launches()
    o, lse = B.dit_attn_partial(q, k, v)
    rows = CFG5_ROWS(N)
    t0 = time.time()
    ro, rl = O.attention(q[rows.to(DEV)].cpu(), k.cpu(), v.cpu())
    t_or = time.time() - t0
    e = check(o[rows.to(DEV)], ro, torch.bfloat16, f"attention N={N} H={H} sampled rows", rel=4e-3, maxabs=2.5e-2)
    e_lse = float((lse[rows.to(DEV)].double().cpu() - rl).abs().max())
    assert e_lse < 2e-2
    rec = dict(test="cfg5 attention, sampled rows vs oracle", H=H, N=N, rel_l2=e[0], max_abs_over_rms=e[1], lse_max_abs=e_lse,
               oracle_s=round(t_or, 1))
    for P in ((2, 4, 8) if N <= 32768 else (8,)):
        n = (N + P - 1) // P
        parts = [B.dit_attn_partial(q, k[p * n:(p + 1) * n], v[p * n:(p + 1) * n]) for p in range(P)]
        om, lm = B.dit_attn_merge([x[0] for x in parts], [x[1] for x in parts])
        e_rel, e_max = errors(om, o)
        # both sides are bf16-rounded GPU results and the partials are bf16 as well (R19): the max-abs bar is
        # twice the GPU-vs-oracle one; the oracle comparison of the merged result follows on the sampled rows
        assert e_rel < 4e-3 and e_max < 6e-2, f"P={P}: rel {e_rel:.2e} max {e_max:.2e}"
        em = check(om[rows.to(DEV)], ro, torch.bfloat16, f"merged P={P} sampled rows")
        assert float((lm - lse).abs().max()) < 1e-3
        rec[f"merged_P{P}_rel_l2"] = em[0]
        del parts, om, lm
    assert B.dit_fallback_launches() == n0
    _log(**rec)


def test_cfg2_full_size_guided_step_packed_vs_two_passes(lib):
    """configs[1] shape, one guided Euler step of dit_sample: on a handle with room for both requests the step runs as
    ONE packed pass of two requests (include/dit.h), on a handle without it as two passes.  Both combine fp32 velocities
    and round x_1 once, so they agree to a bf16 rounding flip here and there — the property that holds at any size (the
    oracle checks both forms at small sizes).  A second, looser look against two plain dit_step calls, whose bf16-rounded
    velocities the guidance scale amplifies."""
    s = synth.cfg2()
    W = synth.make_weights(s, device=DEV)
    I = synth.make_inputs(s, device=DEV)
    lat, temb, cond = I["latents"], I["temb"][0].contiguous(), I["cond"]
    unc = synth.normal(s.seed, "uncond", (192, s.cond_dim), dtype=s.torch_dtype, device=DEV)   # n_uncond != n_cond
    g, sig = 3.5, [1.0, 0.75]
    m1 = B.Dit(B.make_config(s), W, DEV)
    two = m1.dit_sample(lat, temb.reshape(1, -1), sig, cond, unc, g, use_graph=False)
    v_c = m1.dit_step(lat, temb, cond).float()
    v_u = m1.dit_step(lat, temb, unc).float()
    loose = lat.float() + (sig[1] - sig[0]) * (v_u + g * (v_c - v_u))
    T2 = 2 * s.n_tokens + s.n_cond + 192
    m2 = B.Dit(B.make_config(s, max_requests=2, max_tokens=T2, max_cond_tokens=s.n_cond + 192), W, DEV)
    for use_graph in (False, True):
        got = m2.dit_sample(lat, temb.reshape(1, -1), sig, cond, unc, g, use_graph=use_graph)
        torch.cuda.synchronize()
        assert torch.isfinite(got.float()).all()
        e_rel, e_max = errors(got.float() - lat.float(), two.float() - lat.float())
        assert e_rel < 2e-3 and e_max < 3e-2, f"packed vs two passes (graph={use_graph}): rel {e_rel:.2e} max {e_max:.2e}"
        l_rel, _ = errors(got.float() - lat.float(), loose - lat.float())
        assert l_rel < 2e-2, f"packed vs two dit_step calls (graph={use_graph}): rel {l_rel:.2e}"
