"""GPU parity, step level: dit_step / dit_step_varlen / dit_step_host against the CPU oracle on the same
seeded inputs — final output AND per-stage taps (SURVEY §8(c) sensitivity warning: end-to-end tolerances alone
would pass a wrong attention kernel), split degree P, cond modes, packing invariance."""
import pytest
import torch

from oracle import dit_oracle as O
from paper_2606_13501_b200 import binding as B
from paper_2606_13501_b200 import synth
from util import check, errors

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _gpu_inputs(s, I):
    return I["latents"].to(DEV), I["temb"][0].to(DEV), None if I["cond"] is None else I["cond"].to(DEV)


def _run_both(s, split_p=1, taps=None):
    W, I = synth.make_weights(s), synth.make_inputs(s)
    ref = O.dit_step(O.cfg_from_shape(s), W, I["latents"], I["temb"], I["cond"], split_p=1, taps=taps)
    m = B.Dit(B.make_config(s, split_p=split_p), W, DEV)
    lat, temb, cond = _gpu_inputs(s, I)
    out = m.dit_step(lat, temb, cond)
    torch.cuda.synchronize()
    return out, ref, m, (lat, temb, cond)


def _tap_checks(s, m, inputs, taps, blocks):
    """Stop the GPU step after each stage of each block and compare the workspace buffers with the oracle."""
    lat, temb, cond = inputs
    D, F, dt = s.hidden, s.mlp_dim, s.torch_dtype
    T = s.n_tokens + (s.n_cond if s.cond_mode == "joint" else 0)
    tight = dict(rel=2e-6, maxabs=5e-5) if dt == torch.float32 else {}
    for l in blocks:
        for stage, tap, shape, tdt, key in (
                ("y1", "y", (T, D), dt, f"b{l}.y1"), ("qkv", "qkv", (T, 3 * D), dt, None),
                ("attn", "o", (T, D), dt, f"b{l}.o"), ("y2", "y", (T, D), dt, f"b{l}.y2"),
                ("y2", "x", (T, D), torch.float32, f"b{l}.x_cross" if s.cond_mode == "cross" else f"b{l}.x_attn"),
                ("fc1", "u", (T, F), dt, f"b{l}.u")):
            m.dit_debug_stop_after(l, stage)
            m.dit_step(lat, temb, cond)
            got = m.dit_get_tap(tap, shape, tdt)
            torch.cuda.synchronize()
            if key is None:
                ref = torch.cat([taps[f"b{l}.q"], taps[f"b{l}.k"], taps[f"b{l}.v"]], dim=1)
            else:
                ref = taps[key]
            check(got, ref, dt, f"tap {stage}/{tap} block {l}", **tight)
    m.dit_debug_stop_after(-1, 0)


# ------------------------------------------------------------------------------ config 1 (fp32, rel-L2 1e-5)
@pytest.mark.parametrize("P", [1, 2, 4])
def test_cfg1_fp32_matches_oracle_for_every_split_degree(lib, P):
    s = synth.cfg1()
    taps = {}
    out, ref, m, inputs = _run_both(s, split_p=P, taps=taps)
    e = check(out, ref, torch.float32, f"cfg1 P={P}")
    print("cfg1 P", P, e)
    if P == 1:
        c = m.dit_get_tap("c", (s.hidden,), torch.float32)
        check(c, taps["c"], torch.float32, "c", rel=2e-6)
        mod = m.dit_get_tap("mod", (s.n_blocks * 6 * s.hidden + 2 * s.hidden,), torch.float32)
        check(mod, torch.cat([taps["mod"].reshape(-1), taps["modf"].reshape(-1)]), torch.float32, "mod", rel=2e-6)
        _tap_checks(s, m, inputs, taps, range(s.n_blocks))


@pytest.mark.parametrize("variant", ["cross", "rope_qknorm", "none_rope3d", "d128"])
def test_cfg1_variants_fp32(lib, variant):
    """R8: every code path (cross-attention, RoPE, QK-norm, no cond, head_dim 128) gets an fp32 1e-5 pin."""
    kw = {"cross": dict(cond_mode="cross", qk_rmsnorm=True),
          "rope_qknorm": dict(rope_dims=(0, 32, 32), qk_rmsnorm=True),
          "none_rope3d": dict(cond_mode="none", rope_dims=(20, 22, 22), qk_rmsnorm=True, latent_grid=(3, 16, 20),
                              patch=(1, 2, 2)),
          "d128": dict(n_heads=2, head_dim=128, rope_dims=(0, 64, 64), qk_rmsnorm=True)}[variant]
    s = synth.cfg1(**kw)
    taps = {}
    out, ref, m, inputs = _run_both(s, split_p=2 if variant == "rope_qknorm" else 1, taps=taps)
    check(out, ref, torch.float32, f"cfg1 {variant}")
    _tap_checks(s, m, inputs, taps, [s.n_blocks - 1])


def test_zero_gates_identity_and_empty_cond_on_gpu(lib):
    s = synth.cfg1()
    W, I = synth.make_weights(s), synth.make_inputs(s)
    D = s.hidden
    for l in range(s.n_blocks):
        for lo in (2 * D, 5 * D):
            W[f"blocks.{l}.mod.w"][lo:lo + D] = 0
            W[f"blocks.{l}.mod.b"][lo:lo + D] = 0
    m = B.Dit(B.make_config(s), W, DEV)
    lat, temb, cond = _gpu_inputs(s, I)
    m.dit_debug_stop_after(0, "y1")
    m.dit_step(lat, temb, cond)
    x0 = m.dit_get_tap("x", (288, D), torch.float32)
    m.dit_debug_stop_after(-1, 0)
    m.dit_step(lat, temb, cond)
    x1 = m.dit_get_tap("x", (288, D), torch.float32)
    assert torch.equal(x0, x1)                                 # zero gates: blocks are the identity, bit exact
    # joint with zero cond tokens == cond-less sequence
    s2 = synth.cfg1()
    W2, I2 = synth.make_weights(s2), synth.make_inputs(s2)
    m2 = B.Dit(B.make_config(s2), W2, DEV)
    lat, temb, _ = _gpu_inputs(s2, I2)
    out = m2.dit_step(lat, temb, None)
    ref = O.dit_step(O.cfg_from_shape(s2), W2, I2["latents"], I2["temb"], I2["cond"][:0])
    check(out, ref, torch.float32, "joint, n_cond = 0")


# ------------------------------------------------------------------------------ bf16, reduced sizes
def _small_bf16(**kw):
    d = dict(name="small_bf16", dtype="bf16", n_blocks=2, hidden=512, n_heads=4, head_dim=128, mlp_dim=2048,
             latent_channels=16, cond_dim=512, rope_dims=(0, 64, 64), qk_rmsnorm=True, latent_grid=(1, 36, 44),
             n_cond=70, extras={})
    d.update(kw)
    return synth.cfg1(**d)


@pytest.mark.parametrize("mode,P", [("joint", 1), ("joint", 4), ("cross", 1), ("none", 2)])
def test_small_bf16_step_and_taps(lib, mode, P):
    s = _small_bf16(cond_mode=mode, rope_dims=(44, 42, 42) if mode == "cross" else (0, 64, 64),
                    latent_grid=(3, 20, 24) if mode == "cross" else (1, 36, 44))
    taps = {}
    out, ref, m, inputs = _run_both(s, split_p=P, taps=taps)
    e = check(out, ref, torch.bfloat16, f"small bf16 {mode} P={P}")
    print("small bf16", mode, P, e)
    if P == 1:
        _tap_checks(s, m, inputs, taps, range(s.n_blocks))


def test_step_host_equals_device_call(lib):
    s = _small_bf16()
    W, I = synth.make_weights(s), synth.make_inputs(s)
    m = B.Dit(B.make_config(s), W, DEV)
    lat, temb, cond = _gpu_inputs(s, I)
    out = m.dit_step(lat, temb, cond)
    oh = m.dit_step_host(I["latents"].pin_memory(), I["temb"][0].contiguous().pin_memory(), I["cond"].pin_memory())
    torch.cuda.synchronize()
    assert torch.equal(oh, out.cpu())
    oh2 = m.dit_step_host(I["latents"], I["temb"][0].contiguous(), I["cond"])       # pageable host memory
    torch.cuda.synchronize()
    assert torch.equal(oh2, out.cpu())


# ------------------------------------------------------------------------------ varlen packing
@pytest.mark.parametrize("dtype,mode", [("f32", "joint"), ("bf16", "joint"), ("bf16", "cross")])
def test_varlen_equals_per_request_steps(lib, dtype, mode):
    """Packing invariance (§8(c) step 8): the packed result for request r == dit_step on request r alone, and
    both match the oracle.  Heterogeneous grids and cond lengths, per-request timesteps."""
    base = dict(cond_mode=mode, dtype=dtype, rope_dims=(0, 32, 32), qk_rmsnorm=True, seed=7)
    if dtype == "bf16":   # a bf16 step runs on the tcgen05 kernels only: head_dim 128
        base.update(hidden=512, n_heads=4, head_dim=128, mlp_dim=1024, cond_dim=512, latent_channels=16, rope_dims=(0, 64, 64))
    grids = [(1, 8, 8), (1, 32, 20), (1, 16, 48), (1, 2, 2)]
    nconds = [5, 32, 0, 17]
    ts = [float(synth.uniform01(7, f"t{r}", 1)[0]) * 1000 for r in range(4)]
    shapes = [synth.cfg1(latent_grid=g, n_cond=max(n, 1), **base) for g, n in zip(grids, nconds)]
    W = synth.make_weights(shapes[0])
    Is = [synth.make_inputs(sh, tag=f"r{r}", t=ts[r]) for r, sh in enumerate(shapes)]
    for r, n in enumerate(nconds):
        Is[r]["cond"] = Is[r]["cond"][:n]
    T_total = sum(sh.n_tokens + (n if mode == "joint" else 0) for sh, n in zip(shapes, nconds))
    cfg = B.make_config(shapes[0], max_tokens=T_total, max_requests=4, max_cond_tokens=sum(nconds))
    m = B.Dit(cfg, W, DEV)
    lats = [i["latents"].to(DEV) for i in Is]
    temb = torch.cat([i["temb"] for i in Is]).to(DEV)
    conds = [i["cond"].to(DEV) if i["cond"].shape[0] else None for i in Is]
    outs = m.dit_step_varlen(lats, temb, conds)
    torch.cuda.synchronize()
    tdt = shapes[0].torch_dtype
    for r in range(4):
        ref = O.dit_step(O.cfg_from_shape(shapes[r]), W, Is[r]["latents"], Is[r]["temb"], Is[r]["cond"])
        check(outs[r], ref, tdt, f"varlen request {r}")
        single = m.dit_step(lats[r], temb[r].contiguous(), conds[r])
        torch.cuda.synchronize()
        e_rel, _ = errors(outs[r], single)
        assert e_rel < (2e-6 if tdt == torch.float32 else 2e-3), f"packing changed request {r}: {e_rel}"


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_same_handle_cross_mode_changing_cond_counts(lib, dtype):
    """The geometry resident on the device (cu_seqlens of the cond tokens included) is keyed by EVERY field: a second
    packed cross-attention call on the same handle with the same latent grids but PERMUTED / changed cond counts
    (fixed image size, other prompt lengths — the normal serving case) must attend to its own context rows."""
    base = dict(cond_mode="cross", dtype=dtype, rope_dims=(0, 32, 32), qk_rmsnorm=True, seed=3)
    if dtype == "bf16":
        base.update(hidden=512, n_heads=4, head_dim=128, mlp_dim=1024, cond_dim=512, latent_channels=16, rope_dims=(0, 64, 64))
    grids = [(1, 16, 16), (1, 16, 16)]
    W = None
    m = None
    n0 = B.dit_fallback_launches()
    for nconds in ((5, 7), (7, 5), (20, 20), (10, 10)):
        shapes = [synth.cfg1(latent_grid=g, n_cond=n, **base) for g, n in zip(grids, nconds)]
        if W is None:
            W = synth.make_weights(shapes[0])
            cfg = B.make_config(shapes[0], max_tokens=sum(sh.n_tokens for sh in shapes), max_requests=2, max_cond_tokens=64)
            m = B.Dit(cfg, W, DEV)
        Is = [synth.make_inputs(sh, tag=f"r{r}", t=300.0 + 200 * r) for r, sh in enumerate(shapes)]
        lats = [i["latents"].to(DEV) for i in Is]
        temb = torch.cat([i["temb"] for i in Is]).to(DEV)
        conds = [i["cond"].to(DEV) for i in Is]
        outs = m.dit_step_varlen(lats, temb, conds)
        torch.cuda.synchronize()
        for r in range(2):
            ref = O.dit_step(O.cfg_from_shape(shapes[r]), W, Is[r]["latents"], Is[r]["temb"], Is[r]["cond"])
            check(outs[r], ref, shapes[0].torch_dtype, f"n_cond {nconds}, request {r}")
    assert B.dit_fallback_launches() == n0


def test_varlen_host_equals_device_call(lib):
    """dit_step_varlen_host (host buffers, copies enqueued by the library) == dit_step_varlen, bit for bit."""
    shapes = [_small_bf16(latent_grid=g, n_cond=n) for g, n in (((1, 12, 20), 9), ((1, 36, 44), 70), ((1, 4, 4), 33))]
    W = synth.make_weights(shapes[0])
    Is = [synth.make_inputs(sh, tag=f"h{r}", t=100.0 + 300 * r) for r, sh in enumerate(shapes)]
    T_total = sum(sh.n_tokens + sh.n_cond for sh in shapes)
    m = B.Dit(B.make_config(shapes[0], max_tokens=T_total, max_requests=3, max_cond_tokens=sum(sh.n_cond for sh in shapes)), W, DEV)
    n0 = B.dit_fallback_launches()
    lats = [i["latents"].to(DEV) for i in Is]
    temb = torch.cat([i["temb"] for i in Is])
    conds = [i["cond"].to(DEV) for i in Is]
    outs = m.dit_step_varlen(lats, temb.to(DEV), conds)
    packed_h = torch.cat([i["latents"].reshape(-1) for i in Is]).pin_memory()
    cond_h = torch.cat([i["cond"] for i in Is]).pin_memory()
    out_h = torch.empty_like(packed_h).pin_memory()
    m.dit_step_varlen_host(packed_h, [i["latents"].shape for i in Is], temb.contiguous().pin_memory(), cond_h,
                           [sh.n_cond for sh in shapes], out_h)
    torch.cuda.synchronize()
    assert torch.equal(out_h, torch.cat([o.reshape(-1) for o in outs]).cpu())
    assert B.dit_fallback_launches() == n0


def test_bf16_step_never_substitutes_the_ffma_kernels(lib):
    """A bf16 config the tcgen05 kernels cannot serve is refused at dit_init (DIT_ERR_UNSUPPORTED), not run ~100x slower
    on the fp32-path kernels; the kernel-level entry points do run such shapes and count them."""
    s = synth.cfg1(dtype="bf16")                                  # head_dim 64
    with pytest.raises(B.DitError, match="head_dim 128"):
        B.Dit(B.make_config(s), synth.make_weights(s), DEV)
    n0 = B.dit_fallback_launches()
    q, k, v = synth.make_attention_qkv(1, 40, 50, 2, 64, device=DEV)
    B.dit_attn_partial(q, k, v)
    A = synth.normal(1, "A", (33, 20), dtype=torch.bfloat16, device=DEV)     # K % 8 != 0
    Wt = synth.normal(1, "W", (16, 20), dtype=torch.bfloat16, device=DEV)
    B.dit_linear(A, Wt)
    torch.cuda.synchronize()
    assert B.dit_fallback_launches() == n0 + 2


# ------------------------------------------------------------------------------ dual-stream joint blocks (R37)
@pytest.mark.parametrize("dtype,P", [("f32", 1), ("f32", 2), ("bf16", 1), ("bf16", 4)])
def test_dual_stream_step_and_taps(lib, dtype, P):
    """cond_mode joint2: text and image rows have their own per-block weights, one attention over [txt ; img].  Output,
    the residual stream after every block and the attention output of the last block against the oracle."""
    if dtype == "f32":
        s = synth.cfg1(cond_mode="joint2", rope_dims=(0, 32, 32), qk_rmsnorm=True)
    else:
        s = _small_bf16(cond_mode="joint2")
    taps = {}
    out, ref, m, (lat, temb, cond) = _run_both(s, split_p=P, taps=taps)
    dt = s.torch_dtype
    check(out, ref, dt, f"dual-stream {dtype} P={P}")
    T, D = s.n_tokens + s.n_cond, s.hidden
    tight = dict(rel=2e-6, maxabs=5e-5) if dt == torch.float32 else {}
    for l in range(s.n_blocks):
        m.dit_debug_stop_after(l, "fc2")
        m.dit_step(lat, temb, cond)
        check(m.dit_get_tap("x", (T, D), torch.float32), taps[f"b{l}.x_mlp"], dt, f"dual-stream x after block {l}", **tight)
    m.dit_debug_stop_after(s.n_blocks - 1, "attn")
    m.dit_step(lat, temb, cond)
    check(m.dit_get_tap("o", (T, D), dt), taps[f"b{s.n_blocks - 1}.o"], dt, "dual-stream attention output", **tight)
    m.dit_debug_stop_after(-1, 0)


@pytest.mark.parametrize("dtype,mode,F", [("f32", "joint", 1024), ("f32", "joint2", 1000), ("bf16", "joint", 2048),
                                          ("bf16", "cross", 1992), ("bf16", "joint2", 1096)])
def test_gated_mlp_step_and_taps(lib, dtype, mode, F):
    """mlp_gated (SwiGLU, R40): u = SiLU(W1 y + b1) (.) (W3 y + b3) — on the bf16 path one tcgen05 kernel whose CTA pair
    stages W1 | W3 halves (F = 1992 / 1096: ragged last 128-column tile), on the fp32 path two GEMMs + a product.  Output,
    u of every block and the residual stream after the MLP against the oracle."""
    if dtype == "f32":
        s = synth.cfg1(cond_mode=mode, mlp_dim=F, extras={"t": 500.0, "mlp_gated": True})
    else:
        s = _small_bf16(cond_mode=mode, mlp_dim=F, extras={"mlp_gated": True})
    taps = {}
    n0 = B.dit_fallback_launches()
    out, ref, m, (lat, temb, cond) = _run_both(s, taps=taps)
    dt = s.torch_dtype
    check(out, ref, dt, f"gated MLP {dtype} {mode}")
    T, D = s.n_tokens + (s.n_cond if mode in ("joint", "joint2") else 0), s.hidden
    tight = dict(rel=2e-6, maxabs=5e-5) if dt == torch.float32 else {}
    for l in range(s.n_blocks):
        m.dit_debug_stop_after(l, "fc1")
        m.dit_step(lat, temb, cond)
        u_ref = torch.cat([taps[f"b{l}.txt.u"], taps[f"b{l}.img.u"]], 0) if mode == "joint2" else taps[f"b{l}.u"]
        u_got = m.dit_get_tap("u", (T, F), dt)
        if dt == torch.float32:
            check(u_got, u_ref, dt, f"gated MLP u block {l}", **tight)
        else:
            # u is a product of two near-Gaussian factors: heavy-tailed (max ~ 20 RMS), so the bf16 rounding of the stored
            # value alone (<= 2^-9 |u|) exceeds 3e-2 RMS at the largest elements.  rel-L2 keeps the usual bar; the
            # element-wise bar is the usual 3e-2 RMS plus a term relative to the element, 2^-7 |u| (its own rounding and
            # the input rounding of one factor scaled by a large other factor).
            e_rel, _ = errors(u_got, u_ref)
            assert e_rel <= 5e-3, f"gated MLP u block {l}: rel-L2 {e_rel:.3e}"
            diff = (u_got.double().cpu() - u_ref).abs()
            bound = u_ref.abs() * 2.0 ** -7 + 3e-2 * u_ref.pow(2).mean().sqrt()
            assert bool((diff <= bound).all()), f"gated MLP u block {l}: worst excess {float((diff - bound).max()):.3e}"
        m.dit_debug_stop_after(l, "fc2")
        m.dit_step(lat, temb, cond)
        check(m.dit_get_tap("x", (T, D), torch.float32), taps[f"b{l}.x_mlp"], dt, f"gated MLP x block {l}", **tight)
    m.dit_debug_stop_after(-1, 0)
    assert B.dit_fallback_launches() == n0
    # a handle built without w3 / b3 for a gated config is refused
    W = synth.make_weights(s)
    W.pop("blocks.0.mlp.w3")
    with pytest.raises(B.DitError):
        B.Dit(B.make_config(s), W, DEV)


def test_dual_stream_varlen_and_empty_text(lib):
    """Packed dual-stream batch: heterogeneous grids and text lengths (one request without text), per-request timesteps;
    each request against the oracle's step on that request alone."""
    grids, nconds = [(1, 12, 20), (1, 36, 44), (1, 4, 4)], [9, 70, 0]
    shapes = [_small_bf16(cond_mode="joint2", latent_grid=g, n_cond=max(n, 1)) for g, n in zip(grids, nconds)]
    W = synth.make_weights(shapes[0])
    Is = [synth.make_inputs(sh, tag=f"d{r}", t=150.0 + 250 * r) for r, sh in enumerate(shapes)]
    for r, n in enumerate(nconds):
        Is[r]["cond"] = Is[r]["cond"][:n]
    T_total = sum(sh.n_tokens + n for sh, n in zip(shapes, nconds))
    m = B.Dit(B.make_config(shapes[0], max_tokens=T_total, max_requests=3, max_cond_tokens=sum(nconds)), W, DEV)
    lats = [i["latents"].to(DEV) for i in Is]
    temb = torch.cat([i["temb"] for i in Is]).to(DEV)
    conds = [i["cond"].to(DEV) if i["cond"].shape[0] else None for i in Is]
    n0 = B.dit_fallback_launches()
    outs = m.dit_step_varlen(lats, temb, conds)
    torch.cuda.synchronize()
    for r in range(3):
        ref = O.dit_step(O.cfg_from_shape(shapes[r]), W, Is[r]["latents"], Is[r]["temb"], Is[r]["cond"])
        check(outs[r], ref, torch.bfloat16, f"dual-stream varlen request {r}")
    assert B.dit_fallback_launches() == n0


@pytest.mark.parametrize("mode", ["joint2", "joint"])
def test_sixty_four_tiny_requests_packed(lib, mode):
    """max_requests = 64 (the capacity limit): 64 tiny requests in one packed step — in dual-stream mode 128 row segments, the
    size of the segmented GEMM's table, each far smaller than a 256-row tile pair; every request against the oracle alone."""
    R = 64
    grids = [(1, 4 + 4 * (r % 3), 4 + 4 * (r % 2)) for r in range(R)]
    nconds = [1 + (r * 5) % 7 for r in range(R)]
    shapes = [_small_bf16(cond_mode=mode, latent_grid=g, n_cond=n, n_blocks=1) for g, n in zip(grids, nconds)]
    W = synth.make_weights(shapes[0])
    Is = [synth.make_inputs(sh, tag=f"t{r}", t=20.0 + 15 * r) for r, sh in enumerate(shapes)]
    T_total = sum(sh.n_tokens + n for sh, n in zip(shapes, nconds))
    m = B.Dit(B.make_config(shapes[0], max_tokens=T_total, max_requests=R, max_cond_tokens=sum(nconds)), W, DEV)
    n0 = B.dit_fallback_launches()
    outs = m.dit_step_varlen([i["latents"].to(DEV) for i in Is], torch.cat([i["temb"] for i in Is]).to(DEV),
                             [i["cond"].to(DEV) for i in Is])
    torch.cuda.synchronize()
    assert B.dit_fallback_launches() == n0
    # more than 8 requests: the modulation runs as tensor-core GEMMs on a [hi | lo] bf16 pair of SiLU(c) (dit.cu) — the fp32
    # modulation rows must still be the oracle's to ~2^-16 (the GEMV form, fp32 inputs, holds 2e-6)
    sh0 = shapes[0]
    n_img = sh0.n_blocks * 6 * sh0.hidden + 2 * sh0.hidden
    mod_len = n_img + (sh0.n_blocks * 6 * sh0.hidden if mode == "joint2" else 0)
    mod = m.dit_get_tap("mod", (R, mod_len), torch.float32)
    torch.cuda.synchronize()
    for r in (0, 9, 63):
        cfg_r = O.cfg_from_shape(shapes[r])
        c, mods, modf = O.conditioning(cfg_r, W, Is[r]["temb"])
        want = torch.cat([torch.stack(mods, 0).reshape(-1), modf.reshape(-1)])
        check(mod[r, :n_img], want, torch.float32, f"modulation rows of request {r} ({mode})", rel=2e-5, maxabs=2e-4)
        if mode == "joint2":
            want_t = torch.stack(O.conditioning_txt(cfg_r, W, c), 0).reshape(-1)
            check(mod[r, n_img:], want_t, torch.float32, f"text-stream modulation rows of request {r}", rel=2e-5, maxabs=2e-4)
    for r in (0, 1, 2, 17, 40, 63):
        ref = O.dit_step(O.cfg_from_shape(shapes[r]), W, Is[r]["latents"], Is[r]["temb"], Is[r]["cond"])
        check(outs[r], ref, torch.bfloat16, f"64 packed requests ({mode}), request {r}")


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
def test_step_graph_replay_is_bit_identical(lib, dtype):
    """dit_step_graph: one cudaGraphLaunch per step.  Bit-identical to dit_step; a replay sees NEW buffer contents (the graph
    holds pointers, not values); other pointers / geometry capture another graph; more than 8 argument sets evict the least
    recently used graph and everything still matches."""
    s = synth.cfg1(cond_mode="joint", rope_dims=(0, 32, 32), qk_rmsnorm=True) if dtype == "f32" else _small_bf16(cond_mode="joint")
    W, I = synth.make_weights(s), synth.make_inputs(s)
    m = B.Dit(B.make_config(s), W, DEV)
    lat, temb, cond = _gpu_inputs(s, I)
    ref = m.dit_step(lat, temb, cond).clone()
    out = torch.empty_like(lat)
    n0 = B.dit_kernel_launches()
    m.dit_step_graph(lat, temb, cond, out)                      # capture + launch
    torch.cuda.synchronize()
    assert torch.equal(out, ref)
    out.zero_()
    m.dit_step_graph(lat, temb, cond, out)                      # replay
    torch.cuda.synchronize()
    assert torch.equal(out, ref)
    # new contents in the same buffers
    I2 = synth.make_inputs(s, tag="other", t=123.0)
    lat.copy_(I2["latents"].to(DEV)); temb.copy_(I2["temb"][0].to(DEV)); cond.copy_(I2["cond"].to(DEV))
    ref2 = m.dit_step(lat, temb, cond).clone()
    m.dit_step_graph(lat, temb, cond, out)
    torch.cuda.synchronize()
    assert torch.equal(out, ref2) and not torch.equal(ref2, ref)
    # other geometry (fewer cond tokens) and ten different output buffers: captures, evictions, replays
    refc = m.dit_step(lat, temb, cond[:7]).clone()
    outs = [torch.empty_like(lat) for _ in range(10)]
    for rep in range(2):
        for o in outs:
            o.zero_()
            m.dit_step_graph(lat, temb, cond[:7], o)
        torch.cuda.synchronize()
        assert all(torch.equal(o, refc) for o in outs)
    m.dit_step_graph(lat, temb, cond, out)
    torch.cuda.synchronize()
    assert torch.equal(out, ref2)
    # a debug stop bypasses the graph
    m.dit_debug_stop_after(0, "y1")
    m.dit_step_graph(lat, temb, cond, out)
    m.dit_debug_stop_after(-1, 0)
    m.dit_step_graph(lat, temb, cond, out)
    torch.cuda.synchronize()
    assert torch.equal(out, ref2)


def test_step_varlen_graph_matches_varlen(lib):
    grids, nconds = [(1, 12, 20), (1, 36, 44), (1, 4, 4)], [9, 70, 3]
    shapes = [_small_bf16(cond_mode="joint", latent_grid=g, n_cond=n) for g, n in zip(grids, nconds)]
    W = synth.make_weights(shapes[0])
    Is = [synth.make_inputs(sh, tag=f"g{r}", t=150.0 + 250 * r) for r, sh in enumerate(shapes)]
    T_total = sum(sh.n_tokens + n for sh, n in zip(shapes, nconds))
    m = B.Dit(B.make_config(shapes[0], max_tokens=T_total, max_requests=3, max_cond_tokens=sum(nconds)), W, DEV)
    lats = [i["latents"].to(DEV) for i in Is]
    temb = torch.cat([i["temb"] for i in Is]).to(DEV)
    conds = [i["cond"].to(DEV) for i in Is]
    want = torch.cat([o.reshape(-1) for o in m.dit_step_varlen(lats, temb, conds)])
    packed, cond = torch.cat([l.reshape(-1) for l in lats]), torch.cat(conds)
    out = torch.empty_like(packed)
    for _ in range(3):
        out.zero_()
        m.dit_step_varlen_graph(packed, [tuple(l.shape) for l in lats], temb, cond, nconds, out)
        torch.cuda.synchronize()
        assert torch.equal(out, want)


def test_argument_validation_on_gpu(lib):
    s = synth.cfg1()
    W, I = synth.make_weights(s), synth.make_inputs(s)
    m = B.Dit(B.make_config(s), W, DEV)
    lat, temb, cond = _gpu_inputs(s, I)
    n0 = B.dit_kernel_launches()
    with pytest.raises(B.DitError):                             # too many tokens for the workspace
        m.dit_step(torch.zeros(4, 1, 64, 64, device=DEV), temb, cond)
    with pytest.raises(B.DitError):                             # grid not a multiple of the patch
        m.dit_step(torch.zeros(4, 1, 31, 32, device=DEV), temb, cond)
    assert B.dit_kernel_launches() == n0                        # rejected before any launch
    Wbad = dict(W); Wbad.pop("final.b")
    with pytest.raises(B.DitError):
        B.Dit(B.make_config(s), Wbad, DEV)
    m.dit_step(lat, temb, cond)
    assert B.dit_kernel_launches() > n0


_PACKED_ENDS = r'''
import sys, torch
from paper_2606_13501_b200 import binding as B, synth
B.load()
dev = torch.device("cuda", 0)
res = {}
for mode, dtype in (("joint", "bf16"), ("cross", "bf16"), ("joint2", "bf16"), ("joint", "f32"), ("none", "f32")):
    if dtype == "bf16":
        s = synth.cfg1(name="x", dtype="bf16", hidden=512, n_heads=4, head_dim=128, mlp_dim=2048, cond_dim=512, latent_channels=16,
                       rope_dims=(0, 64, 64), qk_rmsnorm=True, cond_mode=mode)
    else:
        s = synth.cfg1(cond_mode=mode, rope_dims=(0, 32, 32), qk_rmsnorm=True)
    W = synth.make_weights(s, device=dev)
    grids = [(1, 32, 32), (1, 16, 48), (1, 8, 8), (1, 64, 32), (1, 2, 2)]
    ncs = [0 if mode == "none" else n for n in (32, 7, 0, 19, 32)]
    R = len(grids)
    T = sum((g[1] // 2) * (g[2] // 2) + (nc if mode in ("joint", "joint2") else 0) for g, nc in zip(grids, ncs))
    m = B.Dit(B.make_config(s, max_requests=R, max_tokens=T, max_cond_tokens=max(1, sum(ncs))), W, dev)
    lats = [synth.normal(5, f"l{r}", (s.latent_channels,) + g, dtype=s.torch_dtype, device=dev) for r, g in enumerate(grids)]
    conds = None if mode == "none" else [synth.normal(5, f"c{r}", (nc, s.cond_dim), dtype=s.torch_dtype, device=dev) if nc else None
                                         for r, nc in enumerate(ncs)]
    temb = synth.timestep_embedding([100.0 * (r + 1) for r in range(R)], s.temb_dim, device=dev).contiguous()
    n0 = B.dit_kernel_launches()
    outs = m.dit_step_varlen(lats, temb, conds)
    torch.cuda.synchronize()
    res[f"{mode}-{dtype}"] = ([o.cpu() for o in outs], B.dit_kernel_launches() - n0)
torch.save(res, sys.argv[1])
'''


def test_packed_step_ends_launched_once_are_bit_identical_to_per_request_launches(lib, tmp_path):
    """A packed step launches patchify, the patch-embed GEMM, the final GEMM and unpatchify ONCE for all requests;
    DIT_VARLEN_PER_REQUEST=1 (read once per process, hence the two subprocesses) launches them per request.  Five requests of
    unequal grids and cond counts (one without cond tokens, one of a single token), every cond mode: same bits, 4 (R - 1) = 16
    launches fewer (18 in the joint modes)."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    got = {}
    for knob in ("0", "1"):
        path = tmp_path / f"ends{knob}.pt"
        env = dict(os.environ, DIT_VARLEN_PER_REQUEST=knob, PYTHONPATH=root + os.pathsep + os.environ.get("PYTHONPATH", ""))
        r = subprocess.run([sys.executable, "-c", _PACKED_ENDS, str(path)], env=env, capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr[-2000:]
        got[knob] = torch.load(path)
    for key, (outs, n_launch) in got["0"].items():
        ref, n_ref = got["1"][key]
        assert all(torch.isfinite(o.float()).all() for o in outs)
        assert all(torch.equal(a, b) for a, b in zip(outs, ref)), key
        # joint modes: the four per-request cond projections become one GEMM + one row scatter as well
        assert n_ref - n_launch == (18 if key.startswith("joint") else 16), (key, n_launch, n_ref)
