"""GPU parity of dit_sample (a request's denoising trajectory: steps chained by the Euler update, optional
classifier-free guidance, optional CUDA-graph replay) against the CPU oracle's dit_sample on the same seeded inputs."""
import pytest
import torch

from oracle import dit_oracle as O
from paper_2606_13501_b200 import binding as B
from paper_2606_13501_b200 import synth
from util import check, errors

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _traj(s, n_steps, n_unc=None):
    I = synth.make_inputs(s)
    ts = [900.0 - 700.0 * i / max(1, n_steps) for i in range(n_steps)]
    tembs = synth.timestep_embedding(ts, s.temb_dim) if n_steps else torch.zeros(0, s.temb_dim)
    sigmas = [1.0 - (i / max(1, n_steps)) ** 1.5 for i in range(n_steps + 1)]
    unc = None
    if n_unc is not None and s.cond_mode != "none":
        unc = synth.normal(s.seed, "uncond", (n_unc, s.cond_dim), dtype=s.torch_dtype)
    return I, tembs, sigmas, unc


def _packed_caps(s, n_unc):
    """Handle capacities that let dit_sample run a guided step as ONE packed pass of two requests (include/dit.h)."""
    joint = s.cond_mode in ("joint", "joint2")
    return dict(max_requests=2, max_tokens=2 * s.n_tokens + (s.n_cond + n_unc if joint else 0), max_cond_tokens=s.n_cond + n_unc)


def _both(s, n_steps, n_unc=None, g=1.0, use_graph=False, split_p=1, packed=False):
    W = synth.make_weights(s)
    I, tembs, sigmas, unc = _traj(s, n_steps, n_unc)
    ref = O.dit_sample(O.cfg_from_shape(s), W, I["latents"], tembs, sigmas, I["cond"], unc, g)
    m = B.Dit(B.make_config(s, split_p=split_p, **(_packed_caps(s, n_unc) if packed else {})), W, DEV)
    dev = lambda t: None if t is None else t.to(DEV)
    args = (dev(I["latents"]), dev(tembs), sigmas, dev(I["cond"]), dev(unc), g)
    out = m.dit_sample(*args, use_graph=use_graph)
    torch.cuda.synchronize()
    return out, ref, m, args, I


def _check_traj(out, ref, I, dt, what, disp_rel):
    check(out, ref, dt, what)
    x0 = I["latents"].double()
    e_rel, _ = errors(out.double().cpu() - x0, ref - x0)      # the displacement: x_0 does not mask the velocity error
    assert e_rel <= disp_rel, f"{what}: displacement rel-L2 {e_rel:.3e} > {disp_rel:.1e}"


@pytest.mark.parametrize("use_graph", [False, True])
def test_cfg1_fp32_trajectory(lib, use_graph):
    s = synth.cfg1()
    out, ref, *_, I = _both(s, 3, use_graph=use_graph)
    _check_traj(out, ref, I, torch.float32, "cfg1 3 steps", 2e-5)


@pytest.mark.parametrize("packed", [False, True])
@pytest.mark.parametrize("mode,n_unc,use_graph", [("joint", 16, False), ("joint", 32, True), ("cross", 16, True)])
def test_fp32_guided_trajectory(lib, mode, n_unc, use_graph, packed):
    """Two passes per step: joint mode with n_uncond != n_cond changes the sequence geometry between the passes (no
    graph).  packed: the handle has room for both requests, the step is ONE varlen pass of two requests."""
    s = synth.cfg1(cond_mode=mode, rope_dims=(0, 32, 32), qk_rmsnorm=True)
    out, ref, *_, I = _both(s, 2, n_unc=n_unc, g=4.0, use_graph=use_graph or packed, split_p=2, packed=packed)
    _check_traj(out, ref, I, torch.float32, f"cfg1 guided {mode} packed={packed}", 5e-5)


@pytest.mark.parametrize("packed", [False, True])
@pytest.mark.parametrize("use_graph", [False, True])
def test_bf16_guided_trajectory(lib, use_graph, packed):
    s = synth.cfg1(name="traj_bf16", dtype="bf16", hidden=512, n_heads=4, head_dim=128, mlp_dim=2048, cond_dim=512,
                   latent_channels=16, rope_dims=(0, 64, 64), qk_rmsnorm=True, n_blocks=3)
    out, ref, *_, I = _both(s, 4, n_unc=32, g=3.0, use_graph=use_graph, packed=packed)
    _check_traj(out, ref, I, torch.bfloat16, f"bf16 guided 4 steps packed={packed}", 2e-2)


@pytest.mark.parametrize("dtype,packed,use_graph", [("bf16", False, False), ("bf16", True, True), ("f32", True, False)])
def test_dual_stream_gated_guided_trajectory(lib, dtype, packed, use_graph):
    """Dual-stream blocks with the gated MLP through dit_sample: two passes per step, or ONE packed pass of two requests that
    share a modulation row (row stride 0) while each request has its own text / image segments (segmented GEMM launches, one
    adaLN launch over the four segments); n_uncond != n_cond."""
    if dtype == "bf16":
        s = synth.cfg1(name="traj_dual", dtype="bf16", cond_mode="joint2", hidden=512, n_heads=4, head_dim=128, mlp_dim=1096,
                       cond_dim=512, latent_channels=16, rope_dims=(0, 64, 64), qk_rmsnorm=True, n_blocks=2,
                       extras={"t": 500.0, "mlp_gated": True})
        bar = 2e-2
    else:
        s = synth.cfg1(cond_mode="joint2", rope_dims=(0, 32, 32), qk_rmsnorm=True, extras={"t": 500.0, "mlp_gated": True})
        bar = 5e-5
    n0 = B.dit_fallback_launches()
    out, ref, *_, I = _both(s, 3, n_unc=20, g=3.0, use_graph=use_graph, packed=packed)
    _check_traj(out, ref, I, s.torch_dtype, f"dual-stream gated guided {dtype} packed={packed}", bar)
    if dtype == "bf16":
        assert B.dit_fallback_launches() == n0


def test_packed_guidance_needs_room_for_both_requests(lib):
    """One request short of room in max_tokens: the same call falls back to two passes per step and still matches."""
    s = synth.cfg1(cond_mode="joint", rope_dims=(0, 32, 32), qk_rmsnorm=True)
    W = synth.make_weights(s)
    I, tembs, sigmas, unc = _traj(s, 2, 16)
    ref = O.dit_sample(O.cfg_from_shape(s), W, I["latents"], tembs, sigmas, I["cond"], unc, 2.5)
    caps = _packed_caps(s, 16)
    caps["max_tokens"] -= 1
    m = B.Dit(B.make_config(s, **caps), W, DEV)
    out = m.dit_sample(I["latents"].to(DEV), tembs.to(DEV), sigmas, I["cond"].to(DEV), unc.to(DEV), 2.5, use_graph=False)
    torch.cuda.synchronize()
    _check_traj(out, ref, I, torch.float32, "guided, capacity one row short", 5e-5)


def test_graph_replay_is_bit_identical_and_recaptures_on_change(lib):
    s = synth.cfg1(name="traj_bf16", dtype="bf16", hidden=512, n_heads=4, head_dim=128, mlp_dim=2048, cond_dim=512,
                   latent_channels=16, rope_dims=(0, 64, 64), qk_rmsnorm=True)
    out_e, ref, m, args, I = _both(s, 3, n_unc=32, g=2.0, use_graph=False)
    lat, tembs, sigmas, cond, unc, g = args
    out_g = torch.empty_like(lat)
    for _ in range(3):                                   # capture, then two replays of the cached graph
        out_g.zero_()
        m.dit_sample(lat, tembs, sigmas, cond, unc, g, use_graph=True, out=out_g)
        torch.cuda.synchronize()
        assert torch.equal(out_g, out_e)
    sig2 = [x * 0.5 for x in sigmas]                     # a changed schedule must not replay the stale graph
    m.dit_sample(lat, tembs, sig2, cond, unc, g, use_graph=True, out=out_g)
    want = m.dit_sample(lat, tembs, sig2, cond, unc, g, use_graph=False)
    torch.cuda.synchronize()
    assert torch.equal(out_g, want) and not torch.equal(out_g, out_e)
    # another call with a different latent grid in between leaves its geometry (cu_seqlens, RoPE table) on the device:
    # the replay must restore its own
    small = lat[:, :, :16, :16].contiguous()
    m.dit_step(small, tembs[0], cond)
    m.dit_sample(lat, tembs, sig2, cond, unc, g, use_graph=True, out=out_g)
    torch.cuda.synchronize()
    assert torch.equal(out_g, want)
    # the plain step still works after a trajectory (geometry cache, workspace) and matches a fresh run
    v = m.dit_step(lat, tembs[0], cond)
    v2 = B.Dit(B.make_config(s), synth.make_weights(s), DEV).dit_step(lat, tembs[0], cond)
    torch.cuda.synchronize()
    assert torch.equal(v, v2)


@pytest.mark.parametrize("dtype", ["f32", "bf16"])
@pytest.mark.parametrize("mode", ["plain", "two_pass", "packed"])
def test_modulation_computed_ahead_is_bit_identical(lib, dtype, mode):
    """dit_config.max_sample_steps: the timestep MLP and the modulation GEMV of (chunks of) the trajectory's steps run ahead
    of the steps, 8 rows per pass over the weights.  11 steps with room for 1, 4 (chunks 4 4 3), 11 and 16 steps (a 9-row
    launch = an 8-row and a 1-row pass), stream launches and graph: every result equals max_sample_steps = 0 bit for bit."""
    if dtype == "f32":
        s = synth.cfg1(cond_mode="joint", rope_dims=(0, 32, 32), qk_rmsnorm=True)
    else:
        s = synth.cfg1(name="traj_bf16", dtype="bf16", hidden=512, n_heads=4, head_dim=128, mlp_dim=2048, cond_dim=512,
                       latent_channels=16, rope_dims=(0, 64, 64), qk_rmsnorm=True, cond_mode="joint2" if mode == "packed" else "joint")
    n_steps, n_unc = 11, 24
    W = synth.make_weights(s)
    I, tembs, sigmas, unc = _traj(s, n_steps, n_unc)
    caps = _packed_caps(s, n_unc) if mode == "packed" else {}
    dev = lambda t: None if t is None else t.to(DEV)
    args = (dev(I["latents"]), dev(tembs), sigmas, dev(I["cond"]), dev(unc) if mode != "plain" else None, 3.0 if mode != "plain" else 1.0)
    base = B.Dit(B.make_config(s, **caps), W, DEV).dit_sample(*args)
    torch.cuda.synchronize()
    for S in (1, 4, 11, 16):
        m = B.Dit(B.make_config(s, max_sample_steps=S, **caps), W, DEV)
        for use_graph in (False, True, True):
            out = m.dit_sample(*args, use_graph=use_graph)
            torch.cuda.synchronize()
            assert torch.equal(out, base), f"max_sample_steps={S} graph={use_graph}"
        # the single step of the same handle is untouched by the trajectory buffers
        v = m.dit_step(args[0], args[1][0], args[3])
        v0 = B.Dit(B.make_config(s, **caps), W, DEV).dit_step(args[0], args[1][0], args[3])
        torch.cuda.synchronize()
        assert torch.equal(v, v0)
    bad = B.make_config(s, max_sample_steps=5000)
    with pytest.raises(B.DitError):
        B.Dit(bad, W, DEV)


def test_packed_guided_cross_graph_with_changing_uncond_count(lib):
    """Cross-attention, packed guided step (R = 2), CUDA-graph replay: a second trajectory on the SAME handle with the
    same latents but another number of unconditional tokens changes only the cond-token offsets (cu_cond) — the resident
    geometry must be refreshed and the graph re-captured, each call matching the oracle."""
    s = synth.cfg1(cond_mode="cross", rope_dims=(0, 32, 32), qk_rmsnorm=True)
    W = synth.make_weights(s)
    m = B.Dit(B.make_config(s, max_requests=2, max_tokens=2 * s.n_tokens, max_cond_tokens=s.n_cond + 32), W, DEV)
    for n_unc in (16, 32, 8, 16):
        I, tembs, sigmas, unc = _traj(s, 2, n_unc)
        ref = O.dit_sample(O.cfg_from_shape(s), W, I["latents"], tembs, sigmas, I["cond"], unc, 3.0)
        out = m.dit_sample(I["latents"].to(DEV), tembs.to(DEV), sigmas, I["cond"].to(DEV), unc.to(DEV), 3.0, use_graph=True)
        torch.cuda.synchronize()
        _check_traj(out, ref, I, torch.float32, f"packed guided cross, n_uncond={n_unc}", 5e-5)


def test_zero_steps_and_argument_errors(lib):
    s = synth.cfg1()
    W = synth.make_weights(s)
    I, tembs, sigmas, _ = _traj(s, 0)
    m = B.Dit(B.make_config(s), W, DEV)
    lat = I["latents"].to(DEV)
    out = m.dit_sample(lat, tembs.to(DEV), sigmas, I["cond"].to(DEV))
    torch.cuda.synchronize()
    assert torch.equal(out, lat)
    I, tembs, sigmas, _ = _traj(s, 2)
    with pytest.raises(B.DitError):
        m.dit_sample(lat, tembs.to(DEV), sigmas, I["cond"].to(DEV), out=lat)          # out aliases latents


def test_one_step_equals_step_plus_update(lib):
    """dit_sample with one step against dit_step on the same handle: out = x + dsigma v up to the bf16 rounding of v."""
    s = synth.cfg1()
    W = synth.make_weights(s)
    I, tembs, sigmas, _ = _traj(s, 1)
    m = B.Dit(B.make_config(s), W, DEV)
    lat, cond, te = I["latents"].to(DEV), I["cond"].to(DEV), tembs.to(DEV)
    out = m.dit_sample(lat, te, sigmas, cond)
    v = m.dit_step(lat, te[0], cond)
    torch.cuda.synchronize()
    want = lat.double() + (sigmas[1] - sigmas[0]) * v.double()
    assert float((out.double() - want).abs().max()) <= 1e-6
