"""Shared helpers for the parity tests: error metrics (R17) and tolerance bars (BASELINE.json north_star)."""
import math

import torch

# north_star: bf16 paths rel-L2 <= 5e-3 and max-abs <= 3e-2 x RMS(output); fp32 path rel-L2 <= 1e-5
TOL = {torch.bfloat16: dict(rel=5e-3, maxabs=3e-2), torch.float32: dict(rel=1e-5, maxabs=1e-4)}


def errors(got: torch.Tensor, ref: torch.Tensor):
    g, r = got.detach().double().cpu().reshape(-1), ref.detach().double().cpu().reshape(-1)
    assert g.shape == r.shape, (got.shape, ref.shape)
    assert torch.isfinite(g).all(), "non-finite values in the CUDA result"
    rn = float(r.norm())
    rel = float((g - r).norm()) / (rn if rn > 0 else 1.0)
    rms = rn / math.sqrt(max(1, r.numel()))
    mx = float((g - r).abs().max()) / (rms if rms > 0 else 1.0)
    return rel, mx


def check(got, ref, dtype, what="", rel=None, maxabs=None):
    t = TOL[dtype]
    rel_bar = t["rel"] if rel is None else rel
    max_bar = t["maxabs"] if maxabs is None else maxabs
    e_rel, e_max = errors(got, ref)
    assert e_rel <= rel_bar and e_max <= max_bar, (
        f"{what}: rel-L2 {e_rel:.3e} (bar {rel_bar:.1e}), max-abs/RMS {e_max:.3e} (bar {max_bar:.1e})")
    return e_rel, e_max


def check_rounding(got, ref, what="", ulps=1.0, atol_rms=2e-3):
    """Element-wise bound for a bf16 kernel whose only error is the final rounding (plus fp32 arithmetic noise):
    |got - ref| <= ulps * 2^-8 |ref| + atol_rms * RMS(ref).  Tighter than max-abs/RMS for wide-range outputs."""
    g, r = got.detach().double().cpu().reshape(-1), ref.detach().double().cpu().reshape(-1)
    assert torch.isfinite(g).all()
    rms = float(r.norm()) / math.sqrt(max(1, r.numel()))
    bad = (g - r).abs() > ulps * 2.0 ** -8 * r.abs() + atol_rms * rms
    assert not bad.any(), f"{what}: {int(bad.sum())} elements outside the bf16 rounding bound"
