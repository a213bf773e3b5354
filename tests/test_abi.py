"""The C-ABI library loads without a GPU and exports every symbol include/dit.h declares; host-side
argument validation works without launching anything.  CPU only."""
import ctypes as C
import os
import re

import pytest

from paper_2606_13501_b200 import binding, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    names = set()
    for hdr in ("dit.h", "dit_sim.h"):
        src = open(os.path.join(ROOT, "include", hdr)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(dit_[a-z_0-9]+)\s*\(", src))
    return sorted(names)


def test_library_exports_every_declared_symbol(lib):
    names = _declared()
    assert "dit_step" in names and "dit_attn_merge" in names and len(names) >= 14
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/dit.h but not exported"
    assert sorted(binding.SYMBOLS) == names


def test_config_struct_matches_header():
    src = open(os.path.join(ROOT, "include", "dit.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} dit_config;", src, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = [re.sub(r"\[.*\]", "", f.split()[-1]) for f in body.split(";") if f.strip()]
    assert fields == [f[0] for f in binding.dit_config._fields_]


def test_workspace_bytes_and_validation_without_gpu(lib):
    for s in (synth.cfg1(), synth.cfg2(), synth.cfg3()):
        cfg = binding.make_config(s, split_p=4)
        n = lib.dit_workspace_bytes(C.byref(cfg))
        D, T = s.hidden, cfg.max_tokens
        assert n > T * D * 4 and n % 256 == 0
    bad = binding.make_config(synth.cfg1())
    bad.head_dim = 48
    assert lib.dit_workspace_bytes(C.byref(bad)) == 0
    bad = binding.make_config(synth.cfg1())
    bad.struct_size = 4
    assert lib.dit_workspace_bytes(C.byref(bad)) == 0
    bad = binding.make_config(synth.cfg2())
    bad.rope_dims = (C.c_int32 * 3)(0, 64, 32)
    assert lib.dit_workspace_bytes(C.byref(bad)) == 0
    bad = binding.make_config(synth.cfg1(), split_p=3)
    assert lib.dit_workspace_bytes(C.byref(bad)) == 0
    # dit_init rejects a NULL workspace before touching the device
    h = C.c_void_p()
    st = lib.dit_init(C.byref(binding.make_config(synth.cfg1())), None, 0, None, 0, C.byref(h))
    assert st == -3 and b"workspace" in lib.dit_last_error(None)
    # every step / trajectory entry point rejects a NULL handle before touching the device
    grid = (C.c_int32 * 3)(1, 8, 8)
    sig = (C.c_float * 2)(1.0, 0.0)
    assert lib.dit_step(None, None, None, None, 0, grid, None, None) == -1
    assert lib.dit_step_host(None, None, None, None, 0, grid, None, None) == -1
    assert lib.dit_step_varlen_host(None, None, None, None, None, None, grid, 1, None, None) == -1
    assert lib.dit_sample(None, None, None, sig, None, 0, None, 0, 1.0, grid, 1, 0, None, None) == -1
    assert b"handle" in lib.dit_last_error(None)
    assert lib.dit_kernel_launches() == 0 and lib.dit_fallback_launches() == 0
    # a bf16 config the tcgen05 kernels cannot serve is refused (no FFMA substitute inside a step), so is a row width
    # the adaLN kernel is not instantiated for
    assert lib.dit_workspace_bytes(C.byref(binding.make_config(synth.cfg1(dtype="bf16")))) == 0      # head_dim 64
    assert b"head_dim 128" in lib.dit_last_error(None)
    assert lib.dit_workspace_bytes(C.byref(binding.make_config(synth.cfg1(hidden=1792, n_heads=28)))) == 0
    assert lib.dit_workspace_bytes(C.byref(binding.make_config(synth.cfg2(latent_channels=3)))) == 0  # C*pv = 12


def test_missing_library_fails_loudly(tmp_path, monkeypatch):
    monkeypatch.setattr(binding, "_lib", None)
    with pytest.raises(binding.DitError):
        binding.load(str(tmp_path / "nope.so"))
