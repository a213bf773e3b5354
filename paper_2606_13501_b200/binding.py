"""Thin ctypes binding over libdit_b200.so (include/dit.h).  Argument marshalling only: every step of the
path runs in the library's CUDA kernels; torch is used for device memory and streams.  Same names as the C
ABI.  `load()` raises if the library is missing — there is no fallback of any kind."""
from __future__ import annotations

import ctypes as C
import os

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libdit_b200.so")

DIT_OK = 0
DIT_F32, DIT_BF16 = 0, 1
COND = {"none": 0, "joint": 1, "cross": 2, "joint2": 3}
EPI_BIAS, EPI_BIAS_GELU, EPI_BIAS_F32 = 0, 1, 2
TAP = dict(x=0, y=1, qkv=2, o=3, u=5, c=6, mod=7, tok=8)
STAGE = dict(y1=0, qkv=1, attn=2, oproj=3, cross=4, y2=5, fc1=6, fc2=7)

SYMBOLS = ["dit_workspace_bytes", "dit_init", "dit_step", "dit_step_host", "dit_step_varlen", "dit_step_varlen_host", "dit_step_graph", "dit_step_varlen_graph", "dit_sample", "dit_attn_partial",
           "dit_attn_merge", "dit_static_scratch_bytes", "dit_attn_split_static", "dit_relayout_plan", "dit_relayout", "dit_linear", "dit_linear_swiglu", "dit_quantize_fp8", "dit_linear_fp8", "dit_quantize_mxfp8", "dit_linear_mxfp8", "dit_linear_residual", "dit_linear_qkv", "dit_adaln", "dit_gemv", "dit_qknorm_rope", "dit_debug_stop_after",
           "dit_get_tap", "dit_profile_begin", "dit_profile_end", "dit_last_error", "dit_kernel_launches", "dit_fallback_launches", "dit_sim_run",
           "dit_free"]


class dit_config(C.Structure):
    _fields_ = [("struct_size", C.c_int32), ("dtype", C.c_int32), ("n_blocks", C.c_int32), ("hidden", C.c_int32),
                ("n_heads", C.c_int32), ("head_dim", C.c_int32), ("mlp_dim", C.c_int32), ("latent_channels", C.c_int32),
                ("patch", C.c_int32 * 3), ("temb_dim", C.c_int32), ("cond_dim", C.c_int32), ("cond_mode", C.c_int32),
                ("rope_dims", C.c_int32 * 3), ("rope_theta", C.c_float), ("ln_eps", C.c_float), ("rms_eps", C.c_float),
                ("qk_rmsnorm", C.c_int32), ("split_p", C.c_int32), ("max_tokens", C.c_int32),
                ("max_requests", C.c_int32), ("max_cond_tokens", C.c_int32), ("mlp_gated", C.c_int32),
                ("max_sample_steps", C.c_int32)]


class dit_weight(C.Structure):
    _fields_ = [("name", C.c_char_p), ("dev_ptr", C.c_void_p), ("numel", C.c_int64)]


class dit_transfer(C.Structure):
    _fields_ = [("src_rank", C.c_int32), ("dst_rank", C.c_int32), ("src_row", C.c_int64), ("dst_row", C.c_int64),
                ("n_rows", C.c_int64)]


class dit_cost_entry(C.Structure):
    _fields_ = [("shape_class", C.c_int32), ("degree", C.c_int32), ("step_s", C.c_double)]


class dit_sim_request(C.Structure):
    _fields_ = [("shape_class", C.c_int32), ("n_steps", C.c_int32), ("arrival_s", C.c_double), ("deadline_s", C.c_double)]


class dit_sim_config(C.Structure):
    _fields_ = [("struct_size", C.c_int32), ("policy", C.c_int32), ("n_ranks", C.c_int32), ("fcfs_group", C.c_int32),
                ("n_classes", C.c_int32), ("state_mb", C.c_double * 16), ("relayout_gbps", C.c_double), ("timeout_s", C.c_double)]


class dit_sim_result(C.Structure):
    _fields_ = [("finish_s", C.c_double), ("busy_rank_s", C.c_double), ("n_migrations", C.c_int32), ("max_degree", C.c_int32),
                ("met_deadline", C.c_int32), ("failed", C.c_int32)]


class dit_sim_summary(C.Structure):
    _fields_ = [("makespan_s", C.c_double), ("throughput_rps", C.c_double), ("mean_latency_s", C.c_double),
                ("p95_latency_s", C.c_double), ("slo_attainment", C.c_double), ("utilisation", C.c_double), ("n_events", C.c_int64)]


POLICY = {"fcfs": 0, "srtf": 1, "edf": 2}


class DitError(RuntimeError):
    pass


_lib = None


def load(path: str = LIB_PATH):
    """dlopen the C-ABI library.  Raises (never falls back) when it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise DitError(f"{path} not found: build it with `python -m paper_2606_13501_b200.build` "
                       "(there is no CPU / PyTorch fallback)")
    lib = C.CDLL(path)
    lib.dit_workspace_bytes.restype = C.c_size_t
    lib.dit_workspace_bytes.argtypes = [C.POINTER(dit_config)]
    lib.dit_last_error.restype = C.c_char_p
    lib.dit_last_error.argtypes = [C.c_void_p]
    lib.dit_kernel_launches.restype = C.c_int32
    lib.dit_fallback_launches.restype = C.c_int32
    lib.dit_relayout_plan.restype = C.c_int32
    lib.dit_static_scratch_bytes.restype = C.c_size_t
    lib.dit_static_scratch_bytes.argtypes = []
    lib.dit_free.restype = None
    lib.dit_free.argtypes = [C.c_void_p]
    vp, i32, i64, f32 = C.c_void_p, C.c_int32, C.c_int64, C.c_float
    pi32 = C.POINTER(C.c_int32)
    sig = {
        "dit_init": [C.POINTER(dit_config), C.POINTER(dit_weight), i32, vp, C.c_size_t, C.POINTER(vp)],
        "dit_step": [vp, vp, vp, vp, i32, pi32, vp, vp],
        "dit_step_host": [vp, vp, vp, vp, i32, pi32, vp, vp],
        "dit_step_graph": [vp, vp, vp, vp, i32, pi32, vp, vp],
        "dit_step_varlen_graph": [vp, vp, vp, vp, pi32, pi32, pi32, i32, vp, vp],
        "dit_step_varlen": [vp, vp, vp, vp, pi32, pi32, pi32, i32, vp, vp],
        "dit_step_varlen_host": [vp, vp, vp, vp, pi32, pi32, pi32, i32, vp, vp],
        "dit_sample": [vp, vp, vp, C.POINTER(C.c_float), vp, i32, vp, i32, f32, pi32, i32, i32, vp, vp],
        "dit_attn_partial": [i32, vp, vp, vp, i32, i32, i32, i32, i64, i64, f32, vp, vp, vp],
        "dit_attn_merge": [i32, C.POINTER(vp), C.POINTER(vp), i32, i32, i32, i32, vp, vp, vp],
        "dit_attn_split_static": [i32, vp, vp, vp, i32, i32, i32, i32, i64, i64, f32, i32, vp, vp, vp],
        "dit_relayout_plan": [i64, i32, i32, C.POINTER(dit_transfer), i32],
        "dit_relayout": [C.POINTER(dit_transfer), i32, C.POINTER(vp), C.POINTER(vp), i64, vp],
        "dit_linear": [i32, i32, vp, i64, vp, vp, vp, i64, i32, i32, i32, vp],
        "dit_linear_swiglu": [i32, vp, i64, vp, vp, vp, vp, vp, i64, vp, i32, i32, i32, vp],
        "dit_quantize_fp8": [i32, vp, i64, i32, i32, vp, i64, vp, vp],
        "dit_linear_fp8": [i32, vp, i64, vp, vp, vp, vp, vp, i64, i32, i32, i32, vp],
        "dit_quantize_mxfp8": [i32, vp, i64, i32, i32, vp, i64, vp, vp],
        "dit_linear_mxfp8": [i32, vp, i64, vp, vp, vp, vp, vp, i64, i32, i32, i32, vp],
        "dit_linear_residual": [i32, vp, i64, vp, vp, vp, i64, vp, i64, vp, i32, i32, i32, i32, vp],
        "dit_linear_qkv": [i32, vp, i64, vp, vp, vp, i64, vp, vp, f32, vp, vp, i32, i32, i32, vp],
        "dit_adaln": [i32, vp, vp, vp, vp, vp, i64, vp, i32, vp, i32, i32, f32, vp],
        "dit_gemv": [i32, vp, vp, vp, vp, i32, i32, i32, i32, vp],
        "dit_qknorm_rope": [i32, vp, i64, i32, i32, i32, i32, vp, vp, f32, vp, vp, vp],
        "dit_debug_stop_after": [vp, i32, i32],
        "dit_get_tap": [vp, i32, vp, C.c_size_t, vp],
        "dit_profile_begin": [i32],
        "dit_profile_end": [C.POINTER(C.c_float), pi32],
        "dit_sim_run": [C.POINTER(dit_sim_config), C.POINTER(dit_cost_entry), i32, C.POINTER(dit_sim_request), i32,
                        C.POINTER(dit_sim_result), C.POINTER(dit_sim_summary)],
    }
    for name, argtypes in sig.items():
        fn = getattr(lib, name)
        fn.restype = C.c_int32
        fn.argtypes = argtypes
    _lib = lib
    return lib


def _check(status: int, what: str):
    if status != DIT_OK:
        msg = load().dit_last_error(None)
        raise DitError(f"{what} failed with status {status}: {msg.decode() if msg else ''}")


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def _dt(t: torch.Tensor) -> int:
    if t.dtype == torch.float32:
        return DIT_F32
    if t.dtype == torch.bfloat16:
        return DIT_BF16
    raise DitError(f"unsupported dtype {t.dtype}")


def _i32arr(vals):
    vals = [int(v) for v in vals]
    return (C.c_int32 * len(vals))(*vals)


def make_config(shape, split_p=1, max_tokens=None, max_requests=1, max_cond_tokens=None, max_sample_steps=0) -> dit_config:
    """dit_config from a synth.DiTShape-like object (duck typed)."""
    c = dit_config()
    c.struct_size = C.sizeof(dit_config)
    c.dtype = DIT_F32 if shape.dtype == "f32" else DIT_BF16
    c.n_blocks, c.hidden, c.n_heads, c.head_dim, c.mlp_dim = shape.n_blocks, shape.hidden, shape.n_heads, shape.head_dim, shape.mlp_dim
    c.latent_channels = shape.latent_channels
    c.patch = (C.c_int32 * 3)(*shape.patch)
    c.temb_dim, c.cond_dim, c.cond_mode = shape.temb_dim, shape.cond_dim, COND[shape.cond_mode]
    c.rope_dims = (C.c_int32 * 3)(*shape.rope_dims)
    c.rope_theta, c.ln_eps, c.rms_eps = shape.rope_theta, shape.ln_eps, shape.rms_eps
    c.qk_rmsnorm, c.split_p = int(shape.qk_rmsnorm), split_p
    n = shape.n_tokens + (shape.n_cond if shape.cond_mode in ("joint", "joint2") else 0)
    c.max_tokens = int(max_tokens if max_tokens is not None else n)
    c.max_requests = max_requests
    c.max_cond_tokens = int(max_cond_tokens if max_cond_tokens is not None else (shape.n_cond if shape.cond_mode != "none" else 0))
    c.mlp_gated = int(bool(shape.extras.get("mlp_gated", False)))
    c.max_sample_steps = int(max_sample_steps)
    return c


class Dit:
    """Owns a dit_handle plus the torch allocations (workspace, weights) that must outlive it."""

    def __init__(self, cfg: dit_config, weights: dict, device="cuda:0"):
        self.lib = load()
        self.cfg = cfg
        self.device = torch.device(device)
        self.tdtype = torch.float32 if cfg.dtype == DIT_F32 else torch.bfloat16
        nbytes = self.lib.dit_workspace_bytes(C.byref(cfg))
        if nbytes == 0:
            _check(-1, "dit_workspace_bytes")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.weights = {k: v.to(self.device, self.tdtype).contiguous() for k, v in weights.items()}
        arr = (dit_weight * len(self.weights))()
        for i, (k, v) in enumerate(self.weights.items()):
            arr[i].name, arr[i].dev_ptr, arr[i].numel = k.encode(), v.data_ptr(), v.numel()
        h = C.c_void_p()
        _check(self.lib.dit_init(C.byref(cfg), arr, len(self.weights), _ptr(self.workspace), nbytes, C.byref(h)), "dit_init")
        self.handle = h

    def __del__(self):
        if getattr(self, "handle", None):
            self.lib.dit_free(self.handle)
            self.handle = None

    def dit_step(self, latents, temb, cond=None, out=None, stream=None):
        """latents [C,F,H,W] (device, config dtype), temb [temb_dim] fp32, cond [n_cond, cond_dim]."""
        out = torch.empty_like(latents) if out is None else out
        grid = _i32arr(latents.shape[1:])
        n_cond = 0 if cond is None else cond.shape[0]
        _check(self.lib.dit_step(self.handle, _ptr(latents), _ptr(temb), _ptr(cond), n_cond, grid, _ptr(out),
                                 _stream(stream)), "dit_step")
        return out

    def dit_step_graph(self, latents, temb, cond=None, out=None, stream=None):
        """dit_step replayed from a CUDA graph cached in the handle (key: the pointers and the geometry)."""
        out = torch.empty_like(latents) if out is None else out
        grid = _i32arr(latents.shape[1:])
        n_cond = 0 if cond is None else cond.shape[0]
        _check(self.lib.dit_step_graph(self.handle, _ptr(latents), _ptr(temb), _ptr(cond), n_cond, grid, _ptr(out),
                                       _stream(stream)), "dit_step_graph")
        return out

    def dit_step_varlen_graph(self, packed, shapes, temb, cond, n_cond, out, stream=None):
        """Packed step replayed from a CUDA graph: packed = the R latents back to back (1-D, device), shapes their
        [C,F_r,H_r,W_r] shapes, temb [R, temb_dim], cond [sum n_cond, cond_dim] or None, out like packed."""
        cu, grids = self._varlen_geom(shapes, n_cond)
        _check(self.lib.dit_step_varlen_graph(self.handle, _ptr(packed), _ptr(temb), _ptr(cond), _i32arr(cu), _i32arr(n_cond),
                                              _i32arr(grids), len(shapes), _ptr(out), _stream(stream)), "dit_step_varlen_graph")
        return out

    def dit_sample(self, latents, tembs, sigmas, cond=None, uncond=None, guidance_scale=1.0, use_graph=False, out=None,
                   stream=None):
        """n_steps = tembs.shape[0] denoising steps chained by the Euler update; tembs [n_steps, temb_dim] fp32 (device),
        sigmas: n_steps + 1 host floats; uncond given = classifier-free guidance (one packed pass of two requests per step when
        the handle has room for both — make_config(max_requests=2, max_tokens=2T, max_cond_tokens=n_cond + n_uncond) — else
        two passes per step)."""
        out = torch.empty_like(latents) if out is None else out
        n_steps = int(tembs.shape[0])
        assert len(sigmas) == n_steps + 1
        sig = (C.c_float * (n_steps + 1))(*[float(x) for x in sigmas])
        grid = _i32arr(latents.shape[1:])
        n_cond = 0 if cond is None else cond.shape[0]
        n_unc = 0 if uncond is None else uncond.shape[0]
        _check(self.lib.dit_sample(self.handle, _ptr(latents), _ptr(tembs), sig, _ptr(cond), n_cond, _ptr(uncond), n_unc,
                                   float(guidance_scale), grid, n_steps, int(bool(use_graph)), _ptr(out), _stream(stream)),
               "dit_sample")
        return out

    def dit_step_host(self, latents_host, temb_host, cond_host=None, out_host=None, stream=None):
        out_host = torch.empty_like(latents_host) if out_host is None else out_host
        grid = _i32arr(latents_host.shape[1:])
        n_cond = 0 if cond_host is None else cond_host.shape[0]
        _check(self.lib.dit_step_host(self.handle, _ptr(latents_host), _ptr(temb_host), _ptr(cond_host), n_cond, grid,
                                      _ptr(out_host), _stream(stream)), "dit_step_host")
        return out_host

    def _varlen_geom(self, shapes, n_cond):
        joint = self.cfg.cond_mode in (COND["joint"], COND["joint2"])
        p = self.cfg.patch
        cu, grids = [0], []
        for r, shp in enumerate(shapes):
            f, h, w = shp[1:]
            grids += [f, h, w]
            cu.append(cu[-1] + (f // p[0]) * (h // p[1]) * (w // p[2]) + (n_cond[r] if joint else 0))
        return cu, grids

    def dit_step_varlen(self, latents_list, temb, cond_list=None, stream=None):
        """latents_list: R tensors [C,F_r,H_r,W_r]; temb [R, temb_dim]; cond_list: R tensors or None.
        Packs (torch.cat: memory plumbing only), calls the C ABI once, returns the R outputs (views)."""
        R = len(latents_list)
        packed = torch.cat([l.reshape(-1) for l in latents_list])
        n_cond = [0 if (cond_list is None or cond_list[r] is None) else cond_list[r].shape[0] for r in range(R)]
        cond = torch.cat([c for c in cond_list if c is not None]) if cond_list is not None and sum(n_cond) else None
        cu, grids = self._varlen_geom([l.shape for l in latents_list], n_cond)
        out = torch.empty_like(packed)
        _check(self.lib.dit_step_varlen(self.handle, _ptr(packed), _ptr(temb), _ptr(cond), _i32arr(cu), _i32arr(n_cond),
                                        _i32arr(grids), R, _ptr(out), _stream(stream)), "dit_step_varlen")
        outs, off = [], 0
        for l in latents_list:
            outs.append(out[off:off + l.numel()].reshape(l.shape))
            off += l.numel()
        return outs

    def dit_step_varlen_host(self, packed_host, shapes, temb_host, cond_host, n_cond, out_host, stream=None):
        """HOST buffers, already packed by the caller: packed_host = the R latents back to back (1-D), shapes = their
        [C,F_r,H_r,W_r] shapes, temb_host [R, temb_dim] fp32, cond_host [sum n_cond, cond_dim] or None, out_host like
        packed_host.  One C-ABI call: H2D copies, the packed step and the D2H copy are enqueued by the library."""
        cu, grids = self._varlen_geom(shapes, n_cond)
        _check(self.lib.dit_step_varlen_host(self.handle, _ptr(packed_host), _ptr(temb_host), _ptr(cond_host), _i32arr(cu),
                                             _i32arr(n_cond), _i32arr(grids), len(shapes), _ptr(out_host), _stream(stream)),
               "dit_step_varlen_host")
        return out_host

    def dit_debug_stop_after(self, block, stage):
        _check(self.lib.dit_debug_stop_after(self.handle, block, STAGE[stage] if isinstance(stage, str) else stage),
               "dit_debug_stop_after")

    def dit_get_tap(self, tap, shape, dtype, stream=None):
        dst = torch.empty(shape, dtype=dtype, device=self.device)
        _check(self.lib.dit_get_tap(self.handle, TAP[tap], _ptr(dst), dst.numel() * dst.element_size(), _stream(stream)),
               "dit_get_tap")
        return dst


# ---- handle-less entry points -------------------------------------------------------------------
def dit_attn_partial(q, k, v, softmax_scale=None, want_lse=True, stream=None):
    """q [Nq,H,d], k/v [Nk,H,d] (last two dims contiguous; row stride free) -> o [Nq,H,d], lse [Nq,H] fp32."""
    lib = load()
    nq, H, d = q.shape
    nk = k.shape[0]
    assert q.stride(2) == 1 and q.stride(1) == d and k.stride(2) == 1 and k.stride(1) == d and v.stride(1) == d
    assert nk == 0 or k.stride(0) == v.stride(0)
    o = torch.empty((nq, H, d), dtype=q.dtype, device=q.device)
    lse = torch.empty((nq, H), dtype=torch.float32, device=q.device) if want_lse else None
    scale = d ** -0.5 if softmax_scale is None else softmax_scale
    _check(lib.dit_attn_partial(_dt(q), _ptr(q), _ptr(k), _ptr(v), nq, nk, H, d, q.stride(0) if nq else H * d,
                                k.stride(0) if nk else H * d, scale, _ptr(o), _ptr(lse), _stream(stream)),
           "dit_attn_partial")
    return o, lse


def dit_static_scratch_bytes() -> int:
    return int(load().dit_static_scratch_bytes())


def dit_attn_split_static(q, k, v, split_p, o, lse=None, softmax_scale=None, stream=None):
    """Split-KV attention + merge with the partials in the library's static device array: allocates nothing (the caller
    passes the outputs o [Nq,H,d] and, optionally, lse [Nq,H] fp32)."""
    lib = load()
    nq, H, d = q.shape
    nk = k.shape[0]
    scale = d ** -0.5 if softmax_scale is None else softmax_scale
    _check(lib.dit_attn_split_static(_dt(q), _ptr(q), _ptr(k), _ptr(v), nq, nk, H, d, q.stride(0) if nq else H * d,
                                     k.stride(0) if nk else H * d, scale, split_p, _ptr(o), _ptr(lse), _stream(stream)),
           "dit_attn_split_static")
    return o, lse


def dit_attn_merge(o_parts, lse_parts, want_lse=True, stream=None):
    lib = load()
    P = len(o_parts)
    nq, H, d = o_parts[0].shape
    o = torch.empty_like(o_parts[0])
    lse = torch.empty((nq, H), dtype=torch.float32, device=o.device) if want_lse else None
    op = (C.c_void_p * P)(*[t.data_ptr() for t in o_parts])
    lp = (C.c_void_p * P)(*[t.data_ptr() for t in lse_parts])
    _check(lib.dit_attn_merge(_dt(o), op, lp, P, nq, H, d, _ptr(o), _ptr(lse), _stream(stream)), "dit_attn_merge")
    return o, lse


def dit_relayout_plan(n_rows: int, p_src: int, p_dst: int):
    """The transfer entries of a P -> P' re-layout of an n_rows-row artifact: list of (src_rank, dst_rank, src_row, dst_row,
    n_rows) tuples (host only, no GPU needed)."""
    lib = load()
    arr = (dit_transfer * 64)()
    n = lib.dit_relayout_plan(n_rows, p_src, p_dst, arr, 64)
    if n < 0:
        _check(n, "dit_relayout_plan")
    return [(arr[i].src_rank, arr[i].dst_rank, arr[i].src_row, arr[i].dst_row, arr[i].n_rows) for i in range(n)]


def dit_relayout(src_shards, p_dst: int, stream=None):
    """src_shards: P tensors [rows_p, ...] (the R20 shards of one artifact) -> the P' destination shards (new tensors)."""
    lib = load()
    n_rows = sum(int(t.shape[0]) for t in src_shards)
    P = len(src_shards)
    ref = src_shards[0]
    row_shape = tuple(ref.shape[1:])
    row_bytes = ref.element_size()
    for d in row_shape:
        row_bytes *= int(d)
    sz = -(-n_rows // p_dst) if n_rows else 0
    dst = [torch.empty((max(0, min((q + 1) * sz, n_rows) - min(q * sz, n_rows)),) + row_shape, dtype=ref.dtype, device=ref.device)
           for q in range(p_dst)]
    arr = (dit_transfer * 64)()
    n = lib.dit_relayout_plan(n_rows, P, p_dst, arr, 64)
    if n < 0:
        _check(n, "dit_relayout_plan")
    sp = (C.c_void_p * P)(*[t.data_ptr() if t.numel() else None for t in src_shards])
    dp = (C.c_void_p * p_dst)(*[t.data_ptr() if t.numel() else None for t in dst])
    _check(lib.dit_relayout(arr, n, sp, dp, row_bytes, _stream(stream)), "dit_relayout")
    return dst


def dit_linear(A, W, bias=None, epilogue=EPI_BIAS, out=None, stream=None):
    lib = load()
    M, K = A.shape
    N = W.shape[0]
    if out is None:
        out = torch.empty((M, N), dtype=torch.float32 if epilogue == EPI_BIAS_F32 else A.dtype, device=A.device)
    _check(lib.dit_linear(_dt(A), epilogue, _ptr(A), A.stride(0), _ptr(W), _ptr(bias), _ptr(out), out.stride(0), M, N, K,
                          _stream(stream)), "dit_linear")
    return out


def dit_linear_swiglu(A, W1, b1, W3, b3, out=None, stream=None):
    """out [M, N] = SiLU(A W1^T + b1) (.) (A W3^T + b3)."""
    lib = load()
    M, K = A.shape
    N = W1.shape[0]
    if out is None:
        out = torch.empty((M, N), dtype=A.dtype, device=A.device)
    tmp = torch.empty((M, N), dtype=A.dtype, device=A.device) if A.dtype == torch.float32 else None
    _check(lib.dit_linear_swiglu(_dt(A), _ptr(A), A.stride(0), _ptr(W1), _ptr(b1), _ptr(W3), _ptr(b3), _ptr(out), out.stride(0),
                                 _ptr(tmp), M, N, K, _stream(stream)), "dit_linear_swiglu")
    return out


def dit_quantize_fp8(x, stream=None):
    """Rows of x [M, K] (bf16 / fp32) -> (e4m3 codes uint8 [M, K], fp32 row scales [M])."""
    lib = load()
    M, K = x.shape
    q = torch.empty((M, K), dtype=torch.uint8, device=x.device)
    scale = torch.empty((M,), dtype=torch.float32, device=x.device)
    _check(lib.dit_quantize_fp8(_dt(x), _ptr(x), x.stride(0), M, K, _ptr(q), q.stride(0), _ptr(scale), _stream(stream)),
           "dit_quantize_fp8")
    return q, scale


def dit_linear_fp8(Aq, a_scale, Wq, w_scale, bias=None, epilogue=EPI_BIAS, out=None, stream=None):
    """out [M, N] = epilogue(a_scale w_scale^T (.) (val(Aq) val(Wq)^T) + bias); bf16 out, fp32 for EPI_BIAS_F32."""
    lib = load()
    M, K = Aq.shape
    N = Wq.shape[0]
    if out is None:
        out = torch.empty((M, N), dtype=torch.float32 if epilogue == EPI_BIAS_F32 else torch.bfloat16, device=Aq.device)
    _check(lib.dit_linear_fp8(epilogue, _ptr(Aq), Aq.stride(0), _ptr(a_scale), _ptr(Wq), _ptr(w_scale), _ptr(bias), _ptr(out),
                              out.stride(0), M, N, K, _stream(stream)), "dit_linear_fp8")
    return out


def dit_quantize_mxfp8(x, stream=None):
    """Rows of x [M, K] (bf16 / fp32) -> (e4m3 codes uint8 [M, K], E8M0 block scales uint8 [M, K / 32])."""
    lib = load()
    M, K = x.shape
    q = torch.empty((M, K), dtype=torch.uint8, device=x.device)
    sc = torch.empty((M, K // 32), dtype=torch.uint8, device=x.device)
    _check(lib.dit_quantize_mxfp8(_dt(x), _ptr(x), x.stride(0), M, K, _ptr(q), q.stride(0), _ptr(sc), _stream(stream)),
           "dit_quantize_mxfp8")
    return q, sc


def dit_linear_mxfp8(Aq, a_scales, Wq, w_scales, bias=None, epilogue=EPI_BIAS, out=None, stream=None):
    """Block-scaled MXFP8 product: out [M, N] = epilogue(sum over 32-blocks of Xa Xw (val(Aq) val(Wq)^T) + bias)."""
    lib = load()
    M, K = Aq.shape
    N = Wq.shape[0]
    if out is None:
        out = torch.empty((M, N), dtype=torch.float32 if epilogue == EPI_BIAS_F32 else torch.bfloat16, device=Aq.device)
    _check(lib.dit_linear_mxfp8(epilogue, _ptr(Aq), Aq.stride(0), _ptr(a_scales), _ptr(Wq), _ptr(w_scales), _ptr(bias), _ptr(out),
                                out.stride(0), M, N, K, _stream(stream)), "dit_linear_mxfp8")
    return out


def dit_linear_residual(A, W, x, bias=None, gate=None, gate_stride=0, cu_seqlens=None, n_requests=1, stream=None):
    """x [M,N] fp32 <- x + gate[req(row)] (.) (A W^T + bias), in place."""
    lib = load()
    M, K = A.shape
    N = W.shape[0]
    _check(lib.dit_linear_residual(_dt(A), _ptr(A), A.stride(0), _ptr(W), _ptr(bias), _ptr(x), x.stride(0), _ptr(gate),
                                   gate_stride, _ptr(cu_seqlens), n_requests, M, N, K, _stream(stream)),
           "dit_linear_residual")
    return x


def dit_linear_qkv(A, W, bias, hidden, gq=None, gk=None, eps=1e-6, rope_cos=None, rope_sin=None, stream=None):
    """[q | k | v] = A W^T + bias with QK-RMSNorm + RoPE in the GEMM epilogue -> [M, 3 hidden] (bf16, head_dim 128)."""
    lib = load()
    M, K = A.shape
    out = torch.empty((M, 3 * hidden), dtype=A.dtype, device=A.device)
    _check(lib.dit_linear_qkv(_dt(A), _ptr(A), A.stride(0), _ptr(W), _ptr(bias), _ptr(out), out.stride(0), _ptr(gq), _ptr(gk),
                              eps, _ptr(rope_cos), _ptr(rope_sin), hidden, M, K, _stream(stream)), "dit_linear_qkv")
    return out


def dit_adaln(x, y_dtype, h=None, gate=None, shift=None, scale=None, mod_stride=0, cu_seqlens=None, n_requests=1,
              eps=1e-6, stream=None):
    """x [T,D] fp32 (updated in place when h is given) -> y [T,D] in y_dtype."""
    lib = load()
    T, D = x.shape
    y = torch.empty((T, D), dtype=y_dtype, device=x.device)
    _check(lib.dit_adaln(_dt(y), _ptr(x), _ptr(h), _ptr(gate), _ptr(shift), _ptr(scale), mod_stride, _ptr(cu_seqlens),
                         n_requests, _ptr(y), T, D, eps, _stream(stream)), "dit_adaln")
    return y


def dit_gemv(inp, W, b=None, silu_input=False, stream=None):
    lib = load()
    R, K = inp.shape
    N = W.shape[0]
    out = torch.empty((R, N), dtype=torch.float32, device=inp.device)
    _check(lib.dit_gemv(_dt(W), _ptr(inp), _ptr(W), _ptr(b), _ptr(out), R, N, K, int(silu_input), _stream(stream)),
           "dit_gemv")
    return out


def dit_qknorm_rope(qkv, n_heads, head_dim, n_tensors=2, gq=None, gk=None, eps=1e-6, rope_cos=None, rope_sin=None,
                    stream=None):
    lib = load()
    T = qkv.shape[0]
    _check(lib.dit_qknorm_rope(_dt(qkv), _ptr(qkv), qkv.stride(0), T, n_heads, head_dim, n_tensors, _ptr(gq), _ptr(gk),
                               eps, _ptr(rope_cos), _ptr(rope_sin), _stream(stream)), "dit_qknorm_rope")
    return qkv


KC = dict(gemm=0, attn=1, adaln=2, gemv=3, qknorm=4, merge=5, misc=6)


def dit_profile_begin(classes=tuple(KC)):
    mask = 0
    for c in classes:
        mask |= 1 << KC[c]
    _check(load().dit_profile_begin(mask), "dit_profile_begin")


def dit_profile_end() -> dict:
    """{class: (device ms summed over its profiled launches, launches)}"""
    ms = (C.c_float * len(KC))()
    n = (C.c_int32 * len(KC))()
    _check(load().dit_profile_end(ms, n), "dit_profile_end")
    return {k: (float(ms[i]), int(n[i])) for k, i in KC.items()}


def dit_kernel_launches() -> int:
    return int(load().dit_kernel_launches())


def dit_fallback_launches() -> int:
    """bf16 GEMM / attention launches that ran on the FFMA (fp32-path) kernels; 0 for every BASELINE.json config."""
    return int(load().dit_fallback_launches())


def dit_sim_run(cfg: dict, table: dict, requests: list):
    """Scheduling-policy simulator (include/dit_sim.h; host only).  cfg: policy ("fcfs" | "srtf" | "edf" or its number), n_ranks,
    fcfs_group, state_mb (list per class), relayout_gbps, timeout_s.  table: {(shape_class, degree): step seconds}.  requests:
    dicts with shape_class, n_steps, arrival_s, deadline_s.  Returns (list of result dicts, summary dict)."""
    lib = load()
    c = dit_sim_config()
    c.struct_size = C.sizeof(dit_sim_config)
    pol = cfg["policy"]
    c.policy = POLICY[pol] if isinstance(pol, str) else int(pol)
    c.n_ranks, c.fcfs_group = int(cfg["n_ranks"]), int(cfg.get("fcfs_group", 1))
    smb = list(cfg.get("state_mb", [0.0]))
    c.n_classes = max(len(smb), 1 + max([k[0] for k in table] + [q["shape_class"] for q in requests] + [0]))
    for i, v in enumerate(smb):
        c.state_mb[i] = float(v)
    c.relayout_gbps, c.timeout_s = float(cfg.get("relayout_gbps", 0.0)), float(cfg.get("timeout_s", 0.0))
    tab = (dit_cost_entry * max(1, len(table)))()
    for i, ((cls, deg), sec) in enumerate(sorted(table.items())):
        tab[i].shape_class, tab[i].degree, tab[i].step_s = int(cls), int(deg), float(sec)
    n = len(requests)
    rq = (dit_sim_request * max(1, n))()
    for i, q in enumerate(requests):
        rq[i].shape_class, rq[i].n_steps, rq[i].arrival_s, rq[i].deadline_s = int(q["shape_class"]), int(q["n_steps"]), float(q["arrival_s"]), float(q["deadline_s"])
    res = (dit_sim_result * max(1, n))()
    summ = dit_sim_summary()
    _check(lib.dit_sim_run(C.byref(c), tab, len(table), rq, n, res, C.byref(summ)), "dit_sim_run")
    results = [dict(finish_s=res[i].finish_s, busy_rank_s=res[i].busy_rank_s, n_migrations=res[i].n_migrations,
                    max_degree=res[i].max_degree, met_deadline=res[i].met_deadline, failed=res[i].failed) for i in range(n)]
    summary = {k: getattr(summ, k) for k, _ in dit_sim_summary._fields_}
    return results, summary
