#!/usr/bin/env python
"""bench.py — denoising steps/s of one DiT step on B200 (BASELINE.json `metric`), with the roofline of the
dominant kernel class and the CPU oracle timed beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg2|cfg3|cfg4]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

A "step" is one pass of the whole hot path (all rows) over one request: `dit_step` through the
C ABI.  Workload at N=1: BASELINE.json configs[1] (image DiT bf16: 8 blocks, D=3072, 24x128 heads, 4096 image +
256 text tokens, joint).  N>1: every rank runs the same step on its own request (independent requests shard
with no data-path collective: weak scaling) and the value is N*K / max-over-ranks time.

Prints ONE JSON line (rank 0).  `value` = steps/s with inputs resident in HBM, timed with no per-launch
instrumentation; `e2e` = the same through `dit_step_host` / `dit_step_varlen_host` (pinned HOST buffers in, host
buffer out, copies inside the timed region); `roofline` (block GEMMs) and `roofline_attention` come from a second
region of the same K steps with those launches bracketed by CUDA events, against the measured peak that matches
the SM clock sampled during that region.
`--impl reference` times the CPU oracle (oracle/dit_oracle.py, as it stands) on the host cores instead.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import torch  # noqa: E402

from paper_2606_13501_b200 import synth  # noqa: E402

METRIC = "denoising steps/s"
UNIT = "steps/s"


def _shape(workload: str):
    if workload in ("cfg2", "cfg4"):
        return synth.cfg2()
    if workload == "cfg3":
        return synth.cfg3()
    if workload.startswith("cfg2_"):   # block variants of SURVEY 8(f) item 2 at the cfg 2 shape: dual-stream (MMDiT) blocks, gated MLP
        kw = {}
        if "dual" in workload:
            kw["cond_mode"] = "joint2"
        if "gated" in workload:
            kw["extras"] = {"mlp_gated": True}
        return synth.cfg2(name="cfg2_image_bf16_" + workload[5:], **kw)
    raise SystemExit(f"unknown workload {workload}")


CFG4_NAME = ("BASELINE.json configs[3]: packed varlen batch bf16, cfg2 block shape, 6 requests "
             "{1024,1024,4096,4096,9216,16384} + 256 text tokens each (37376 packed tokens)")


def _workload_name(s) -> str:
    if s.name.startswith("cfg2_image_bf16_"):
        return ("cfg 2 shape (image DiT bf16, 8 blocks, D=3072, 24x128, 4096+256 joint tokens) with " +
                " + ".join((["dual-stream (MMDiT) joint blocks"] if s.cond_mode == "joint2" else []) +
                           (["gated (SwiGLU) MLP"] if s.extras.get("mlp_gated") else [])) + " — a block variant, not a BASELINE.json config")
    return {"cfg2_image_bf16": "BASELINE.json configs[1]: image DiT bf16, 8 blocks, D=3072, 24x128, 4096+256 joint tokens",
            "cfg3_video_bf16": "BASELINE.json configs[2]: video DiT bf16, 4 blocks, D=5120, 40x128, 32760 tokens, cross-attn 512"}[s.name]


def bench_config(s, wl_name: str, split_p: int, req_per_gpu: int, world: int) -> dict:
    """The `config` object of the JSON line — the same for both arms (`--impl ours` and `--impl reference`)."""
    weight_gb = sum(math.prod(shp) for shp in synth.weight_shapes(s).values()) * (4 if s.dtype == "f32" else 2) / 1e9
    return {"workload": wl_name, "split_p": split_p, "requests_per_gpu": req_per_gpu,
            "l2": f"inputs exceed L2: every step streams {weight_gb:.1f} GB of weights (plus activations) "
                  "through a 126 MB L2, so no step starts with its operands cached",
            "parallelism": f"replicas x{world} (independent requests, no data-path collective)"}


def step_flops(s, seq_lens=None) -> dict:
    """Algorithmic FLOPs of one step (2 per multiply-add; dense non-causal attention 4*Nq*Nk*d*H) — DESIGN.md §6.
    seq_lens: per-request sequence lengths of a packed batch (attention is block-diagonal)."""
    D, F, H, d, L = s.hidden, s.mlp_dim, s.n_heads, s.head_dim, s.n_blocks
    N = s.n_tokens
    T = N + (s.n_cond if s.cond_mode in ("joint", "joint2") else 0)
    if seq_lens is not None:
        T = sum(seq_lens)
    n_up = 3 if s.extras.get("mlp_gated") else 2     # fc1 (+ the gate's second up-projection) + fc2
    gemm = L * (2 * T * D * 3 * D + 2 * T * D * D + 2 * n_up * T * D * F)
    attn = L * 4 * (T * T if seq_lens is None else sum(t * t for t in seq_lens)) * d * H
    n_gemm = 4 * L
    if s.cond_mode == "cross":
        gemm += L * (2 * 2 * T * D * D + 2 * s.n_cond * D * 2 * D)
        attn += L * 4 * T * s.n_cond * d * H
        n_gemm += 3 * L
    return dict(gemm=gemm, attn=attn, n_gemm_launches=n_gemm, T=T)


# --------------------------------------------------------------------------------------------------------
# clocks
# --------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(gpu_index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2])); pw.append(float(c[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        os.unlink(self.f.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw), "samples": len(sm),
                "reasons": sorted(reasons)}


def _driver_version(gpu_index: int):
    try:
        r = subprocess.run(["nvidia-smi", "-i", str(gpu_index), "--query-gpu=driver_version", "--format=csv,noheader"],
                           capture_output=True, text=True, timeout=10)
        return r.stdout.strip().splitlines()[0] if r.returncode == 0 and r.stdout.strip() else None
    except (OSError, subprocess.TimeoutExpired):
        return None


def _gpu_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except (ValueError, IndexError):
            return local_rank
    return local_rank


def max_over_ranks(values, world: int, device="cpu"):
    """Per-rank device times -> the job's times: MAX over ranks (the slowest rank defines the step; contract:
    "time on the device, max over ranks").  One all_reduce on the default process group (nccl on GPUs, gloo in
    the CPU test of this function)."""
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def job_throughput(world: int, steps: int, ms_max: float) -> float:
    """Whole-job steps/s of `world` independent replicas that each ran `steps` steps: world * steps / slowest rank."""
    return world * steps / (ms_max * 1e-3)


def _peaks() -> dict:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], tf_burst=d["bf16_tflops"], tf_sust=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    src="MEASURED_PEAKS.json")
    return dict(hbm=6650.0, tf_burst=1590.0, tf_sust=1400.0, src="fallback (B200_PROFILING.md)")


# --------------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline and --impl reference)
# --------------------------------------------------------------------------------------------------------
class OracleSample:
    """The oracle (oracle/dit_oracle.py, as it stands) on a bounded sample of the workload: `dit_step` on the
    workload's own inputs with ONE of its L blocks, full token sequence.  The full-step time is extrapolated as
    t0 + L * (t1 - t0), t0 = the same call with zero blocks (embedding + conditioning + final layer)."""

    def __init__(self, s):
        from oracle import dit_oracle as O
        self.O, self.s = O, s
        import dataclasses
        one = dataclasses.replace(s, n_blocks=1)
        self.cfg1b = O.cfg_from_shape(one)
        self.cfg0b = dict(self.cfg1b, n_blocks=0)
        self.W = synth.make_weights(one)
        self.I = synth.make_inputs(s)
        self.t0 = None
        self.sample = (f"oracle dit_step (torch CPU float64) on the workload's inputs with 1 of {s.n_blocks} blocks, all "
                       f"{s.n_tokens + (s.n_cond if s.cond_mode in ('joint', 'joint2') else 0)} tokens; step time extrapolated t0 + "
                       f"{s.n_blocks}*(t1 - t0), t0 = zero-block call")

    def _run(self, cfg):
        t = time.perf_counter()
        self.O.dit_step(cfg, self.W, self.I["latents"], self.I["temb"], self.I["cond"])
        return time.perf_counter() - t

    def step_seconds(self) -> float:
        if self.t0 is None:
            self.t0 = self._run(self.cfg0b)
        t1 = self._run(self.cfg1b)
        return self.t0 + self.s.n_blocks * max(t1 - self.t0, 0.0)


REF_BUDGET_S = 240.0


def run_reference(args, rank: int):
    if rank != 0:
        return
    if args.workload == "cfg4":
        raise SystemExit("--impl reference: the oracle arm is defined for cfg2 / cfg3")
    s = _shape(args.workload)
    torch.set_num_threads(os.cpu_count() or 1)
    smp = OracleSample(s)
    # K + W samples of ~3-10 s each; a wall-clock bound keeps a large --steps within a few minutes on any host: once
    # REF_BUDGET_S are spent, no further sample is run and the line says how many were timed
    t_start = time.perf_counter()
    for i in range(args.warmup):
        if i > 0 and time.perf_counter() - t_start > REF_BUDGET_S / 4:
            break
        smp.step_seconds()
    times = []
    for _ in range(args.steps):
        if times and time.perf_counter() - t_start > REF_BUDGET_S:
            break
        times.append(smp.step_seconds())
    sec = sum(times) / len(times)
    val = 1.0 / sec
    cores = torch.get_num_threads()
    if len(times) < args.steps:
        smp.sample += f"; {len(times)} of {args.steps} steps timed ({REF_BUDGET_S:.0f} s wall-clock bound)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": len(times),
            "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": bench_config(s, _workload_name(s), args.split_p, 1, args.gpus),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": smp.sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------------------------------------
# CUDA arm
# --------------------------------------------------------------------------------------------------------
def run_ours(args, rank: int, local_rank: int, world: int):
    from paper_2606_13501_b200 import binding as B
    B.load()  # raises if the CUDA library is missing: there is no fallback
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    import torch.distributed as dist
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()

    s = _shape(args.workload)
    W = synth.make_weights(s, device=dev)
    K, Wm = args.steps, args.warmup
    if args.workload == "cfg4":
        # packed varlen batch: R requests through ONE dit_step_varlen call per step
        shapes = synth.cfg4_requests()
        R = len(shapes)
        ts = [float(synth.uniform01(7, f"t{r}", 1)[0]) * 1000 for r in range(R)]
        Is = [synth.make_inputs(sh, device=dev, tag=f".r{r}.rank{rank}", t=ts[r]) for r, sh in enumerate(shapes)]
        seq = [sh.n_tokens + sh.n_cond for sh in shapes]
        fl = step_flops(s, seq)
        m = B.Dit(B.make_config(shapes[-1], split_p=args.split_p, max_tokens=sum(seq), max_requests=R,
                                max_cond_tokens=sum(sh.n_cond for sh in shapes)), W, dev)
        lats, conds = [i["latents"] for i in Is], [i["cond"] for i in Is]
        tembs = torch.cat([i["temb"] for i in Is]).contiguous()
        packed_h = torch.cat([l.reshape(-1) for l in lats]).cpu().pin_memory()
        cond_h = torch.cat(conds).cpu().pin_memory()
        tembs_h = tembs.cpu().pin_memory()
        out_h = torch.empty_like(packed_h).pin_memory()
        lat_shapes, n_conds = [tuple(l.shape) for l in lats], [int(c.shape[0]) for c in conds]
        h2d = sum(t.numel() * t.element_size() for t in (packed_h, cond_h, tembs_h))
        d2h = out_h.numel() * out_h.element_size()

        def step():
            return m.dit_step_varlen(lats, tembs, conds)

        def step_e2e():   # dit_step_varlen_host: ONE C-ABI call with HOST buffers (the library enqueues H2D, step, D2H)
            m.dit_step_varlen_host(packed_h, lat_shapes, tembs_h, cond_h, n_conds, out_h)
        wl_name, req_per_gpu = CFG4_NAME, R
    else:
        fl = step_flops(s)
        m = B.Dit(B.make_config(s, split_p=args.split_p), W, dev)
        I = synth.make_inputs(s, device=dev, tag=f".rank{rank}")
        lat, temb, cond = I["latents"], I["temb"][0].contiguous(), I["cond"]
        out = torch.empty_like(lat)
        lat_h, temb_h = lat.cpu().pin_memory(), temb.cpu().pin_memory()
        cond_h = None if cond is None else cond.cpu().pin_memory()
        out_h = torch.empty_like(lat_h).pin_memory()
        h2d = lat_h.numel() * lat_h.element_size() + temb_h.numel() * 4 + (0 if cond_h is None else cond_h.numel() * cond_h.element_size())
        d2h = out_h.numel() * out_h.element_size()

        def step():
            return m.dit_step(lat, temb, cond, out)

        def step_e2e():   # dit_step_host: the C-ABI call with HOST buffers (copies are enqueued by the library)
            m.dit_step_host(lat_h, temb_h, cond_h, out_h)
        wl_name, req_per_gpu = _workload_name(s), 1

    for _ in range(Wm):
        step()
    torch.cuda.synchronize()

    # ---- timed region: K steps, device-resident inputs, NO per-launch instrumentation (this is `value`)
    sampler = ClockSampler(_gpu_index(local_rank))
    time.sleep(0.25)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier(); torch.cuda.synchronize()
    n0 = B.dit_kernel_launches()
    e0.record()
    for _ in range(K):
        step()
    e1.record()
    torch.cuda.synchronize(); barrier()
    launches = B.dit_kernel_launches() - n0
    clocks = sampler.stop()
    ms_total = e0.elapsed_time(e1)

    # ---- roofline region: the same K back-to-back steps again with every block-GEMM and attention launch bracketed by a
    # CUDA-event pair on the launching stream (dit_profile_begin).  Kept apart from the region above: the event pairs
    # (2 x 40 per cfg 2 step) stop PDL overlap between neighbours and would perturb `value`.
    sampler_r = ClockSampler(_gpu_index(local_rank))
    torch.cuda.synchronize()
    r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    B.dit_profile_begin(("gemm", "attn"))
    r0.record()
    for _ in range(K):
        step()
    r1.record()
    torch.cuda.synchronize()
    prof = B.dit_profile_end()
    clocks_r = sampler_r.stop()
    ms_roof = r0.elapsed_time(r1)

    # ---- e2e: dit_step_host / dit_step_varlen_host, pinned host buffers, H2D + step + D2H per step inside the timed region
    for _ in range(min(Wm, 3)):
        step_e2e()
    torch.cuda.synchronize()
    barrier(); torch.cuda.synchronize()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    f0.record()
    for _ in range(K):
        step_e2e()
        torch.cuda.current_stream().synchronize()      # the step's result is on the host before the next step starts
    f1.record()
    torch.cuda.synchronize(); barrier()
    ms_e2e = f0.elapsed_time(f1)

    # ---- burst: single steps with >= 200 ms of idle before each ("state burst vs sustained"); median and best
    burst_ms = []
    if world == 1:
        for _ in range(max(3, min(K, 8))):
            torch.cuda.synchronize()
            time.sleep(0.2)
            b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            b0.record(); step(); b1.record()
            torch.cuda.synchronize()
            burst_ms.append(b0.elapsed_time(b1))

    # ---- per-class breakdown (separate, untimed-for-value pass with every class bracketed)
    B.dit_profile_begin()
    for _ in range(max(1, min(K, 5))):
        step()
    torch.cuda.synchronize()
    prof_all = B.dit_profile_end()
    nb = max(1, min(K, 5))

    ms_total, ms_e2e = max_over_ranks([ms_total, ms_e2e], world, dev)

    if rank == 0:
        pk = _peaks()

        def roof(cls, flops_per_step, kernel, wl_key):
            ms, n = prof[cls]
            ach = (flops_per_step * K) / (ms * 1e-3) / 1e12 if ms > 0 else 0.0
            # which measured peak applies is decided by the SM clock sampled DURING this region: at >= 0.9 of the maximum
            # the part is in its burst regime (MEASURED_PEAKS.json bf16_tflops), below it under the power cap (sustained)
            sm, mx = clocks_r.get("sm_mhz"), clocks_r.get("sm_max_mhz")
            burst = bool(sm and mx and sm >= 0.9 * mx)
            peak = pk["tf_burst"] if burst else pk["tf_sust"]
            traffic = None
            tp = os.path.join(ROOT, "profiles", "traffic.csv")   # DRAM bytes per launch from the ncu --set full capture
            if os.path.exists(tp):
                for ln in open(tp).read().splitlines()[1:]:
                    f = ln.split(",")
                    if len(f) >= 3 and f[0] == ("cfg2" if args.workload == "cfg4" else args.workload) and f[1] == wl_key:
                        traffic = int(f[2])
            return {"bound": "tensor", "kernel": kernel, "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                    "frac": ach / peak, "peak_source": pk["src"] + (" bf16_tflops (burst: " if burst else " bf16_tflops_sustained (") +
                    f"SM clock {sm} of {mx} MHz sampled during the region)",
                    "frac_burst": ach / pk["tf_burst"], "frac_sustained": ach / pk["tf_sust"], "frac_of_nominal_2250": ach / 2250.0,
                    "launches": n, "avg_launch_ms": ms / max(1, min(n, 16384)), "share_of_step": ms / ms_roof,
                    "flops_per_step": flops_per_step, "traffic": traffic,
                    "timed": f"CUDA events around every launch of the class over {K} back-to-back steps (a second region; "
                             "`value` is timed without them)"}

        line = {
            "metric": METRIC, "value": job_throughput(world, K, ms_total), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16",
            "data": "synthetic",
            "config": bench_config(s, wl_name, args.split_p, req_per_gpu, world),
            "clocks": clocks,
            "device": {"name": torch.cuda.get_device_name(dev), "sms": torch.cuda.get_device_properties(dev).multi_processor_count,
                       "torch": torch.__version__, "cuda": torch.version.cuda, "driver": _driver_version(_gpu_index(local_rank)), "peaks": pk,
                       "timing": f"{K} back-to-back steps after {Wm} warm-ups, CUDA events, no per-launch instrumentation"},
            "e2e": {"value": job_throughput(world, K, ms_e2e), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "call": "dit_step_varlen_host" if args.workload == "cfg4" else "dit_step_host"},
            "gpu_launches": launches, "fallback_launches": B.dit_fallback_launches(),
            "roofline": roof("gemm", fl["gemm"], "block GEMMs (QKV, out-proj, fc1, fc2" + (", cross projections)" if s.cond_mode == "cross" else ")"), "gemm"),
            "roofline_attention": roof("attn", fl["attn"], "attention (self" + (" + cross)" if s.cond_mode == "cross" else ")"), "attn"),
            "clocks_roofline_region": clocks_r,
            "burst": ({"ms_per_step_median": statistics.median(burst_ms), "ms_per_step_best": min(burst_ms), "samples": len(burst_ms),
                       "steps_per_s_median": 1e3 / statistics.median(burst_ms),
                       "how": "single steps, each after >= 200 ms of idle (the part boosts; `value` is the sustained back-to-back rate)"}
                      if burst_ms else None),
            "breakdown_ms_per_step": {k: round(v[0] / nb, 4) for k, v in prof_all.items()},
            "tflops": {"attention": (fl["attn"] * nb) / (prof_all["attn"][0] * 1e-3) / 1e12 if prof_all["attn"][0] > 0 else None,
                       "gemm": (fl["gemm"] * nb) / (prof_all["gemm"][0] * 1e-3) / 1e12 if prof_all["gemm"][0] > 0 else None,
                       "step_total": (fl["gemm"] + fl["attn"]) * K / (ms_total * 1e-3) / 1e12},
        }
        if world == 1 and not args.no_cpu_baseline and args.workload != "cfg4":
            torch.set_num_threads(os.cpu_count() or 1)
            smp = OracleSample(s)
            sec = smp.step_seconds()
            line["cpu_baseline"] = {"value": 1.0 / sec, "unit": UNIT, "cores": torch.get_num_threads(), "kind": "oracle",
                                    "sample": smp.sample}
        if world == 1 and not args.no_cpu_baseline and args.workload == "cfg4":
            # The packed batch is DEFINED as its requests one by one (DESIGN.md section 3 step 8): the oracle is timed on the
            # two smallest distinct requests (1024 and 4096 image tokens), one block each, and the others are extrapolated
            # with t(T) = a T + b T^2 (per-token work + attention) fitted to the two.
            torch.set_num_threads(os.cpu_count() or 1)
            reqs = synth.cfg4_requests()
            Ts = [sh.n_tokens + sh.n_cond for sh in reqs]
            t_of = {}
            for sh in (reqs[0], reqs[2]):
                t_of[sh.n_tokens + sh.n_cond] = OracleSample(sh).step_seconds()
            (T1, t1), (T2, t2) = sorted(t_of.items())
            b_ = (t2 / T2 - t1 / T1) / (T2 - T1)
            a_ = t1 / T1 - b_ * T1
            sec = sum(a_ * T + b_ * T * T for T in Ts)
            line["cpu_baseline"] = {"value": 1.0 / sec, "unit": UNIT, "cores": torch.get_num_threads(), "kind": "oracle",
                                    "sample": f"oracle dit_step (torch CPU float64) on requests 0 and 2 alone ({T1} and {T2} tokens, 1 of "
                                              f"{s.n_blocks} blocks each, extrapolated to the step as in the other workloads: {t1:.1f} s and "
                                              f"{t2:.1f} s); the six requests' times from t(T) = a T + b T^2 fitted to the two, summed"}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# --------------------------------------------------------------------------------------------------------
# trajectory arm: dit_sample over a whole request, stream launches vs one CUDA-graph launch
# --------------------------------------------------------------------------------------------------------
def run_traj(args):
    """`--workload traj`: one request of cfg 2 shape through `dit_sample` (n denoising steps chained by the Euler
    update on the device, no host round trip between steps).  Reports denoising steps/s of the trajectory when its
    kernels are launched one by one on the stream and when the captured CUDA graph is replayed with one launch, plus a
    classifier-free-guided trajectory as two passes per step and as ONE packed pass of two requests per step (a handle with
    room for both).  `--steps` = trajectories timed, `--traj-steps` = n."""
    from paper_2606_13501_b200 import binding as B
    B.load()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    s = _shape("cfg2")
    n = args.traj_steps
    W = synth.make_weights(s, device=dev)
    m1 = B.Dit(B.make_config(s, split_p=args.split_p), W, dev)
    m2 = B.Dit(B.make_config(s, split_p=args.split_p, max_requests=2, max_tokens=2 * (s.n_tokens + s.n_cond),
                             max_cond_tokens=2 * s.n_cond), W, dev)
    # the same two handles with room for the whole trajectory's modulation vectors (dit_config.max_sample_steps)
    m1a = B.Dit(B.make_config(s, split_p=args.split_p, max_sample_steps=n), W, dev)
    m2a = B.Dit(B.make_config(s, split_p=args.split_p, max_requests=2, max_tokens=2 * (s.n_tokens + s.n_cond),
                              max_cond_tokens=2 * s.n_cond, max_sample_steps=n), W, dev)
    I = synth.make_inputs(s, device=dev)
    lat, cond = I["latents"], I["cond"]
    unc = synth.normal(s.seed, "uncond", tuple(cond.shape), dtype=s.torch_dtype, device=dev)
    tembs = synth.timestep_embedding([1000.0 * (1 - i / n) for i in range(n)], s.temb_dim, device=dev).contiguous()
    sigmas = [1.0 - i / n for i in range(n + 1)]
    out = torch.empty_like(lat)
    K, Wm = max(1, min(args.steps, 10)), max(1, min(args.warmup, 3))
    rows = []
    for name, m, u, graph in (("stream launches", m1, None, False), ("cuda graph", m1, None, True),
                              ("guided (2 passes/step), cuda graph", m1, unc, True),
                              ("guided (1 packed pass of 2 requests/step), cuda graph", m2, unc, True),
                              ("cuda graph, modulation of all steps computed ahead", m1a, None, True),
                              ("guided (2 passes/step), cuda graph, modulation ahead", m1a, unc, True),
                              ("guided (1 packed pass/step), cuda graph, modulation ahead", m2a, unc, True)):
        for _ in range(Wm):
            m.dit_sample(lat, tembs, sigmas, cond, u, 4.0, use_graph=graph, out=out)
        torch.cuda.synchronize()
        n0 = B.dit_kernel_launches()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record()
        for _ in range(K):
            m.dit_sample(lat, tembs, sigmas, cond, u, 4.0, use_graph=graph, out=out)
        t_enq = time.perf_counter() - t0
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / K
        rows.append({"mode": name, "ms_per_trajectory": ms, "denoising_steps_per_s": n / (ms * 1e-3),
                     "model_passes_per_s": (2 if u is not None else 1) * n / (ms * 1e-3),
                     "host_enqueue_ms_per_trajectory": t_enq / K * 1e3,
                     "library_launch_calls_per_trajectory": (B.dit_kernel_launches() - n0) / K})
    # ONE step per C-ABI call (what the headline bench times), launched kernel by kernel and replayed from the graph the
    # handle caches (dit_step_graph): device time per step and what the call costs the calling thread
    single = []
    for name, fn in (("dit_step", m1.dit_step), ("dit_step_graph", m1.dit_step_graph)):
        for _ in range(3):
            fn(lat, tembs[0], cond, out=out)
        torch.cuda.synchronize()
        reps = 8                                          # 8 x 65 launches stay below the driver's launch queue depth: no back-pressure in the host time
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record()
        for _ in range(reps):
            fn(lat, tembs[0], cond, out=out)
        t_enq = time.perf_counter() - t0
        e1.record()
        torch.cuda.synchronize()
        single.append({"call": name, "ms_per_step": e0.elapsed_time(e1) / reps, "host_enqueue_us_per_step": t_enq / reps * 1e6})
    print(json.dumps({"metric": "trajectory denoising steps/s", "unit": UNIT, "n_gpus": 1, "trajectories": K, "warmup": Wm,
                      "config": {"workload": _workload_name(s), "traj_steps": n, "split_p": args.split_p}, "dtype": "bf16",
                      "data": "synthetic", "rows": rows, "single_step": single}), flush=True)


# --------------------------------------------------------------------------------------------------------
# per-kernel arm: every HBM-bound kernel and the attention sweep (BASELINE.json configs[4]) timed ALONE
# --------------------------------------------------------------------------------------------------------
def run_kernels(args):
    """`--workload kernels`: one JSON line with a list of per-kernel measurements.  Every kernel is launched through
    the C ABI at the sizes it has inside cfg 2 / cfg 3 / cfg 5, timed with CUDA events on the launching stream; between
    timed launches a 512 MB buffer is overwritten so nothing is served from the 126 MB L2.  `frac` is against
    MEASURED_PEAKS.json: the burst figures, because each kernel is timed alone (HBM GB/s copy peak; bf16 TFLOP/s)."""
    from paper_2606_13501_b200 import binding as B
    B.load()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    pk = _peaks()
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    reps = max(3, min(args.steps, 20))
    bf = torch.bfloat16

    def timeit(fn):
        ts = []
        for i in range(args.warmup + reps):
            flush.fill_(i & 0xff)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record()
            torch.cuda.synchronize()
            if i >= args.warmup:
                ts.append(e0.elapsed_time(e1))
        return statistics.median(ts), min(ts)

    rows = []

    def hbm(name, nbytes, fn):
        if args.only and args.only not in name:
            return
        med, best = timeit(fn)
        gbs = nbytes / (med * 1e-3) / 1e9
        rows.append({"kernel": name, "bound": "hbm", "bytes": nbytes, "ms": round(med, 5), "ms_best": round(best, 5),
                     "achieved": round(gbs, 1), "unit": "GB/s", "peak": pk["hbm"], "frac": round(gbs / pk["hbm"], 4)})

    def tensor(name, flops, fn, fp8=False):
        if args.only and args.only not in name:
            return
        med, best = timeit(fn)
        tf = flops / (med * 1e-3) / 1e12
        # an e4m3 contraction takes the peak for its own dtype: the measured bf16 figure x the nominal 2 : 1 ratio (4.5 : 2.25 PFLOP/s)
        peak, nominal = (2 * pk["tf_burst"], 4500.0) if fp8 else (pk["tf_burst"], 2250.0)
        row = {"kernel": name, "bound": "tensor", "flops": flops, "ms": round(med, 5), "ms_best": round(best, 5),
               "achieved": round(tf, 1), "unit": "TFLOP/s", "peak": peak, "frac": round(tf / peak, 4)}
        row["frac_of_nominal_4500" if fp8 else "frac_of_nominal_2250"] = round(tf / nominal, 4)
        rows.append(row)

    rn = lambda name, shape, dt, std=1.0: synth.normal(5, name, shape, std=std, dtype=dt, device=dev)
    # ---- adaLN (a5 / a9): 4D read + 2D write per token
    for T, D in ((4352, 3072), (32760, 5120)):
        x, mod = rn("x", (T, D), torch.float32), rn("mod", (1, 2 * D), torch.float32, 0.3)
        hbm(f"adaln T={T} D={D}", T * D * 6, lambda: B.dit_adaln(x, bf, shift=mod[:, :D], scale=mod[:, D:], mod_stride=2 * D))
        del x
    # ---- modulation GEMV (a2): weights streamed once
    for L, D in ((8, 3072), (4, 5120)):
        N = L * 6 * D + 2 * D
        Wm, bm, c = rn("Wmod", (N, D), bf, 0.02), rn("bmod", (N,), bf, 0.02), rn("c", (1, D), torch.float32)
        hbm(f"gemv modulation N={N} K={D}", N * D * 2 + N * 2 + N * 4, lambda: B.dit_gemv(c, Wm, bm, silu_input=True))
        del Wm
    # ---- QK-RMSNorm + RoPE in place on q,k (read + write 2 of the 3 thirds of qkv)
    for T, H in ((4352, 24), (32760, 40)):
        D = H * 128
        qkv = rn("qkv", (T, 3 * D), bf)
        g = rn("g", (128,), bf, 0.02) + 1
        rc, rs = rn("rc", (T, 64), torch.float32), rn("rs", (T, 64), torch.float32)
        hbm(f"qknorm_rope T={T} H={H}", 2 * 2 * T * D * 2 + 2 * T * 64 * 4,
            lambda: B.dit_qknorm_rope(qkv, H, 128, 2, g, g, 1e-6, rc, rs))
        del qkv
    # ---- LSE merge (a14)
    for Nq, H, P in ((32768, 40, 4), (4352, 24, 2), (32768, 40, 8)):
        op = [rn(f"o{p}", (Nq, H, 128), bf) for p in range(P)]
        lp = [rn(f"l{p}", (Nq, H), torch.float32) for p in range(P)]
        hbm(f"merge Nq={Nq} H={H} P={P}", P * (Nq * H * 128 * 2 + Nq * H * 4) + Nq * H * 128 * 2 + Nq * H * 4,
            lambda: B.dit_attn_merge(op, lp))
        del op
    # ---- re-layout P -> P' of the residual stream: reads and writes the artifact once
    for T, D, ps, pd in ((32760, 5120, 4, 8), (4352, 3072, 2, 4)):
        full = rn("relayout", (T, D), torch.float32)
        sz = -(-T // ps)
        src = [full[p * sz:min((p + 1) * sz, T)].contiguous() for p in range(ps)]
        hbm(f"relayout T={T} D={D} P={ps}->{pd}", 2 * T * D * 4, lambda: B.dit_relayout(src, pd))
        del full, src
    # ---- block GEMMs.  Order of this arm: everything small first; the 3 ms cfg 3 GEMMs and the 10-17 ms attention launches at
    #      N >= 32768 sit on the power cap and depress whatever is timed in the seconds after them (measured: cfg 2 GEMMs
    #      1337 instead of 1615 TFLOP/s, attention N = 4096 540 instead of 1004 when timed after them).
    def gemm_rows(cfg, T, D, F_):
        for nm, M, N, K, epi in ((f"qkv {cfg}", T, 3 * D, D, B.EPI_BIAS), (f"fc1 {cfg}", T, F_, D, B.EPI_BIAS_GELU)):
            A, Wt, b = rn("A", (M, K), bf), rn("W", (N, K), bf, 0.02), rn("b", (N,), bf, 0.02)
            o = torch.empty((M, N), dtype=bf, device=dev)
            tensor(f"gemm {nm} {M}x{N}x{K}", 2 * M * N * K, lambda: B.dit_linear(A, Wt, b, epi, out=o))
            # fp8 (e4m3) linear layer (R42) and its row quantisation kernel, same shape
            hbm(f"quantize fp8 {nm} {M}x{K}", 3 * M * K + 4 * M, lambda: B.dit_quantize_fp8(A))
            Aq, sa = B.dit_quantize_fp8(A)
            Wq, sw = B.dit_quantize_fp8(Wt)
            del A, Wt
            tensor(f"gemm fp8 {nm} {M}x{N}x{K}", 2 * M * N * K, lambda: B.dit_linear_fp8(Aq, sa, Wq, sw, b, epi, out=o), fp8=True)
            del Aq, Wq
            # block-scaled MXFP8 (R43): E8M0 scale per 32 elements, applied by the tensor core
            A2, W2 = rn("A", (M, K), bf), rn("W", (N, K), bf, 0.02)
            hbm(f"quantize mxfp8 {nm} {M}x{K}", 3 * M * K + M * K // 32, lambda: B.dit_quantize_mxfp8(A2))
            Am, sam = B.dit_quantize_mxfp8(A2)
            Wm, swm = B.dit_quantize_mxfp8(W2)
            del A2, W2
            tensor(f"gemm mxfp8 {nm} {M}x{N}x{K}", 2 * M * N * K, lambda: B.dit_linear_mxfp8(Am, sam, Wm, swm, b, epi, out=o), fp8=True)
            del Am, Wm, o
        # gated-MLP up-projection (R40): W1 | W3 in one kernel, 2 x 2 T F D flops
        y = rn("y", (T, D), bf)
        w1, w3 = rn("w1", (F_, D), bf, 0.02), rn("w3", (F_, D), bf, 0.02)
        b1, b3 = rn("b1", (F_,), bf, 0.02), rn("b3", (F_,), bf, 0.02)
        o = torch.empty((T, F_), dtype=bf, device=dev)
        tensor(f"gemm swiglu fc1 {cfg} {T}x2x{F_}x{D}", 4 * T * F_ * D, lambda: B.dit_linear_swiglu(y, w1, b1, w3, b3, out=o))
        del y, w1, w3, o
        for nm, M, N, K in ((f"out-proj {cfg}", T, D, D), (f"fc2 {cfg}", T, D, F_)):
            A, Wt, b = rn("A", (M, K), bf), rn("W", (N, K), bf, 0.02), rn("b", (N,), bf, 0.02)
            x, g = rn("x", (M, N), torch.float32), rn("g", (1, N), torch.float32, 0.02)
            tensor(f"gemm+gate-residual {nm} {M}x{N}x{K}", 2 * M * N * K, lambda: B.dit_linear_residual(A, Wt, x, b, g, N))
            del A, Wt, x

    # ---- attention sweep (cfg 5): unsplit, d=128
    def attn_rows(Ns):
        for N in Ns:
            for H in (24, 40):
                q, k, v = synth.make_attention_qkv(11, N, N, H, 128, device=dev)
                tensor(f"attention H={H} N={N}", 4 * N * N * 128 * H, lambda: B.dit_attn_partial(q, k, v, want_lse=True))
                del q, k, v

    # ---- split-KV partial attention + LSE merge (cfg 5: P contiguous KV shards, the single-GPU analogue of SP degree P)
    def split_rows(N, H, Ps):
        q, k, v = synth.make_attention_qkv(11, N, N, H, 128, device=dev)
        for P in Ps:
            sz = -(-N // P)                                  # R20: contiguous shards of ceil(N / P) keys

            def run():
                parts = [B.dit_attn_partial(q, k[p * sz:(p + 1) * sz], v[p * sz:(p + 1) * sz], want_lse=True) for p in range(P)]
                return B.dit_attn_merge([o for o, _ in parts], [l for _, l in parts])
            tensor(f"attention split-KV P={P} + merge H={H} N={N}", 4 * N * N * 128 * H, run)
        del q, k, v

    gemm_rows("cfg2", 4352, 3072, 12288)
    attn_rows((1024, 2048, 4096, 8192, 16384))
    split_rows(16384, 24, (2, 4, 8))
    gemm_rows("cfg3", 32760, 5120, 13824)
    attn_rows((32768,) if args.steps < 20 else (32768, 65536, 131072))
    print(json.dumps({"metric": "per-kernel roofline", "n_gpus": 1, "reps": reps, "warmup": args.warmup,
                      "l2": "512 MB overwritten between timed launches", "peaks": pk, "kernels": rows}), flush=True)



# --------------------------------------------------------------------------------------------------------
# policy-simulator arm: measured step times -> cost model -> FCFS / SRTF / EDF on a synthetic trace
# --------------------------------------------------------------------------------------------------------
def run_sim(args):
    """`--workload sim`: times `dit_step` (cfg 2 block shape, 8 blocks) at the paper's three image request shapes
    (512^2 / 1024^2 / 1536^2 -> 1024 / 4096 / 9216 image tokens + 256 text tokens) on this GPU, builds the cost
    table cost(shape, P) for P = 1, 2, 4, 8 — P = 1 measured; P > 1 modelled as per-row work / P plus one all-gather of the
    block's K | V shards per block at the measured NVLink peer bandwidth (B200_PROFILING.md: 770 GB/s per direction) — and
    replays one seeded Poisson trace (S : M : L = 5 : 3 : 2, 20 steps per request, the paper's Qwen-Image SLO multipliers
    1.5 / 2.0 / 6.0 + 1 s) through `dit_sim_run` for the three policies of PAPER.md:299-303 on 8 ranks."""
    from paper_2606_13501_b200 import binding as B
    B.load()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    base = synth.cfg2()
    W = synth.make_weights(base, device=dev)
    sides = (64, 128, 192)                                   # latent side; patch 2 -> 1024 / 4096 / 9216 tokens
    m = B.Dit(B.make_config(synth.cfg2(latent_grid=(1, sides[-1], sides[-1]))), W, dev)
    step_s, tokens = [], []
    for side in sides:
        sh = synth.cfg2(latent_grid=(1, side, side))
        I = synth.make_inputs(sh, device=dev)
        lat, temb, cond = I["latents"], I["temb"][0].contiguous(), I["cond"]
        out = torch.empty_like(lat)
        for _ in range(3):
            m.dit_step(lat, temb, cond, out)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        K = max(5, min(args.steps, 20))
        e0.record()
        for _ in range(K):
            m.dit_step(lat, temb, cond, out)
        e1.record()
        torch.cuda.synchronize()
        step_s.append(e0.elapsed_time(e1) / K * 1e-3)
        tokens.append(sh.n_tokens + sh.n_cond)
    D, L, nvlink = base.hidden, base.n_blocks, 770e9
    table = {}
    for c, (t1, T) in enumerate(zip(step_s, tokens)):
        for P in (1, 2, 4, 8):
            gather = 0.0 if P == 1 else L * (2 * T * D * 2) * (P - 1) / P / nvlink      # K | V of the other P - 1 shards, per block
            table[(c, P)] = t1 / P + gather
    n_req, n_steps, rate = 400, 20, 0.9 / (sum(w * t for w, t in zip((0.5, 0.3, 0.2), step_s)) * 20 / 8)   # ~90 % load of 8 ranks at P = 1
    u = synth.uniform01(17, "sim.trace", 2 * n_req).tolist()
    t, reqs = 0.0, []
    alpha = (1.5, 2.0, 6.0)
    for i in range(n_req):
        t += -math.log(u[2 * i]) / rate
        c = 0 if u[2 * i + 1] < 0.5 else (1 if u[2 * i + 1] < 0.8 else 2)
        reqs.append(dict(shape_class=c, n_steps=n_steps, arrival_s=t, deadline_s=t + alpha[c] * n_steps * step_s[c] + 1.0))
    state_mb = [(T * 64 * 2 + 256 * D * 2) / 1e6 for T in tokens]                       # latents + text embeddings
    rows = []
    for pol, grp in (("fcfs", 1), ("fcfs", 4), ("srtf", 1), ("edf", 1)):
        cfg = dict(policy=pol, n_ranks=8, fcfs_group=grp, state_mb=state_mb, relayout_gbps=nvlink / 1e9, timeout_s=1500.0)
        t0 = time.perf_counter()
        _, summ = B.dit_sim_run(cfg, table, reqs)
        wall = time.perf_counter() - t0
        rows.append(dict(policy=pol + (f"-SP{grp}" if pol == "fcfs" else ""), **{k: round(v, 6) if isinstance(v, float) else v for k, v in summ.items()},
                         sim_wall_ms=round(wall * 1e3, 3), events_per_s=round(summ["n_events"] / wall) if wall > 0 else None))
    print(json.dumps({"metric": "policy simulation on measured step times", "n_gpus": 1, "data": "synthetic",
                      "config": {"workload": "cfg2 block shape at 512^2 / 1024^2 / 1536^2 (+256 text tokens), 20-step requests, 8 simulated ranks",
                                 "trace": f"{n_req} requests, Poisson rate {rate:.2f}/s, S:M:L = 5:3:2, deadline = a + alpha T + 1 s"},
                      "measured_step_s_P1": step_s, "cost_table": {f"{c},{P}": round(v, 6) for (c, P), v in sorted(table.items())},
                      "policies": rows}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=["cfg2", "cfg3", "cfg4", "kernels", "traj", "sim", "cfg2_dual", "cfg2_gated", "cfg2_dual_gated"])
    ap.add_argument("--traj-steps", type=int, default=20, help="--workload traj: denoising steps per trajectory")
    ap.add_argument("--split-p", type=int, default=1)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--only", default="", help="--workload kernels: time only the kernels whose name contains this")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.workload == "kernels":
        if rank == 0:
            run_kernels(args)
    elif args.workload == "traj":
        if rank == 0:
            run_traj(args)
    elif args.workload == "sim":
        if rank == 0:
            run_sim(args)
    elif args.impl == "reference":
        run_reference(args, rank)
    else:
        run_ours(args, rank, local_rank, world)


if __name__ == "__main__":
    main()
