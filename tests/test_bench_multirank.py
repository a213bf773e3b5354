"""The N > 1 path of bench.py on CPU: world_size-2 `gloo` processes (replicas only — every rank runs
its own request, no data-path collective; the only exchange is the MAX over ranks of the device times), and the
rank gating of the reference arm (rank 0 alone runs the oracle)."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    # rank r "measured" (10 + 5 r) ms for the device-resident loop and (20 - 3 r) ms end to end
    ms_total, ms_e2e = bench.max_over_ranks([10.0 + 5.0 * rank, 20.0 - 3.0 * rank], world)
    dist.barrier()
    q.put((rank, ms_total, ms_e2e, bench.job_throughput(world, 4, ms_total)))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_throughput_gloo_world2():
    world, port = 2, 29500 + os.getpid() % 2000
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms_total, ms_e2e, value in res:
        assert ms_total == 15.0 and ms_e2e == 20.0            # the slowest rank of each measurement
        assert abs(value - 2 * 4 / 15e-3) < 1e-9              # whole-job steps/s: world * steps / max time


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.max_over_ranks([3.0, 4.0], 1) == [3.0, 4.0]
    assert bench.job_throughput(1, 50, 500.0) == 100.0


def test_reference_arm_runs_on_rank0_only():
    import argparse
    import bench
    args = argparse.Namespace(workload="cfg2", steps=1, warmup=0, gpus=2)
    assert bench.run_reference(args, rank=1) is None         # returns before touching the oracle


def test_step_flops_and_workload_shapes():
    """The algorithmic flop counts behind bench.py's roofline lines, written out by hand, and the
    block-variant workloads' shapes."""
    import bench
    from paper_2606_13501_b200 import synth
    s = bench._shape("cfg2")
    T, D, F, L = 4096 + 256, 3072, 12288, 8
    fl = bench.step_flops(s)
    assert fl["gemm"] == L * (2 * T * D * 3 * D + 2 * T * D * D + 2 * 2 * T * D * F) and fl["T"] == T
    assert fl["attn"] == L * 4 * T * T * 128 * 24
    assert abs(fl["gemm"] / 1e12 - 7.886) < 1e-3 and abs(fl["attn"] / 1e12 - 1.862) < 1e-3
    g = bench._shape("cfg2_dual_gated")
    assert g.cond_mode == "joint2" and g.extras.get("mlp_gated") and g.hidden == D and g.n_blocks == L
    fg = bench.step_flops(g)
    assert fg["gemm"] - fl["gemm"] == L * 2 * T * D * F          # the gate's second up-projection; the two streams share T
    assert fg["attn"] == fl["attn"]
    assert "blocks.0.txt.mlp.w3" in synth.weight_shapes(g) and "blocks.0.mlp.w3" not in synth.weight_shapes(s)
    c3 = bench.step_flops(bench._shape("cfg3"))
    assert abs(c3["gemm"] / 1e12 - 78.54) < 0.01 and abs(c3["attn"] / 1e12 - 89.29) < 0.01
    seq = [sh.n_tokens + sh.n_cond for sh in synth.cfg4_requests()]
    c4 = bench.step_flops(bench._shape("cfg4"), seq)
    assert sum(seq) == 37376 and abs(c4["gemm"] / 1e12 - 67.72) < 0.01 and abs(c4["attn"] / 1e12 - 40.09) < 0.01
    assert "dual-stream" in bench._workload_name(g) and "BASELINE.json configs[1]" in bench._workload_name(s)
