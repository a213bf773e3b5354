"""Writes tests/golden/cfg3_oracle_rows.pt: sampled rows of ONE FULL END-TO-END oracle step at BASELINE.json's full
size, for the configuration whose whole-step oracle is too slow to run inside `pytest -m gpu` (cfg 3: 168 TFLOP of fp64
CPU work and ~65 GB of host memory: the oracle materialises the 32760 x 32760 fp64 score matrix of a head, as the plain
definition says).

    python tests/golden/make_fullsize_oracle.py --cfg 3 [--out FILE]     # CPU only; needs a host with > 70 GB of RAM

It calls ONLY `oracle/dit_oracle.py` (as it stands) and the seeded input generator `paper_2606_13501_b200/synth.py`
(which holds none of the method's arithmetic).  No value comes from the CUDA path.  The GPU test
(tests/test_gpu_fullsize.py) regenerates the same inputs from the same seeds, runs the whole step on the device and
compares the same rows.

Stored (float32, a few hundred kB to ~2 MB):
  rows_tok [n]        sampled token indices (seeded), tok [n, C*pv] = the final layer's output rows ("tok" tap; `out` is
                      its unpatchify), i.e. the END-TO-END result of all blocks;
  rows_x [m]          sampled sequence rows, x_blocks [L, m, D] = the residual stream after every block at those rows
                      (the accumulation curve of the error across blocks);
  out_rms             RMS of the whole oracle output (the max-abs bar is 3e-2 x this);
  meta                config name, seeds, sha256 of oracle/dit_oracle.py at the time of writing, wall time, host.
"""
from __future__ import annotations

import argparse
import hashlib
import os
import platform
import sys
import time

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import dit_oracle as O  # noqa: E402
from paper_2606_13501_b200 import synth  # noqa: E402


class KeepTaps(dict):
    """A taps dict that keeps only the named intermediates (the others are GBs each at this size)."""

    def __init__(self, keep):
        super().__init__()
        self.keep = set(keep)

    def __setitem__(self, k, v):
        if k in self.keep:
            super().__setitem__(k, v)


def sample_rows(seed: int, name: str, n_total: int, n: int) -> torch.Tensor:
    """n distinct row indices in [0, n_total), seeded; always holds row 0, a tile boundary (127, 128) and the last row."""
    fixed = [r for r in (0, 127, 128, n_total - 1) if 0 <= r < n_total]
    picked = list(dict.fromkeys(fixed + [int(x * n_total) for x in synth.uniform01(seed, name, 4 * n).tolist()]))
    return torch.tensor(sorted(picked[:n]), dtype=torch.int64)


def run_cfg3(out_path: str, n_tok: int, n_x: int, smoke: bool = False):
    s = synth.cfg3() if not smoke else synth.cfg3(n_blocks=2, hidden=256, n_heads=2, mlp_dim=512, cond_dim=256,
                                                   latent_grid=(3, 12, 16), n_cond=40)
    torch.set_num_threads(os.cpu_count() or 1)
    t0 = time.time()
    W = synth.make_weights(s)
    I = synth.make_inputs(s)
    print(f"inputs generated in {time.time() - t0:.0f} s", flush=True)
    keep = ["tok"] + [f"b{l}.x_mlp" for l in range(s.n_blocks)]
    taps = KeepTaps(keep)
    t1 = time.time()
    out = O.dit_step(O.cfg_from_shape(s), W, I["latents"], I["temb"], I["cond"], taps=taps)
    wall = time.time() - t1
    print(f"oracle step: {wall:.0f} s", flush=True)
    rows_tok = sample_rows(s.seed, "golden.rows_tok", s.n_tokens, n_tok)
    rows_x = sample_rows(s.seed, "golden.rows_x", s.n_tokens, n_x)
    blob = {
        "rows_tok": rows_tok, "tok": taps["tok"][rows_tok].to(torch.float32),
        "rows_x": rows_x, "x_blocks": torch.stack([taps[f"b{l}.x_mlp"][rows_x] for l in range(s.n_blocks)]).to(torch.float32),
        "out_rms": float(out.pow(2).mean().sqrt()), "tok_rms": float(taps["tok"].pow(2).mean().sqrt()),
        "meta": {"config": s.name, "seed": s.seed, "t": I["t"],
                 "oracle_sha256": hashlib.sha256(open(os.path.join(ROOT, "oracle", "dit_oracle.py"), "rb").read()).hexdigest(),
                 "oracle_wall_s": wall, "threads": torch.get_num_threads(), "host": platform.processor() or platform.machine(),
                 "torch": str(torch.__version__), "written_by": "tests/golden/make_fullsize_oracle.py --cfg 3"},
    }
    torch.save(blob, out_path)
    print("wrote", out_path, {k: (tuple(v.shape) if hasattr(v, "shape") else v) for k, v in blob.items() if k != "meta"})


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--cfg", type=int, default=3, choices=[3])
    ap.add_argument("--n-tok", type=int, default=2048)
    ap.add_argument("--n-x", type=int, default=24)
    ap.add_argument("--smoke", action="store_true", help="tiny cfg3-like shape, writes to /tmp (checks this script only)")
    ap.add_argument("--out", default=os.path.join(HERE, "cfg3_oracle_rows.pt"))
    args = ap.parse_args()
    if args.smoke:
        run_cfg3("/tmp/cfg3_oracle_rows_smoke.pt", 64, 8, smoke=True)
    else:
        run_cfg3(args.out, args.n_tok, args.n_x)


if __name__ == "__main__":
    main()
