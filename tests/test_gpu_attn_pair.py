"""The CTA-pair attention kernel (attn_pair_kernel, cta_group::2) serves key sequences from 8192 keys; below that the
launcher picks attn_tc_kernel.  (i) Every attention test of test_gpu_kernels.py is run once more in a child process with
DIT_ATTN_PAIR_MIN_K=0, which sends EVERY bf16 head_dim-128 shape (ragged tails, one key, strided buffers, split-KV,
score jumps, empty shards) through the pair kernel; (ii) pair-kernel cases at sizes that take it by default: ragged
key counts, query blocks whose second CTA has no rows, split-KV shards, packed varlen, the panic / two-pass path."""
import os
import subprocess
import sys

import pytest
import torch

from oracle import dit_oracle as O
from paper_2606_13501_b200 import binding as B
from paper_2606_13501_b200 import synth
from util import check, errors

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
TOL = dict(rel=4e-3, maxabs=2.5e-2)


def test_all_attention_tests_through_the_pair_kernel(lib):
    env = dict(os.environ, DIT_ATTN_PAIR_MIN_K="0")
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_gpu_kernels.py"), "-q", "-x", "-k",
                        "attn or split_kv or merge", "-p", "no:cacheprovider"], cwd=ROOT, env=env, capture_output=True, text=True,
                       timeout=900)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-2000:]
    assert " passed" in r.stdout


@pytest.mark.parametrize("nq,nk,H", [(256, 8192, 2), (130, 8192 + 37, 3), (700, 8192 + 64, 2), (1, 8192 + 1, 1),
                                     (384, 12345, 2)])
def test_pair_kernel_ragged_shapes_vs_oracle(lib, nq, nk, H):
    q, k, v = synth.make_attention_qkv(11, nq, nk, H, 128, dtype=torch.bfloat16, device=DEV)
    n0 = B.dit_fallback_launches()
    o, lse = B.dit_attn_partial(q, k, v)
    ro, rl = O.attention(q.cpu(), k.cpu(), v.cpu())
    check(o, ro, torch.bfloat16, f"pair attention {nq}x{nk}", **TOL)
    assert float((lse.double().cpu() - rl).abs().max()) < 2e-2
    assert B.dit_fallback_launches() == n0


def test_pair_kernel_split_kv_and_panic_path(lib):
    """P = 2 shards of 16500 keys (8250 each: the pair kernel, ragged) merge to the unsplit result; a key 12 x a query row
    deep in the sequence makes that row's pair run the row-max pass and the second P / PV pass (R33)."""
    nq, nk, H = 300, 16500, 2
    q, k, v = synth.make_attention_qkv(11, nq, nk, H, 128, dtype=torch.bfloat16, device=DEV)
    k[9000] = (12.0 * q[5].float()).to(torch.bfloat16)
    o, lse = B.dit_attn_partial(q, k, v)
    torch.cuda.synchronize()
    assert torch.isfinite(o.float()).all() and torch.isfinite(lse).all()
    ro, rl = O.attention(q.cpu(), k.cpu(), v.cpu())
    assert errors(o, ro)[0] <= 4e-3
    assert float((lse.double().cpu() - rl).abs().max()) < 5e-2
    assert float((o[5].float().cpu() - v[9000].float().cpu()).abs().max()) < 2e-2       # row 5 sees only that key
    o2, lse2 = B.dit_attn_partial(q, k, v)
    assert torch.equal(o, o2) and torch.equal(lse, lse2)                                 # deterministic
    half = nk // 2
    parts = [B.dit_attn_partial(q, k[a:b], v[a:b]) for a, b in ((0, half), (half, nk))]
    om, lm = B.dit_attn_merge([x[0] for x in parts], [x[1] for x in parts])
    torch.cuda.synchronize()
    assert errors(om, ro)[0] <= 5e-3 and float((lm.double().cpu() - rl).abs().max()) < 5e-2
