"""dit_attn_split_static — the entry point that allocates nothing (partials in a static device array of the library) —
against the existing path (dit_attn_partial on the KV shards + dit_attn_merge with caller tensors), on calls in a row that
share the array.  Collected last on purpose (file name): a failure here must not hide other tests under `pytest -x`."""
import pytest
import torch

from paper_2606_13501_b200 import binding as B
from paper_2606_13501_b200 import synth
from util import check

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _existing_path(q, k, v, P):
    nk = k.shape[0]
    sz = -(-nk // P) if nk else 0                       # R20: contiguous shards of ceil(n_k / P) keys
    parts = [B.dit_attn_partial(q, k[min(p * sz, nk):min((p + 1) * sz, nk)], v[min(p * sz, nk):min((p + 1) * sz, nk)], want_lse=True)
             for p in range(P)]
    return B.dit_attn_merge([o for o, _ in parts], [l for _, l in parts])


def _static_path(q, k, v, P):
    o = torch.empty_like(q)
    lse = torch.empty(q.shape[:2], dtype=torch.float32, device=q.device)
    before = torch.cuda.memory_allocated()
    B.dit_attn_split_static(q, k, v, P, o, lse)
    assert torch.cuda.memory_allocated() == before      # (torch's allocator only; the library itself never allocates)
    torch.cuda.synchronize()
    return o, lse


@pytest.mark.parametrize("dtype,d", [(torch.bfloat16, 128), (torch.float32, 64)])
def test_static_scratch_matches_existing_path_on_calls_in_a_row(lib, dtype, d):
    assert B.dit_static_scratch_bytes() == 8 << 20
    # call 1 fills most of the array; calls 2 and 3 are smaller, with other shard counts, ragged tiles and EMPTY shards
    # (n_k < P): they read nothing of what call 1 left behind
    shapes = [(700, 2500, 4, 4), (300, 130, 4, 3), (129, 5, 2, 8), (700, 2500, 4, 4)]
    if dtype == torch.float32:
        shapes = [(260, 300, 4, 4), (100, 130, 4, 3), (33, 5, 2, 8), (260, 300, 4, 4)]
    for i, (nq, nk, H, P) in enumerate(shapes):
        q, k, v = synth.make_attention_qkv(31 + i, nq, nk, H, d, dtype=dtype, device=DEV)
        o_ref, lse_ref = _existing_path(q, k, v, P)
        o, lse = _static_path(q, k, v, P)
        check(o, o_ref, dtype, f"static-scratch attention, call {i}: o")
        check(lse, lse_ref, torch.float32, f"static-scratch attention, call {i}: lse", rel=1e-5, maxabs=1e-4)


def test_static_scratch_rejects_sizes_beyond_the_array(lib):
    q, k, v = synth.make_attention_qkv(5, 4096, 256, 8, 128, dtype=torch.bfloat16, device=DEV)
    o = torch.empty_like(q)
    # 4 partials of 4096 x 8 x 128 bf16 = 32 MiB + LSEs > 8 MiB
    with pytest.raises(B.DitError, match="static array holds"):
        B.dit_attn_split_static(q, k, v, 4, o)
    # one partial of the same shape (8 MiB + its LSE) is still too large; a quarter of the rows fits
    with pytest.raises(B.DitError):
        B.dit_attn_split_static(q, k, v, 1, o)
    o4 = torch.empty_like(q[:1024])
    B.dit_attn_split_static(q[:1024], k, v, 3, o4)
    o_ref, _ = _existing_path(q[:1024], k, v, 3)
    torch.cuda.synchronize()
    check(o4, o_ref, torch.bfloat16, "static-scratch attention after a rejected call")
    with pytest.raises(B.DitError):
        B.dit_attn_split_static(q[:8], k, v, 9, o[:8])          # split_p outside 1..8
