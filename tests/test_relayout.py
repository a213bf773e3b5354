"""Re-layout of a row-sharded artifact between split degrees P -> P' (§5.3):
the planner (host, C ABI) against a brute-force per-row ownership map, the oracle's relayout against the row map, and
the device kernel against the oracle, bit for bit (byte work)."""
import itertools

import pytest
import torch

from oracle import dit_oracle as O
from paper_2606_13501_b200 import binding as B
from paper_2606_13501_b200 import synth

DEV = "cuda:0"


def _owner(n, P):
    """brute force: row -> (shard, row inside the shard) under R20 (ceil(n / P) rows per shard)."""
    sz = -(-n // P) if n else 1
    return [(i // sz, i % sz) for i in range(n)]


@pytest.mark.parametrize("n", [0, 1, 5, 8, 37, 288, 4095, 4352])
def test_plan_is_the_slice_intersection_brute_force(lib, n):
    for ps, pd in itertools.product((1, 2, 3, 4, 8, 32), repeat=2):
        plan = B.dit_relayout_plan(n, ps, pd)
        src, dst = _owner(n, ps), _owner(n, pd)
        covered = {}
        for sr, dr, s0, d0, cnt in plan:
            assert cnt > 0 and 0 <= sr < ps and 0 <= dr < pd
            for i in range(cnt):
                covered[(dr, d0 + i)] = (sr, s0 + i)
        # every destination row is written exactly once, from the source location that owns the same global row
        assert len(covered) == n == sum(e[4] for e in plan)
        for g in range(n):
            assert covered[dst[g]] == src[g]
        assert len(plan) <= ps + pd - 1 or n == 0
        # entries are maximal: two consecutive entries never continue the same (src, dst) pair
        assert len({(e[0], e[1]) for e in plan}) == len(plan)
    assert B.dit_relayout_plan(10, 2, 2) == [(0, 0, 0, 0, 5), (1, 1, 0, 0, 5)]          # same layout: identity entries
    assert B.dit_relayout_plan(10, 1, 4) == [(0, 0, 0, 0, 3), (0, 1, 3, 0, 3), (0, 2, 6, 0, 3), (0, 3, 9, 0, 1)]
    with pytest.raises(B.DitError):
        B.dit_relayout_plan(10, 0, 2)
    with pytest.raises(B.DitError):
        B.dit_relayout_plan(10, 2, 33)


def test_oracle_relayout_is_the_row_map_and_round_trips():
    for n, ps, pd in ((37, 4, 3), (8, 8, 2), (5, 2, 8), (288, 1, 4)):
        full = torch.arange(n * 3, dtype=torch.float64).reshape(n, 3)
        src = [full[a:b] for a, b in O.shard_bounds(n, ps)]
        dst = O.relayout(src, pd)
        own = _owner(n, pd)
        for g in range(n):
            q, r = own[g]
            assert torch.equal(dst[q][r], full[g])
        back = O.relayout(dst, ps)
        assert all(torch.equal(a, b) for a, b in zip(back, src))


@pytest.mark.gpu
@pytest.mark.parametrize("n,width,dtype", [(4352, 3072, torch.float32), (32760, 5120, torch.bfloat16), (37, 5, torch.bfloat16),
                                           (1000, 7, torch.float32), (3, 64, torch.float32)])
def test_device_relayout_matches_oracle_bit_for_bit(lib, n, width, dtype):
    full = synth.normal(9, "relayout", (n, width), dtype=dtype, device=DEV)
    for ps, pd in ((1, 4), (4, 1), (2, 8), (8, 3), (4, 4), (3, 32)):
        src = [full[a:b].contiguous() for a, b in O.shard_bounds(n, ps)]
        dst = B.dit_relayout(src, pd)
        want = O.relayout([t.cpu() for t in src], pd)
        torch.cuda.synchronize()
        assert len(dst) == pd
        for a, b in zip(dst, want):
            assert a.shape == b.shape and torch.equal(a.cpu(), b)
        back = B.dit_relayout(dst, ps)                       # P -> P' -> P is the identity
        torch.cuda.synchronize()
        assert all(torch.equal(a, b) for a, b in zip(back, src))
