"""Host logic of the fused 3-D level half: the work split (paper_2304_08159_b200/csrc/wl_plan.h through the C-ABI, no GPU).

Every (tile, plane) must be covered exactly once by items with even z0 and even nz >= 2 (the kernel's restriction pairs
planes 2k, 2k+1 inside an item), the reported load must be the largest per-CTA sum of (nz + 9) — an item costs its planes, 6
run-in plane steps and about 3 steps' worth of pipeline fill — and it may never exceed the uniform-chunk split it replaces."""
import numpy as np
import pytest

from paper_2304_08159_b200 import binding as wl, build

TILE = {"float32": (64, 16), "float64": (32, 14)}
ITEM_COST = 9   # WL_PLAN_RUNIN


@pytest.fixture(scope="module", autouse=True)
def _lib():
    build.build_cuda()


def uniform_cost(dims, tile, sms):
    """Round 1's split: nc equal chunks, items dealt round-robin; cost = waves * (planes per item + ITEM_COST)."""
    n = -(-dims[0] // tile[0]) * -(-dims[1] // tile[1])
    half = dims[2] // 2
    return min(-(-n * nc // sms) * (2 * -(-half // nc) + ITEM_COST) for nc in range(1, half + 1))


@pytest.mark.parametrize("dtype", ["float32", "float64"])
@pytest.mark.parametrize("dims", [(512, 512, 512), (256, 256, 256), (128, 128, 128), (64, 64, 64), (32, 32, 32), (16, 16, 16),
                                  (256, 128, 128), (96, 40, 24), (8, 8, 8), (72, 24, 10), (1024, 512, 256)])
@pytest.mark.parametrize("sms", [148, 132, 7])
def test_plan_covers_every_plane_once_and_is_balanced(dims, dtype, sms):
    items, start, load = wl.wl_plan_fused3d(dims, dtype, sms)
    tx, ty = TILE[dtype]
    grid = len(start) - 1
    assert 1 <= grid <= sms and start[0] == 0 and start[-1] == len(items) and np.all(np.diff(start) >= 1)
    assert np.all(items[:, 2] % 2 == 0) and np.all(items[:, 3] % 2 == 0) and np.all(items[:, 3] >= 2)
    assert np.all(items[:, 0] % tx == 0) and np.all(items[:, 1] % ty == 0)
    cover = {}
    for x0, y0, z0, nz in items:
        assert 0 <= x0 < dims[0] and 0 <= y0 < dims[1]
        cover.setdefault((x0, y0), []).append((z0, nz))
    assert len(cover) == -(-dims[0] // tx) * -(-dims[1] // ty)
    for segs in cover.values():
        z = 0
        for z0, nz in sorted(segs):
            assert z0 == z
            z += nz
        assert z == dims[2]
    loads = [int(np.sum(items[start[b]:start[b + 1], 3] + ITEM_COST)) for b in range(grid)]
    assert max(loads) == load
    assert load <= uniform_cost(dims, (tx, ty), sms)
    # never worse than 25 % above perfect balance plus one run-in per item of the busiest CTA (the documented bound is
    # looser than what the search finds: 256^3 on 148 SMs gives 122 against an ideal of 116.7)
    # (only where there is enough work to balance: at least 8 plane pairs per SM)
    ideal = len(cover) * dims[2] / sms
    if ideal >= 16:
        assert load <= 1.25 * ideal + ITEM_COST * int(np.max(np.diff(start))) + 2


def test_plan_256_cubed_fills_the_idle_sms():
    """The case the split was written for: 64 tiles x 2 chunks = 128 CTAs of 128 + 9 became 144 CTAs of <= 118 + 9."""
    items, start, load = wl.wl_plan_fused3d((256, 256, 256), "float32", 148)
    assert len(start) - 1 > 128 and load <= 127


def test_plan_rejects_bad_input():
    lib = wl.load()
    import ctypes
    d = (ctypes.c_int64 * 3)(64, 64, 63)
    assert lib.wl_plan_fused3d(d, 0, 148, 0, None, 0, None, None, None) == wl.WL_EDIMS
    d = (ctypes.c_int64 * 3)(64, 64, 64)
    assert lib.wl_plan_fused3d(d, 5, 148, 0, None, 0, None, None, None) == wl.WL_EINVAL
    assert lib.wl_plan_fused3d(d, 0, 0, 0, None, 0, None, None, None) == wl.WL_EINVAL
    assert lib.wl_plan_fused3d(None, 0, 148, 0, None, 0, None, None, None) == wl.WL_EINVAL
