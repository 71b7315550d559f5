"""inpc_sample_view_static: the sampler for callers that cannot allocate device memory.

Who that is: code that lives inside somebody else's process and memory pool (a renderer plugin, an engine whose
allocator has taken the whole GPU at start-up), or a frame loop in which cudaMalloc's device-wide synchronisation is
not acceptable.  Such a caller cannot provide the workspace inpc_sample_view asks for, so this entry point keeps its
scratch in a fixed 4.25 MiB array inside the library (at most 2^18 leaves) and allocates nothing.

What is checked: the drawn leaves and positions are the SAME BITS as inpc_sample_view's (the sampler's parity bar in
test_gpu_parity.py is bit-exactness; inpc_sample_view itself is compared with the oracle there), on two calls in a
row that share the array -- the first fills all of it (2^18 leaves), the second uses a small corner of it with
other inputs, so anything the second call wrongly took over from the first would show.  Then the limit.

This file is named so that pytest collects it last (-x stops at the first failure; nothing may hide behind this one),
and it makes no assumption about what ran before it: it passes alone in a fresh process, where its first call is the
one that looks up the array's device address, and after the other tests.
"""
import numpy as np
import pytest
import torch

from paper_2403_16862_b200 import raster
from paper_2403_16862_b200.workloads import Camera, make_octree, second_pose

pytestmark = pytest.mark.gpu


def _dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _same_bits(a, b):
    return torch.equal(a.view(torch.int32), b.view(torch.int32))


def test_static_scratch_sampler_matches_the_workspace_sampler_twice_in_a_row():
    max_leaves = raster.inpc_sample_static_max_leaves()
    assert max_leaves == 1 << 18
    cam = Camera(fx=1100.0, fy=1100.0, cx=648.5, cy=420.0, width=1297, height=840)
    calls = [(max_leaves, 1 << 20, 2024, cam),                              # fills the whole array
             (4096, 100_003, 7, cam.with_pose(*second_pose()))]            # then a corner of it: other tree, pose, seed, ragged N
    for call, (n_leaves, N, seed, c) in enumerate(calls):
        centre, level, prob, root = make_octree(n_leaves, seed=21 + n_leaves % 5)
        centre, level, prob = _dev(centre), _dev(level), _dev(prob)
        want_pos, want_leaf, _ = raster.inpc_sample_view(centre, level, prob, root, c, seed=seed, N=N)
        pos = torch.full((N, 3), 123.0, device="cuda")                       # the caller's own output buffers
        leaf = torch.full((N,), -7, dtype=torch.int32, device="cuda")
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        raster.inpc_sample_view_static(centre, level, prob, root, c, seed=seed, N=N, pos=pos, leaf=leaf)
        torch.cuda.synchronize()
        if call > 0:                                                         # (the first call may still load the module)
            assert torch.cuda.mem_get_info()[0] == free_before, "the static-scratch call changed the device's free memory"
        assert int((want_leaf >= 0).sum()) > N // 2, "degenerate test input: hardly any valid sample"
        assert torch.equal(leaf, want_leaf), "drawn leaf indices differ from inpc_sample_view's"
        assert _same_bits(pos, want_pos), "positions differ from inpc_sample_view's"


def test_static_scratch_sampler_rejects_what_does_not_fit():
    cam = Camera(fx=64.0, fy=64.0, cx=32.0, cy=32.0, width=64, height=64)
    n = raster.inpc_sample_static_max_leaves() + 1
    centre = torch.zeros((n, 3), device="cuda"); level = torch.zeros((n,), dtype=torch.int32, device="cuda")
    prob = torch.ones((n,), device="cuda")
    pos = torch.full((16, 3), 5.0, device="cuda"); leaf = torch.full((16,), 9, dtype=torch.int32, device="cuda")
    with pytest.raises(raster.InpcError) as e:
        raster.inpc_sample_view_static(centre, level, prob, 8.0, cam, seed=1, N=16, pos=pos, leaf=leaf)
    assert e.value.status == -6 and "inpc_sample_static_max_leaves" in str(e.value)
    torch.cuda.synchronize()
    assert (pos == 5.0).all() and (leaf == 9).all()                          # nothing was enqueued
    # the other argument checks are inpc_sample_view's
    with pytest.raises(raster.InpcError) as e:
        raster.inpc_sample_view_static(centre[:8], level[:8], prob[:8], -1.0, cam, seed=1, N=16, pos=pos, leaf=leaf)
    assert e.value.status == -1
