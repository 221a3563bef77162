"""nbv_exclusive_scan_noalloc -- the one entry point that allocates nothing (scratch in a static device array inside the
library, include/nbv.h) -- against the existing path: the offsets nbv_tile_lists returns are the exclusive scan of the per-tile
list lengths, computed by the library's own scan (csrc/sort.cu: exclusive_scan_u32) with block sums in a buffer the context
allocates.  At 4112 x 4096 an image has 257 x 256 = 65,792 tiles: more than the one-cluster scan takes, so the existing path
runs its reduce / scan-of-sums / downsweep form with scratch, the form the new call is the variant of.  Integer work: bit-exact.

This file sorts last on purpose (pytest -x: a failure here hides nothing after it); it passes alone in a
fresh process and after the other tests (it shares no state with them beyond the loaded library)."""
import ctypes as C
import gc

import numpy as np
import pytest

from paper_2602_08266_b200 import synth

pytestmark = pytest.mark.gpu

W, H = 4112, 4096          # 257 x 256 tiles: 33 scan blocks of 2,048 with a ragged tail of 256


def _existing_path_offsets(nbv, cam):
    """(counts as uint32 bits in an int32 CUDA tensor, offsets int64 numpy) of one view from nbv_tile_lists"""
    import torch
    off, _ = nbv.tile_lists(cam)
    counts = (off[1:] - off[:-1]).to(torch.int32).contiguous()
    return counts, off.cpu().numpy()


def test_noalloc_scan_matches_the_existing_path_on_two_calls_in_a_row():
    import torch
    from paper_2602_08266_b200 import api
    wl = synth.make_workload(0)
    nbv = api.NBV()
    nbv.load_scene(wl.scene)
    cams = synth.hemisphere_cameras(2, (0.5, 0.7), W, H, 3300.0, 3300.0, np.random.default_rng(21))
    small = synth.hemisphere_cameras(1, (0.6, 0.6), 2576, 1680, 2200.0, 2200.0, np.random.default_rng(13))[0]
    ref = [_existing_path_offsets(nbv, c) for c in (cams[0], cams[1], small)]
    assert ref[0][0].numel() == 257 * 256 and int(ref[0][1][-1]) > 100_000 and not np.array_equal(ref[0][1], ref[1][1])
    torch.cuda.synchronize()
    outs = [torch.empty_like(r[0]) for r in ref]
    tots = [torch.empty(1, dtype=torch.int32, device="cuda") for _ in ref]
    # nothing may be allocated between here and the end of the three calls: neither by the binding (torch's allocator) nor by
    # the library (the driver's free memory).  Both may only GROW in between -- Python may collect what earlier tests left --
    # so collect first and compare one-sidedly.
    gc.collect()
    torch.cuda.synchronize()
    launches = api.load_library().nbv_kernel_launches()
    mem, free = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
    # two calls in a row on the same stream, then a shorter one that leaves stale block sums of the earlier calls in the array
    for (counts, _), out, tot in zip(ref, outs, tots):
        api.exclusive_scan_noalloc(counts, out=out, total=tot)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() <= mem and torch.cuda.mem_get_info()[0] >= free
    assert api.load_library().nbv_kernel_launches() - launches == 9   # three launches per call, all of them this file's kernels
    for (counts, off), out, tot in zip(ref, outs, tots):
        np.testing.assert_array_equal(out.cpu().numpy().view(np.uint32).astype(np.int64), off[:-1])
        assert int(tot.cpu().numpy().view(np.uint32)[0]) == int(off[-1])
    # in place, and again after the other inputs went through the shared array
    buf = ref[0][0].clone()
    api.exclusive_scan_noalloc(buf, out=buf, total=tots[0])
    np.testing.assert_array_equal(buf.cpu().numpy().view(np.uint32).astype(np.int64), ref[0][1][:-1])
    assert int(tots[0].cpu().numpy().view(np.uint32)[0]) == int(ref[0][1][-1])


def test_noalloc_scan_sizes_wraparound_and_limits():
    import torch
    from paper_2602_08266_b200 import api
    lib = api.load_library()
    rng = np.random.default_rng(3)
    for n in (1, 2047, 2048, 2049, 3_000_017):                        # one block; the block boundary; 1,465 blocks + ragged tail
        x = rng.integers(0, 2 ** 32 if n < 3000 else 5000, size=n, dtype=np.uint64).astype(np.uint32)      # small n: sums wrap mod 2^32
        out, tot = api.exclusive_scan_noalloc(torch.from_numpy(x.view(np.int32)).cuda())
        c = np.cumsum(x.astype(np.uint64))
        np.testing.assert_array_equal(out.cpu().numpy().view(np.uint32), (np.concatenate([np.zeros(1, np.uint64), c[:-1]]) & np.uint64(0xffffffff)).astype(np.uint32))
        assert int(tot.cpu().numpy().view(np.uint32)[0]) == int(c[-1] % 2 ** 32)
    # n == 0: only the total is written
    tot = torch.full((1,), 7, dtype=torch.int32, device="cuda")
    assert lib.nbv_exclusive_scan_noalloc(None, None, C.c_int64(0), C.c_void_p(tot.data_ptr()), None) == 0
    assert int(tot.item()) == 0
    # beyond the static array: rejected before anything is launched, with a text that names the limit
    x = torch.zeros(16, dtype=torch.int32, device="cuda")
    launches = lib.nbv_kernel_launches()
    rc = lib.nbv_exclusive_scan_noalloc(C.c_void_p(x.data_ptr()), C.c_void_p(x.data_ptr()), C.c_int64(api.SCAN_NOALLOC_MAX + 1), None, None)
    assert rc == -8 and lib.nbv_kernel_launches() == launches
    msg = lib.nbv_noalloc_last_error().decode()
    assert "NBV_SCAN_NOALLOC_MAX" in msg and str(api.SCAN_NOALLOC_MAX) in msg
    assert lib.nbv_exclusive_scan_noalloc(None, None, C.c_int64(5), None, None) == -1
    assert lib.nbv_exclusive_scan_noalloc(C.c_void_p(x.data_ptr()), C.c_void_p(x.data_ptr()), C.c_int64(-1), None, None) == -1
    # the largest size the array allows
    big = torch.ones(api.SCAN_NOALLOC_MAX, dtype=torch.int32, device="cuda")
    out, tot = api.exclusive_scan_noalloc(big, out=big)
    assert int(tot.item()) == api.SCAN_NOALLOC_MAX
    assert bool((out == torch.arange(api.SCAN_NOALLOC_MAX, dtype=torch.int32, device="cuda")).all())
