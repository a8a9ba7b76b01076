"""tgs_sample_static: the sampling call for hosts that cannot allocate GPU memory (include/tgs.h).

A program that embeds libtgs is sometimes given its buffers and nothing else -- a plug-in inside an application that
budgets HBM itself, a loop that cannot pay for cudaMalloc's device-wide synchronisation, a process whose framework
allocator already holds all of HBM.  For those, tgs_sample_static keeps the scratch that tgs_sample takes as a
workspace in a fixed 640 KiB array inside the library (limit: 16384 tiles), and needs no context.

What is checked: its outputs are bit-identical to tgs_sample's (integer work: the bar is equality, as in
test_sample_parity) on two calls made one after the other that share the one scratch array -- the second on a
smaller image with another mode, so that anything the first call left in the scratch would show --, then the first
again; that an image beyond the limit is refused with a clear message and nothing written; and that the library
launched exactly its three kernels per call.

This file sorts last on purpose: `pytest -x` stops at the first failure, so a failure here hides no other test.  It
makes its own context and inputs, so it passes alone in a fresh process as well as after the rest of the suite.
"""
from types import SimpleNamespace

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


def _cam(W, H):
    return workloads.Camera(W, H, 100.0, 100.0, W / 2, H / 2, np.eye(3, dtype=np.float32), np.zeros(3, np.float32))


def _outputs(torch, cam, fill):
    """Caller-owned outputs of one sampling call, pre-filled so that unwritten words are visible."""
    T, dev = cam.num_tiles, torch.device("cuda", 0)
    i32 = dict(dtype=torch.int32, device=dev)
    return SimpleNamespace(tile_score=torch.full((T,), fill, dtype=torch.int64, device=dev), tiles=torch.full((T,), fill, **i32),
                           tile_pix_offsets=torch.full((T + 1,), fill, **i32), pix=torch.full((cam.width * cam.height,), fill, **i32),
                           tile_select=torch.full((T,), fill, **i32), kn_dev=torch.full((2,), fill, **i32), k=None, n=None)


def _same(torch, a, b):
    assert (a.k, a.n) == (b.k, b.n) and a.n > 0
    assert torch.equal(a.kn_dev, b.kn_dev)
    assert torch.equal(a.tile_score, b.tile_score)
    assert torch.equal(a.tiles[:a.k], b.tiles[:b.k])
    assert torch.equal(a.tile_pix_offsets[:a.k + 1], b.tile_pix_offsets[:b.k + 1])
    assert torch.equal(a.pix[:a.n], b.pix[:b.n])
    assert torch.equal(a.tile_select, b.tile_select)


def test_sample_static_equals_sample_on_consecutive_calls():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_15924_b200 as pk
    from paper_2606_15924_b200 import binding

    tgs = pk.TGS(0)  # only the existing path needs a context
    rng = np.random.default_rng(2606)
    # call A: configs[3]'s image (8487 tiles, several blocks of every kernel), Bernoulli pixels, top 40 %
    # call B: a small ragged image, all pixels of the top 70 % -- fewer tiles than A left in the scratch
    cases = [(_cam(1957, 1091), (40, 100), pk.PIXELS_BERNOULLI_ERR, (1, 2), 11),
             (_cam(250, 35), (70, 100), pk.PIXELS_ALL, (1, 1), 12)]
    cases.append(cases[0])
    errs = {}
    for cam, *_ in cases:
        key = (cam.width, cam.height)
        if key not in errs:
            e = workloads.blob_error_map(rng, cam.width, cam.height, 24)
            e[: cam.height // 3, : cam.width // 4] = 0.0  # zero-error tiles: BERNOULLI keeps one pixel each
            errs[key] = torch.from_numpy(e).cuda()
    # the existing path first (its own workspace), then the static calls back to back on one stream
    want = [tgs.sample(cam, pct, mode, rate, seed, err=errs[(cam.width, cam.height)]) for cam, pct, mode, rate, seed in cases]
    outs = [_outputs(torch, cam, fill=-7) for cam, *_ in cases]
    torch.cuda.synchronize()
    before = tgs.launch_count()
    got = [binding.sample_static(0, cam, pct, mode, outs[i], rate, seed, err=errs[(cam.width, cam.height)], sync=False)
           for i, (cam, pct, mode, rate, seed) in enumerate(cases)]
    assert tgs.launch_count() - before == 3 * len(cases)
    torch.cuda.synchronize()
    for g, w in zip(got, want):
        g.n = int(g.kn_dev[1].item())
        assert int(g.kn_dev[0].item()) == g.k
        _same(torch, g, w)
    assert want[0].n != want[1].n and want[0].k > want[1].k

    # residual input (render, target) instead of an error map, synchronous read-back of (k, n)
    cam = _cam(333, 200)
    render = torch.from_numpy(rng.random((200, 333, 3), dtype=np.float32)).cuda()
    target = torch.from_numpy(rng.random((200, 333, 3), dtype=np.float32)).cuda()
    w = tgs.sample(cam, (25, 100), pk.PIXELS_BERNOULLI_ERR, (3, 4), 5, render=render, target=target)
    g = binding.sample_static(0, cam, (25, 100), pk.PIXELS_BERNOULLI_ERR, _outputs(torch, cam, -7), (3, 4), 5,
                              render=render, target=target, sync=True)
    _same(torch, g, w)


def test_sample_static_refuses_images_beyond_its_scratch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_15924_b200 as pk
    from paper_2606_15924_b200 import binding

    ok = _cam(2048, 2048)  # exactly the limit
    assert ok.num_tiles == pk.SAMPLE_STATIC_MAX_TILES
    err = torch.rand((2048, 2048), device="cuda")
    out = binding.sample_static(0, ok, (10, 100), pk.PIXELS_ALL, _outputs(torch, ok, -7), err=err)
    assert out.k == 1638 and out.n == 1638 * 256
    big = _cam(2049, 2048)  # one more column of tiles
    o = _outputs(torch, big, -7)
    err = torch.rand((2048, 2049), device="cuda")
    before = pk.load_library().tgs_launch_count()
    with pytest.raises(pk.TgsError) as ei:
        binding.sample_static(0, big, (10, 100), pk.PIXELS_ALL, o, err=err)
    assert ei.value.code == 2 and "16512 tiles" in str(ei.value) and "16384" in str(ei.value)
    assert pk.load_library().tgs_launch_count() == before
    torch.cuda.synchronize()
    assert bool((o.kn_dev == -7).all()) and bool((o.tiles == -7).all())
