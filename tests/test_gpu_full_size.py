"""GPU parity at BASELINE.json's FULL sizes (configs 3, 4, 5), in the launch configuration bench.py times
(`SparseRasterStep`: sample -> bin_sort restricted to the sampled tiles -> sparse forward -> backward).

Integer work is compared in full (splat words, pair count, CSR ranges, sorted ids, sampled tiles and pixel
lists).  The floating-point kernels are compared on a SAMPLE of sampled tiles the oracle can afford: the
forward on those tiles' pixels, and the backward with an upstream gradient that is non-zero only on those
pixels (every other pixel then contributes exactly zero, so the oracle's backward over the sample is the whole
gradient).  Properties that hold at any size cover the rest: sum over the image of (1 - T_final) against the
statistics forward, zero gradient for Gaussians no sampled tile lists.
"""
from types import SimpleNamespace

import numpy as np
import pytest

import workloads
from helpers import check_forward, check_grad, dev, pack_splats, scene_dev, tainted_gaussians, u32, unpack_splats

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    return t


@pytest.fixture(scope="module")
def tgs(torch):
    import paper_2606_15924_b200 as pk
    return pk.TGS(0)


def _subsample(samp, binned, n_tiles):
    """A spread of sampled tiles including the longest range and a ragged / partial one if there is any."""
    k = samp.k
    seg = np.diff(binned.tile_offsets.astype(np.int64))[samp.tiles]
    npx = np.diff(samp.tile_pix_offsets.astype(np.int64))
    pick = set(np.linspace(0, k - 1, n_tiles - 3).astype(int).tolist())
    pick.add(int(np.argmax(seg)))
    pick.add(int(np.argmin(npx)))
    pick.add(int(np.argmax(npx)))
    its = np.array(sorted(pick))
    off = samp.tile_pix_offsets.astype(np.int64)
    slots = np.concatenate([np.arange(off[i], off[i + 1]) for i in its])
    tpo = np.concatenate([[0], np.cumsum(npx[its])]).astype(np.uint32)
    sub = SimpleNamespace(k=len(its), n=len(slots), tiles=samp.tiles[its].copy(), tile_pix_offsets=tpo,
                          pix=samp.pix[slots].copy())
    return sub, slots


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_full_size_config(cfg, orc32, orc64, tgs, torch):
    import paper_2606_15924_b200 as pk
    sc = workloads.make(cfg)
    cam = sc.cam
    # ---- oracle: projection, sampling, binning restricted to the sampled tiles (all integer outputs in full) ----
    pre = orc32.preprocess(cam, sc.sh_degree, sc.means3D, sc.scales, sc.quats, sc.opacities, sc.sh)
    samp = orc32.sample(cam, sc.tile_pct, sc.pixel_mode, sc.pix_rate, sc.sample_seed, err=sc.err)
    sel = np.zeros(cam.num_tiles, np.uint32)
    sel[samp.tiles] = 1
    binned = orc32.bin_sort(cam, pre, tile_select=sel)
    # ---- GPU: the bench's step ----
    d = scene_dev(sc, torch)
    step = pk.SparseRasterStep(tgs, cam, sc.N, sc.sh_degree, binned.P + 1024)
    fw = step.forward(d.means3D, d.scales, d.quats, d.opacities, d.sh, sc.tile_pct, sc.pixel_mode, sc.pix_rate,
                      sc.sample_seed, err=dev(sc.err, torch))
    P, k, n = step.counts()
    assert (P, k, n) == (binned.P, samp.k, samp.n)
    got = unpack_splats(step.pre.splats.cpu().numpy())
    assert np.array_equal(got.rect, pre.rect) and np.array_equal(got.depths.view(np.uint32), pre.depths.view(np.uint32))
    assert np.array_equal(got.means2D.view(np.uint32), pre.means2D.view(np.uint32))
    assert np.array_equal(u32(step.samp.tiles)[:k], samp.tiles)
    assert np.array_equal(u32(step.samp.tile_pix_offsets)[:k + 1], samp.tile_pix_offsets)
    assert np.array_equal(u32(step.samp.pix)[:n], samp.pix)
    assert np.array_equal(u32(step.binned.tile_offsets), binned.tile_offsets)
    assert np.array_equal(u32(step.binned.gid_sorted)[:P], binned.gid_sorted)
    # ---- forward on a sample of the sampled tiles ----
    sub, slots = _subsample(samp, binned, 28)
    ofw = orc32.raster_fwd(cam, binned, pre, sub)
    col = fw.color[:n].cpu().numpy()
    Tf = fw.T[:n].cpu().numpy()
    nc = u32(fw.n_contrib)[:n]
    rep = check_forward(col[slots], Tf[slots], nc[slots], ofw)
    assert np.isfinite(col).all() and (Tf >= 0).all() and (Tf <= 1).all()
    # ---- backward: upstream gradient on the sample only ----
    g = np.zeros((n, 3), np.float32)
    g[slots] = workloads.dl_dcolor(cfg, sub.n)
    gd = torch.zeros((cam.width * cam.height, 3), device="cuda")
    gd[:n] = dev(g, torch)
    bw = step.backward(gd)
    torch.cuda.synchronize()
    orb = orc32.raster_bwd(cam, binned, pre, sub, ofw, g[slots])
    opb = orc32.project_bwd(cam, sc.sh_degree, sc.means3D, sc.scales, sc.quats, sc.sh, pre.radii, pre.clamped,
                            orb.dL_dmeans2D, orb.dL_dconic, orb.dL_drgb)
    bad = tainted_gaussians(sc.N, binned, sub, ofw)
    ds = bw.dL_dsplats.cpu().numpy()
    check_grad("dL_dmean2D", ds[:, 0:2], orb.dL_dmeans2D, bad)
    check_grad("dL_dconic", ds[:, 2:5], orb.dL_dconic, bad)
    check_grad("dL_drgb", ds[:, 6:9], orb.dL_drgb, bad)
    # projection stage, isolated: the oracle's chain applied to the GPU's OWN raster gradients (no atomics in this
    # stage).  The chain is ill conditioned for small or edge-on splats (the rotation / scale gradient is a
    # cancelling difference of conic terms; 1 element of 9 M misses the plain bar at config 4), so the referee is the
    # fp64 oracle and the bar is conditioning aware: the kernel must meet the plain bar OR be as close to the fp64
    # result as the oracle's own fp32 build is (x8) -- a plain fp32 evaluation cannot do better.
    args_ = (cam, sc.sh_degree, sc.means3D, sc.scales, sc.quats, sc.sh, pre.radii, pre.clamped,
             ds[:, 0:2].copy(), ds[:, 2:5].copy(), ds[:, 6:9].copy())
    opg32, opg64 = orc32.project_bwd(*args_), orc64.project_bwd(*args_)
    for name_ in ("dL_dmeans3D", "dL_dscales", "dL_dquats", "dL_dsh"):
        got_ = getattr(bw, name_).cpu().numpy().astype(np.float64).reshape(sc.N, -1)
        r64 = np.asarray(getattr(opg64, name_), np.float64).reshape(sc.N, -1)
        r32 = np.asarray(getattr(opg32, name_), np.float64).reshape(sc.N, -1)
        e_gpu, e_o32 = np.abs(got_ - r64), np.abs(r32 - r64)
        miss = (e_gpu > 1e-5 + 1e-3 * np.abs(r64)) & (e_gpu > 8 * e_o32 + 1e-7)
        assert not miss.any(), (name_ + " (projection stage)", int(miss.sum()), float(e_gpu[miss].max()))
        assert (e_gpu > 1e-5 + 1e-3 * np.abs(r64)).sum() <= 2 + 1e-5 * e_gpu.size, name_
        # ... and end to end against the oracle's chain on the ORACLE's raster gradients: the 1e-3 differences the
        # atomics' summation order leaves in dL/dconic pass through the same ill-conditioned chain, so end to end the
        # bar is measured against the largest entry of the array
        ref_ = np.asarray(getattr(opb, name_), np.float64).reshape(sc.N, -1)
        d_ = np.abs(got_ - ref_)
        assert d_.max() <= 1e-5 + 1e-3 * np.abs(ref_).max(), (name_, d_.max(), np.abs(ref_).max())
    # Gaussians that no sampled tile lists get exactly nothing
    listed = np.zeros(sc.N, bool)
    listed[binned.gid_sorted] = True
    assert (ds[~listed] == 0).all() and (bw.dL_dmeans3D.cpu().numpy()[~listed] == 0).all()
    # ---- a property of the whole image: the statistics forward walks what the forward walked ----
    st = tgs.raster_stats_sparse(cam, step.pre.splats, step.binned, step.samp, torch.ones(n, device="cuda"),
                                 n_capacity=cam.width * cam.height)
    torch.cuda.synchronize()
    W = st.stats[:, 2].double().sum().item()
    assert np.isclose(W, (1.0 - Tf.astype(np.float64)).sum(), rtol=2e-4)
    print(f"cfg{cfg}: P={P} k={k} n={n} sample tiles={sub.k} pixels={sub.n} forward {rep}")
