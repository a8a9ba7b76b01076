"""GPU parity: the CUDA path (through the C ABI, via the ctypes binding) against the CPU oracle,
element by element, on the same seeded inputs.  Run on the B200 box with ``-m gpu``.

Bit exact: splat rect / depth / mean2D words, radii, clamp masks, sort keys, sorted ids, per-tile
ranges, tile scores, sampled tiles and pixel lists.  Tolerance: forward 1e-5 rel / 1e-6 abs,
gradients 1e-3 rel / 1e-5 abs (BASELINE.json north_star) plus the summation-order term of
tests/helpers.py on EVERY element; threshold-fragile pixels get a zero upstream gradient on both sides.
"""
from types import SimpleNamespace

import numpy as np
import pytest

import workloads
from helpers import (MARGIN, binned_dev, chain_scale, check_chain_grads, check_forward, check_grad, check_raster_grads,
                     colour_max, dev, drop_pixels, pack_splats, samp_dev, scene_dev, u32, unpack_splats, zero_fragile)

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


def _cfg1_full():
    """configs[0]'s Gaussians and camera under a FULL mask: the config's own top-25 % tiles are the nearly empty ones
    (22 listed Gaussians in total), so this scene carries config 1's raster parity."""
    sc = workloads.make(1)
    sc.tile_pct, sc.err, sc.target, sc.name = (100, 100), np.ones((128, 128), np.float32), None, "cfg1_full"
    return sc


def _scenes():
    return {
        "cfg1": lambda: workloads.make(1),
        "cfg1_full": _cfg1_full,
        "small_rot": lambda: workloads.small_random_scene(7, 3000, 200, 136, sh_degree=3, bg=(0.1, 0.3, 0.2), spread=1.3,
                                                          log_scale=(-2.8, 0.6)),
        "small_d1": lambda: workloads.small_random_scene(8, 2000, 333, 77, sh_degree=1, spread=1.5, log_scale=(-3.0, 0.8)),
        "small_d2": lambda: workloads.small_random_scene(9, 1500, 97, 211, sh_degree=2, bg=(1.0, 1.0, 1.0), spread=1.0,
                                                         log_scale=(-2.5, 0.7)),
        "cfg2": lambda: workloads.make(2),
        # wide, large splats: 311 of the 971 visible Gaussians project beyond the Jacobian clamp (|t_x/t_z| or |t_y/t_z|
        # above 1.3 tan(fov/2)) and still reach into the image; 102 of them receive a gradient (reading R3 / R8)
        "clamp_vis": lambda: workloads.small_random_scene(12, 1500, 200, 136, sh_degree=2, bg=(0.3, 0.2, 0.1), spread=3.4,
                                                          log_scale=(-1.6, 0.6)),
    }


_cache = {}


def oracle_backward(orc32, orc64, sc, r, g):
    """Oracle backward with the upstream gradient zeroed at threshold-fragile pixels, its sum|terms|, and the
    propagated scale of the projection chain (helpers.chain_scale)."""
    r.g, r.n_fragile = zero_fragile(g, r.fwd)
    r.rbwd = orc32.raster_bwd(sc.cam, r.binned, r.pre, r.samp, r.fwd, r.g, want_abs=True)
    # the chain takes no discrete decision of its own (the clamp flags and the cull are inputs): its referee is the
    # fp64 build, evaluated on the fp32 referee's raster gradients
    r.pbwd = orc64.project_bwd(sc.cam, sc.sh_degree, sc.means3D, sc.scales, sc.quats, sc.sh, r.pre.radii,
                               r.pre.clamped, r.rbwd.dL_dmeans2D, r.rbwd.dL_dconic, r.rbwd.dL_drgb)
    r.scale = chain_scale(orc64, sc.cam, sc.sh_degree, sc.means3D, sc.scales, sc.quats, sc.sh, r.pre, r.rbwd.sum_abs,
                          grads=(r.rbwd.dL_dmeans2D, r.rbwd.dL_dconic, r.rbwd.dL_drgb))
    return r


def oracle_run(name, orc32, orc64):
    if name not in _cache:
        sc = _scenes()[name]()
        r = orc32.pipeline(sc, backward=False)
        oracle_backward(orc32, orc64, sc, r, workloads.dl_dcolor(SCENES.index(name), r.samp.n))
        r.sc = sc
        r.cmax = colour_max(r.pre, sc.cam)
        _cache[name] = r
    return _cache[name]


SCENES = ["cfg1", "small_rot", "small_d1", "small_d2", "cfg2", "cfg1_full", "clamp_vis"]


@pytest.mark.parametrize("name", SCENES)
def test_preprocess_parity(name, orc32, orc64, tgs, torch):
    r = oracle_run(name, orc32, orc64)
    sc = r.sc
    d = scene_dev(sc, torch)
    out = tgs.preprocess(sc.cam, sc.sh_degree, d.means3D, d.scales, d.quats, d.opacities, d.sh)
    torch.cuda.synchronize()
    got = out.splats.cpu().numpy()
    want = pack_splats(r.pre)
    gu, wu = got.view(np.uint32), want.view(np.uint32)
    assert np.array_equal(out.radii.cpu().numpy(), r.pre.radii)
    assert np.array_equal(out.clamped.cpu().numpy(), r.pre.clamped)
    for w in (0, 1, 9, 10, 11):  # mean2D, depth, rect: decide integers downstream -> bit exact
        assert np.array_equal(gu[:, w], wu[:, w]), f"word {w}"
    for w in (2, 3, 4, 5):       # conic, opacity: canonical arithmetic makes these bit exact too
        assert np.array_equal(gu[:, w], wu[:, w]), f"word {w}"
    assert np.abs(got[:, 6:9] - want[:, 6:9]).max() <= 1e-6  # rgb
    assert (r.pre.radii > 0).sum() > 0.3 * sc.N


@pytest.mark.parametrize("name", SCENES)
def test_bin_sort_parity(name, orc32, orc64, tgs, torch):
    r = oracle_run(name, orc32, orc64)
    sc = r.sc
    splats = dev(pack_splats(r.pre), torch)  # stage isolated: the oracle's upstream bits
    P = r.binned.P
    out = tgs.bin_sort(sc.cam, splats, P + 17, want_keys=True)
    torch.cuda.synchronize()
    assert out.P == P
    assert np.array_equal(u32(out.tile_offsets), r.binned.tile_offsets)
    assert np.array_equal(u32(out.gid_sorted)[:P], r.binned.gid_sorted)
    assert np.array_equal(out.keys_sorted.cpu().numpy().view(np.uint64)[:P], r.binned.keys_sorted)
    # exact capacity works, one less reports TGS_ERR_CAPACITY with the required size
    out2 = tgs.bin_sort(sc.cam, splats, P)
    assert out2.P == P and np.array_equal(u32(out2.gid_sorted)[:P], r.binned.gid_sorted)
    import paper_2606_15924_b200 as pk
    with pytest.raises(pk.TgsError) as ei:
        tgs.bin_sort(sc.cam, splats, P - 1)
    assert ei.value.code == 2 and str(P) in str(ei.value)
    # restricted to the sampled tiles (tile_select): same lists for those tiles, empty ranges elsewhere
    sel = np.zeros(sc.cam.num_tiles, np.uint32)
    sel[r.samp.tiles] = 1
    rb = orc32.bin_sort(sc.cam, r.pre, tile_select=sel)
    out3 = tgs.bin_sort(sc.cam, splats, rb.P + 5, want_keys=True, tile_select=dev(sel.astype(np.int32), torch))
    assert out3.P == rb.P and (rb.P < P or r.samp.k == sc.cam.num_tiles)
    assert np.array_equal(u32(out3.tile_offsets), rb.tile_offsets)
    assert np.array_equal(u32(out3.gid_sorted)[:rb.P], rb.gid_sorted)
    assert np.array_equal(out3.keys_sorted.cpu().numpy().view(np.uint64)[:rb.P], rb.keys_sorted)


@pytest.mark.parametrize("name", SCENES)
def test_sample_parity(name, orc32, orc64, tgs, torch):
    r = oracle_run(name, orc32, orc64)
    sc = r.sc
    if sc.err is not None:
        out = tgs.sample(sc.cam, sc.tile_pct, sc.pixel_mode, sc.pix_rate, sc.sample_seed, err=dev(sc.err, torch))
    else:
        render = orc32.render_dense(sc.cam, r.binned, r.pre)
        out = tgs.sample(sc.cam, sc.tile_pct, sc.pixel_mode, sc.pix_rate, sc.sample_seed,
                         render=dev(render, torch), target=dev(sc.target, torch))
    torch.cuda.synchronize()
    s = r.samp
    assert (out.k, out.n) == (s.k, s.n)
    assert np.array_equal(out.tile_score.cpu().numpy().view(np.uint64), s.tile_score)
    assert np.array_equal(u32(out.tiles)[:s.k], s.tiles)
    assert np.array_equal(u32(out.tile_pix_offsets)[:s.k + 1], s.tile_pix_offsets)
    assert np.array_equal(u32(out.pix)[:s.n], s.pix)
    sel = np.zeros(sc.cam.num_tiles, np.uint32)
    sel[s.tiles] = 1
    assert np.array_equal(u32(out.tile_select), sel)


@pytest.mark.parametrize("mode,pct,rate", [(0, (100, 100), (1, 1)), (0, (5, 100), (1, 1)), (1, (100, 100), (1, 2)),
                                           (1, (40, 100), (1, 7)), (1, (70, 100), (255, 255)), (0, (0, 100), (1, 1))])
def test_sample_modes(mode, pct, rate, orc32, tgs, torch):
    rng = np.random.default_rng(5)
    for (W, H) in [(1297, 840), (33, 17), (16, 16), (1, 1), (250, 3)]:
        cam = workloads.Camera(W, H, 100.0, 100.0, W / 2, H / 2, np.eye(3, dtype=np.float32), np.zeros(3, np.float32))
        err = workloads.blob_error_map(rng, W, H, 9)
        err[rng.integers(0, H), rng.integers(0, W)] = np.nan
        err[rng.integers(0, H), rng.integers(0, W)] = 1e20
        if W * H > 1000:
            err[:32, :48] = 0.0  # zero-error tiles: BERNOULLI keeps exactly one pixel each
        s = orc32.sample(cam, pct, mode, rate, seed=99, err=err)
        out = tgs.sample(cam, pct, mode, rate, 99, err=dev(err, torch))
        assert (out.k, out.n) == (s.k, s.n)
        assert np.array_equal(out.tile_score.cpu().numpy().view(np.uint64), s.tile_score)
        assert np.array_equal(u32(out.tiles)[:s.k], s.tiles)
        assert np.array_equal(u32(out.tile_pix_offsets)[:s.k + 1], s.tile_pix_offsets)
        assert np.array_equal(u32(out.pix)[:s.n], s.pix)


@pytest.mark.parametrize("name", SCENES)
def test_raster_fwd_parity(name, orc32, orc64, tgs, torch):
    r = oracle_run(name, orc32, orc64)
    sc = r.sc
    splats = dev(pack_splats(r.pre), torch)
    b, s = binned_dev(r.binned, torch, sc.cam.num_tiles), samp_dev(r.samp, torch)
    out = tgs.raster_fwd_sparse(sc.cam, splats, b, s, want_walked=True)
    torch.cuda.synchronize()
    rep = check_forward(out.color.cpu().numpy(), out.T.cpu().numpy(), u32(out.n_contrib), r.fwd, r.cmax)
    ok = r.fwd.margin[:, 0] > MARGIN
    assert np.array_equal(u32(out.n_walked)[ok], r.fwd.n_walked[ok])
    if name != "cfg1":
        assert (r.fwd.n_contrib > 0).mean() > 0.3  # the comparison is about composited pixels, not background
    print(name, rep)


@pytest.mark.parametrize("name", SCENES)
def test_raster_bwd_parity(name, orc32, orc64, tgs, torch):
    r = oracle_run(name, orc32, orc64)
    sc = r.sc
    splats = dev(pack_splats(r.pre), torch)
    b, s = binned_dev(r.binned, torch, sc.cam.num_tiles), samp_dev(r.samp, torch)
    fwd = type("F", (), {})()
    fwd.T = dev(r.fwd.T, torch)
    fwd.n_contrib = dev(r.fwd.n_contrib.astype(np.int64), torch, torch.int32)
    d = scene_dev(sc, torch)
    out = tgs.raster_bwd_sparse(sc.cam, sc.sh_degree, splats, b, s, fwd, dev(r.g, torch), d.means3D, d.scales, d.quats,
                                d.sh, dev(r.pre.radii, torch), dev(r.pre.clamped, torch))
    torch.cuda.synchronize()
    # every element of every row, strict bar + the summation-order term (helpers.check_grad); the upstream gradient
    # is zero at the scene's threshold-fragile pixels on both sides, so no Gaussian is excluded
    rep = check_raster_grads(out.dL_dsplats.cpu().numpy(), r.rbwd)
    rep.update(check_chain_grads(out, r.pbwd, r.rbwd, r.scale))
    if name != "cfg1":
        assert np.abs(r.pbwd.dL_dmeans3D).max() > 1e-3  # a real gradient, not zeros against zeros
    if name == "clamp_vis":  # the clamped branches of preprocess.cu / project_bwd.cu are exercised, with a gradient
        t = sc.means3D.astype(np.float64) @ np.asarray(sc.cam.R, np.float64).T + np.asarray(sc.cam.t, np.float64)
        cl = (np.abs(t[:, 0] / t[:, 2]) > 1.3 * 0.5 * sc.cam.width / sc.cam.fx) | (np.abs(t[:, 1] / t[:, 2]) > 1.3 * 0.5 * sc.cam.height / sc.cam.fy)
        assert (cl & (r.pre.radii > 0) & (np.abs(r.pbwd.dL_dscales).max(axis=1) > 1e-4)).sum() >= 50
    print(name, f"fragile pixels zeroed: {r.n_fragile}", rep)


@pytest.mark.parametrize("name", ["cfg1_full", "small_rot"])
def test_raster_bwd_takes_a_full_tile_listed_in_any_order(name, orc32, orc64, tgs, torch):
    """A caller's own pixel list may give a tile's 256 pixels in any order (tgs.h fixes the order of the TILES, not of
    the pixels inside one).  Per-Gaussian gradients are sums over pixels, so the oracle's result does not change; the
    backward's fast path for full tiles assumes the row-major order tgs_sample writes and must notice when it is absent."""
    r = oracle_run(name, orc32, orc64)
    sc = r.sc
    tpo = r.samp.tile_pix_offsets.astype(np.int64)
    rng = np.random.default_rng(3)
    perm = np.arange(r.samp.n)
    full = 0
    for i in range(r.samp.k):
        if tpo[i + 1] - tpo[i] == 256:
            # reversed, row-swapped and random orders in turn
            sl = perm[tpo[i]:tpo[i + 1]]
            perm[tpo[i]:tpo[i + 1]] = (sl[::-1], sl.reshape(16, 16).T.reshape(-1), rng.permutation(sl))[full % 3]
            full += 1
    assert full >= 3
    splats = dev(pack_splats(r.pre), torch)
    b, s = binned_dev(r.binned, torch, sc.cam.num_tiles), samp_dev(r.samp, torch)
    s.pix = dev(r.samp.pix[perm].astype(np.int64), torch, torch.int32)
    fwd = SimpleNamespace(T=dev(r.fwd.T[perm], torch), n_contrib=dev(r.fwd.n_contrib[perm].astype(np.int64), torch, torch.int32))
    d = scene_dev(sc, torch)
    out = tgs.raster_bwd_sparse(sc.cam, sc.sh_degree, splats, b, s, fwd, dev(np.ascontiguousarray(r.g[perm]), torch),
                                d.means3D, d.scales, d.quats, d.sh, dev(r.pre.radii, torch), dev(r.pre.clamped, torch))
    torch.cuda.synchronize()
    rep = check_raster_grads(out.dL_dsplats.cpu().numpy(), r.rbwd)
    rep.update(check_chain_grads(out, r.pbwd, r.rbwd, r.scale))
    print(name, f"{full} full tiles listed out of order", rep)


@pytest.mark.parametrize("name", ["small_rot", "small_d2", "cfg2", "clamp_vis"])
def test_raster_bwd_sparse_gradients(name, orc32, orc64, tgs, torch):
    """tgs_raster_bwd_sparse with `touched` (tgs.h, sparse gradients): the mask marks exactly the Gaussians with a
    non-zero raster gradient record; their rows equal the dense call's bit for bit where the raster half is
    deterministic... it is not (atomics), so they are held to the oracle with the same bars; the rows of all other
    Gaussians are left unwritten (a canary survives) and are exactly zero in the oracle."""
    r = oracle_run(name, orc32, orc64)
    sc = r.sc
    splats = dev(pack_splats(r.pre), torch)
    b, s = binned_dev(r.binned, torch, sc.cam.num_tiles), samp_dev(r.samp, torch)
    fwd = type("F", (), {})()
    fwd.T = dev(r.fwd.T, torch)
    fwd.n_contrib = dev(r.fwd.n_contrib.astype(np.int64), torch, torch.int32)
    d = scene_dev(sc, torch)
    N, K = sc.N, (sc.sh_degree + 1) ** 2
    CANARY = 12345.5
    f = dict(dtype=torch.float32, device="cuda")
    out = SimpleNamespace(dL_dsplats=torch.empty((N, 12), **f), dL_dmeans3D=torch.full((N, 3), CANARY, **f),
                          dL_dscales=torch.full((N, 3), CANARY, **f), dL_dquats=torch.full((N, 4), CANARY, **f),
                          dL_dopacities=torch.full((N,), CANARY, **f), dL_dsh=torch.full((N, K, 3), CANARY, **f),
                          touched=torch.full((N,), -7, dtype=torch.int32, device="cuda"))
    tgs.raster_bwd_sparse(sc.cam, sc.sh_degree, splats, b, s, fwd, dev(r.g, torch), d.means3D, d.scales, d.quats, d.sh,
                          dev(r.pre.radii, torch), dev(r.pre.clamped, torch), out=out, sparse=True)
    torch.cuda.synchronize()
    touched = out.touched.cpu().numpy()
    assert set(np.unique(touched)) <= {0, 1}
    rec = out.dL_dsplats.cpu().numpy()[:, :9]
    assert np.array_equal(touched == 1, (rec != 0).any(axis=1) & (r.pre.radii > 0))
    on = touched == 1
    assert 0 < on.sum() < N
    # untouched: nothing written, and the oracle's gradient there is exactly zero
    for nm in ("dL_dmeans3D", "dL_dscales", "dL_dquats", "dL_dopacities", "dL_dsh"):
        got = getattr(out, nm).cpu().numpy()
        assert (got[~on] == CANARY).all(), nm + ": a row of an untouched Gaussian was written"
        assert (got[on] != CANARY).all(), nm + ": a row of a touched Gaussian was not written"
        ref = r.rbwd.dL_dopacity if nm == "dL_dopacities" else getattr(r.pbwd, nm)
        assert not np.asarray(ref)[~on].any(), nm + ": the oracle has a gradient where the mask says none"
        getattr(out, nm)[torch.from_numpy(~on).cuda()] = 0.0   # then the dense comparison applies to every row
    rep = check_chain_grads(out, r.pbwd, r.rbwd, r.scale)
    print(name, f"sparse gradients: {int(on.sum())} of {N} Gaussians touched", rep)


def test_raster_bwd_rejects_a_misaligned_sh_gradient(orc32, orc64, tgs, torch):
    """dL_dsh (and sh) are moved with 16-byte accesses: a misaligned slice is an error, not a fault."""
    import paper_2606_15924_b200 as pk
    r = oracle_run("small_d2", orc32, orc64)
    sc = r.sc
    splats = dev(pack_splats(r.pre), torch)
    b, s = binned_dev(r.binned, torch, sc.cam.num_tiles), samp_dev(r.samp, torch)
    fwd = SimpleNamespace(T=dev(r.fwd.T, torch), n_contrib=dev(r.fwd.n_contrib.astype(np.int64), torch, torch.int32))
    d = scene_dev(sc, torch)
    N, K = sc.N, 9
    f = dict(dtype=torch.float32, device="cuda")
    raw = torch.empty(N * K * 3 + 1, **f)
    out = SimpleNamespace(dL_dsplats=torch.empty((N, 12), **f), dL_dmeans3D=torch.empty((N, 3), **f),
                          dL_dscales=torch.empty((N, 3), **f), dL_dquats=torch.empty((N, 4), **f),
                          dL_dopacities=torch.empty((N,), **f), dL_dsh=raw[1:].view(N, K, 3))
    with pytest.raises(pk.TgsError) as e:
        tgs.raster_bwd_sparse(sc.cam, sc.sh_degree, splats, b, s, fwd, dev(r.g, torch), d.means3D, d.scales, d.quats, d.sh,
                              dev(r.pre.radii, torch), dev(r.pre.clamped, torch), out=out)
    assert e.value.code == 1 and "aligned" in str(e.value)


@pytest.mark.parametrize("name", SCENES)
def test_end_to_end_all_gpu(name, orc32, orc64, tgs, torch):
    """preprocess -> bin_sort -> sample -> fwd -> bwd entirely on the GPU, no oracle data in between."""
    import paper_2606_15924_b200 as pk
    r = oracle_run(name, orc32, orc64)
    sc = r.sc
    d = scene_dev(sc, torch)
    step = pk.SparseRasterStep(tgs, sc.cam, sc.N, sc.sh_degree, r.binned.P + 1000, want_walked=True)
    ref = r
    if sc.err is not None:
        kw = dict(err=dev(sc.err, torch))
    else:
        # config 1: the mask comes from the residual of a dense render (full mask) against the target.  The GPU's
        # render differs from the oracle's in the last bits, so the oracle is re-run on the GPU's OWN render: the
        # selection is integer work on those fp32 values and must then agree bit for bit.
        step.forward(d.means3D, d.scales, d.quats, d.opacities, d.sh, (100, 100), 0,
                     err=torch.ones((sc.cam.height, sc.cam.width), device="cuda"))
        P, k, n = step.counts()
        img = torch.zeros((sc.cam.height * sc.cam.width, 3), device="cuda")
        img[step.samp.pix[:n].long()] = step.fwd.color[:n]
        img = img.reshape(sc.cam.height, sc.cam.width, 3).contiguous()
        kw = dict(render=img, target=dev(sc.target, torch))
        ref = SimpleNamespace(pre=r.pre, binned=r.binned, sc=sc, cmax=r.cmax)
        ref.samp = orc32.sample(sc.cam, sc.tile_pct, sc.pixel_mode, sc.pix_rate, sc.sample_seed, render=img.cpu().numpy(),
                                target=sc.target)
        ref.fwd = orc32.raster_fwd(sc.cam, r.binned, r.pre, ref.samp)
        oracle_backward(orc32, orc64, sc, ref, workloads.dl_dcolor(0, ref.samp.n))
    step.forward(d.means3D, d.scales, d.quats, d.opacities, d.sh, sc.tile_pct, sc.pixel_mode, sc.pix_rate,
                 sc.sample_seed, **kw)
    P, k, n = step.counts()
    assert k == ref.samp.k
    # the step bins only the sampled tiles (restrict=True): same ranges for those tiles
    sel = np.zeros(sc.cam.num_tiles, np.uint32)
    sel[ref.samp.tiles] = 1
    rb = orc32.bin_sort(sc.cam, r.pre, tile_select=sel)
    assert P == rb.P
    assert np.array_equal(u32(step.binned.tile_offsets), rb.tile_offsets)
    assert np.array_equal(u32(step.binned.gid_sorted)[:P], rb.gid_sorted)
    assert n == ref.samp.n and np.array_equal(u32(step.samp.pix)[:n], ref.samp.pix)
    assert np.array_equal(u32(step.samp.tiles)[:k], ref.samp.tiles)
    rep = check_forward(step.fwd.color[:n].cpu().numpy(), step.fwd.T[:n].cpu().numpy(),
                        u32(step.fwd.n_contrib)[:n], ref.fwd, ref.cmax)
    g = torch.zeros((sc.cam.height * sc.cam.width, 3), device="cuda")
    g[:n] = dev(ref.g, torch)
    bw = step.backward(g)
    torch.cuda.synchronize()
    rep.update(check_raster_grads(bw.dL_dsplats.cpu().numpy(), ref.rbwd))
    rep.update(check_chain_grads(bw, ref.pbwd, ref.rbwd, ref.scale))
    print(name, rep)


@pytest.mark.parametrize("name", ["small_rot", "cfg2", "clamp_vis"])
def test_end_to_end_in_north_star_call_order(name, orc32, orc64, tgs, torch):
    """SparseRasterStep.forward(restrict=False): preprocess, bin EVERY tile, then sample, forward, backward -- the call
    order BASELINE.json's north_star gives (the default step samples first and bins only the selected tiles).  All on
    the GPU, no oracle data in between; the full binning is held bit for bit against the oracle's unrestricted lists."""
    import paper_2606_15924_b200 as pk
    r = oracle_run(name, orc32, orc64)
    sc = r.sc
    d = scene_dev(sc, torch)
    step = pk.SparseRasterStep(tgs, sc.cam, sc.N, sc.sh_degree, r.binned.P + 1000, want_walked=True)
    step.forward(d.means3D, d.scales, d.quats, d.opacities, d.sh, sc.tile_pct, sc.pixel_mode, sc.pix_rate,
                 sc.sample_seed, err=dev(sc.err, torch), restrict=False)
    P, k, n = step.counts()
    assert (P, k, n) == (r.binned.P, r.samp.k, r.samp.n)
    assert np.array_equal(u32(step.binned.tile_offsets), r.binned.tile_offsets)
    assert np.array_equal(u32(step.binned.gid_sorted)[:P], r.binned.gid_sorted)
    assert np.array_equal(u32(step.samp.tiles)[:k], r.samp.tiles)
    assert np.array_equal(u32(step.samp.tile_pix_offsets)[:k + 1], r.samp.tile_pix_offsets)
    assert np.array_equal(u32(step.samp.pix)[:n], r.samp.pix)
    rep = check_forward(step.fwd.color[:n].cpu().numpy(), step.fwd.T[:n].cpu().numpy(),
                        u32(step.fwd.n_contrib)[:n], r.fwd, r.cmax)
    g = torch.zeros((sc.cam.height * sc.cam.width, 3), device="cuda")
    g[:n] = dev(r.g, torch)
    bw = step.backward(g)
    torch.cuda.synchronize()
    rep.update(check_raster_grads(bw.dL_dsplats.cpu().numpy(), r.rbwd))
    rep.update(check_chain_grads(bw, r.pbwd, r.rbwd, r.scale))
    print(name, "restrict=False", rep)


def test_full_mask_equals_dense_and_empty_gradients(orc32, tgs, torch):
    """north_star: a full mask reproduces dense rendering; zero upstream gradient gives zero gradients."""
    sc = workloads.small_random_scene(21, 4000, 250, 130, sh_degree=3, bg=(0.2, 0.1, 0.4), spread=1.4)
    pre = orc32.preprocess(sc.cam, 3, sc.means3D, sc.scales, sc.quats, sc.opacities, sc.sh)
    b = orc32.bin_sort(sc.cam, pre)
    dense = orc32.render_dense(sc.cam, b, pre).reshape(-1, 3)
    full = orc32.sample(sc.cam, (100, 100), 0, err=np.ones((130, 250), np.float32))
    of = orc32.raster_fwd(sc.cam, b, pre, full)
    splats = dev(pack_splats(pre), torch)
    out = tgs.raster_fwd_sparse(sc.cam, splats, binned_dev(b, torch, sc.cam.num_tiles), samp_dev(full, torch))
    img = np.zeros_like(dense); img[full.pix] = out.color.cpu().numpy()
    ok = np.zeros(len(dense), bool); ok[full.pix] = of.margin[:, 0] > MARGIN
    assert np.abs(img - dense)[ok].max() <= 1e-6 + 1e-5 * np.abs(dense).max()
    fwd = type("F", (), {})(); fwd.T = out.T; fwd.n_contrib = out.n_contrib
    d = scene_dev(sc, torch)
    bw = tgs.raster_bwd_sparse(sc.cam, 3, splats, binned_dev(b, torch, sc.cam.num_tiles), samp_dev(full, torch), fwd,
                               torch.zeros((full.n, 3), device="cuda"), d.means3D, d.scales, d.quats, d.sh,
                               dev(pre.radii, torch), dev(pre.clamped, torch))
    for a in (bw.dL_dsplats, bw.dL_dmeans3D, bw.dL_dscales, bw.dL_dquats, bw.dL_dopacities, bw.dL_dsh):
        assert not a.any().item()


def test_degenerate_inputs(orc32, tgs, torch):
    import paper_2606_15924_b200 as pk
    cam = workloads.Camera(64, 48, 64.0, 64.0, 32.0, 24.0, np.eye(3, dtype=np.float32), np.zeros(3, np.float32))
    # every Gaussian culled (behind the camera): P = 0, all ranges empty, forward = background
    N = 100
    rng = np.random.default_rng(0)
    mu = rng.uniform(-1, 1, (N, 3)).astype(np.float32); mu[:, 2] -= 5
    sc = np.full((N, 3), 0.1, np.float32); q = np.tile(np.array([1, 0, 0, 0], np.float32), (N, 1))
    op = np.full(N, 0.5, np.float32); sh = np.zeros((N, 1, 3), np.float32)
    cam.bg = (0.25, 0.5, 0.75)
    step = pk.SparseRasterStep(tgs, cam, N, 0, 64)
    err = torch.ones((48, 64), device="cuda")
    fw = step.forward(dev(mu, torch), dev(sc, torch), dev(q, torch), dev(op, torch), dev(sh, torch), (100, 100), 0, err=err)
    P, k, n = step.counts()
    assert (P, k, n) == (0, 12, 64 * 48)
    assert not step.pre.splats.any().item() and not step.binned.tile_offsets.any().item()
    assert torch.equal(fw.color[:n], torch.tensor([0.25, 0.5, 0.75], device="cuda").expand(n, 3))
    assert (fw.T[:n] == 1).all().item() and not fw.n_contrib[:n].any().item()
    bw = step.backward(torch.ones((64 * 48, 3), device="cuda"))
    assert not bw.dL_dmeans3D.any().item() and not bw.dL_dsh.any().item()
    # unsupported / invalid arguments fail loudly
    with pytest.raises(pk.TgsError) as ei:
        tgs.preprocess(cam, 4, dev(mu, torch), dev(sc, torch), dev(q, torch), dev(op, torch), dev(sh, torch))
    assert ei.value.code == 4
    with pytest.raises(pk.TgsError):
        tgs.sample(cam, (3, 2), 0, err=err)
    with pytest.raises(pk.TgsError):
        tgs.sample(cam, (1, 2), 0)


def test_sort_stability_with_duplicate_depths(orc32, tgs, torch):
    """Equal depths inside a tile must keep ascending Gaussian id (reading 6)."""
    sc = workloads.small_random_scene(33, 5000, 160, 96, sh_degree=0, spread=1.2, log_scale=(-2.4, 0.5))
    pre = orc32.preprocess(sc.cam, 0, sc.means3D, sc.scales, sc.quats, sc.opacities, sc.sh)
    vis = np.nonzero(pre.radii > 0)[0]
    pre.depths[vis] = np.float32(3.0) + (vis % 5).astype(np.float32)  # only 5 distinct depths
    b = orc32.bin_sort(sc.cam, pre)
    out = tgs.bin_sort(sc.cam, dev(pack_splats(pre), torch), b.P, want_keys=True)
    assert np.array_equal(u32(out.gid_sorted)[:b.P], b.gid_sorted)
    assert np.array_equal(out.keys_sorted.cpu().numpy().view(np.uint64)[:b.P], b.keys_sorted)
    assert np.array_equal(u32(out.tile_offsets), b.tile_offsets)


def _fake_pre(rng, N, gx, gy, rect_fn, depth_fn):
    """Synthetic preprocess output (only rect / depth / radii matter to bin_sort)."""
    from types import SimpleNamespace
    rect = np.zeros((N, 4), np.int32)
    x0, y0, w, h = rect_fn(rng, N)
    rect[:, 0], rect[:, 1] = x0, y0
    rect[:, 2], rect[:, 3] = np.minimum(x0 + w, gx), np.minimum(y0 + h, gy)
    touched = ((rect[:, 2] - rect[:, 0]) * (rect[:, 3] - rect[:, 1])).astype(np.uint32)
    return SimpleNamespace(means2D=np.zeros((N, 2), np.float32), conic_opacity=np.ones((N, 4), np.float32),
                           rgb=np.zeros((N, 3), np.float32), depths=depth_fn(rng, N).astype(np.float32), rect=rect,
                           tiles_touched=touched, radii=(touched > 0).astype(np.int32))


@pytest.mark.parametrize("case", ["huge_segment", "equal_depths", "few_depths", "many_tiles", "wide_rects"])
def test_bin_sort_segment_paths(case, orc32, tgs, torch):
    """Every path of the segment sort: shared-memory small / big blocks, the global ping-pong for
    oversized segments, the tie step and the full-LSD fallback on long tie runs, the global-atomic
    histogram for very large tile grids, warp-cooperative walks of wide rects."""
    rng = np.random.default_rng(11)
    W, H = 128, 96
    uni = lambda lo, hi: (lambda r, n: r.uniform(lo, hi, n))
    if case == "huge_segment":      # one tile with ~45 k pairs, its neighbours 3-24 k
        N = 70000
        rect_fn = lambda r, n: (np.where(r.random(n) < 0.7, 3, r.integers(0, 8, n)), np.where(r.random(n) < 0.8, 2, r.integers(0, 6, n)),
                                r.integers(1, 3, n), r.integers(1, 3, n))
        depth_fn = uni(0.3, 40.0)
    elif case == "equal_depths":    # all depths equal: order is by Gaussian id only
        N = 30000
        rect_fn = lambda r, n: (r.integers(0, 8, n), r.integers(0, 6, n), r.integers(1, 3, n), r.integers(1, 2, n))
        depth_fn = lambda r, n: np.full(n, 2.5)
    elif case == "few_depths":      # 7 distinct depths: tie runs of thousands, in a 20 k segment too
        N = 50000
        rect_fn = lambda r, n: (np.where(r.random(n) < 0.4, 1, r.integers(0, 8, n)), np.where(r.random(n) < 0.5, 1, r.integers(0, 6, n)),
                                r.integers(1, 2, n), r.integers(1, 2, n))
        depth_fn = lambda r, n: 1.0 + r.integers(0, 7, n) * 0.37
    elif case == "many_tiles":      # T = 14124 > 12288: tile histogram in global memory
        W, H, N = 2100, 1700, 40000
        rect_fn = lambda r, n: (r.integers(0, 132, n), r.integers(0, 107, n), r.integers(1, 6, n), r.integers(1, 6, n))
        depth_fn = uni(0.5, 30.0)
    else:                           # wide_rects: splats covering up to the whole grid
        W, H, N = 640, 480, 3000
        rect_fn = lambda r, n: (r.integers(0, 20, n), r.integers(0, 15, n), r.integers(1, 41, n), r.integers(1, 31, n))
        depth_fn = lambda r, n: np.round(r.uniform(1, 3, n), 2)  # with exact ties
    cam = workloads.Camera(W, H, 100.0, 100.0, W / 2, H / 2, np.eye(3, dtype=np.float32), np.zeros(3, np.float32))
    gx, gy = cam.grid
    pre = _fake_pre(rng, N, gx, gy, rect_fn, depth_fn)
    b = orc32.bin_sort(cam, pre)
    splats = dev(pack_splats(pre), torch)
    out = tgs.bin_sort(cam, splats, b.P + 3, want_keys=True)
    assert out.P == b.P
    assert np.array_equal(u32(out.tile_offsets), b.tile_offsets)
    assert np.array_equal(out.keys_sorted.cpu().numpy().view(np.uint64)[:b.P], b.keys_sorted)
    assert np.array_equal(u32(out.gid_sorted)[:b.P], b.gid_sorted)
    seg = np.diff(b.tile_offsets.astype(np.int64))
    if case == "huge_segment":
        assert seg.max() > 8192 and ((seg > 3072) & (seg <= 8192)).any()
    # restricted to a random half of the tiles
    sel = (rng.random(gx * gy) < 0.5).astype(np.uint32)
    rb = orc32.bin_sort(cam, pre, tile_select=sel)
    out = tgs.bin_sort(cam, splats, rb.P, want_keys=True, tile_select=dev(sel.astype(np.int32), torch))
    assert out.P == rb.P
    assert np.array_equal(u32(out.tile_offsets), rb.tile_offsets)
    assert np.array_equal(u32(out.gid_sorted)[:rb.P], rb.gid_sorted)
    assert np.array_equal(out.keys_sorted.cpu().numpy().view(np.uint64)[:rb.P], rb.keys_sorted)


# ---- f1: tgs_loss_sparse against the oracle's O7 (Eq. 9-11, 17-18) ---------------------------
# Tolerance: the kernel sums <= 256 fp32 terms per tile statistic with a fixed
# butterfly, the oracle sums in fp64; a mean / variance is then good to ~ 256 * 2^-24 = 1.5e-5 relative and the
# gradient, a few products and one division of such statistics, to 1e-4 relative of the largest component.
def _check_loss(out, ref, n, k, torch):
    g = out.dL_dcolor[:n].cpu().numpy().astype(np.float64)
    scale = np.abs(ref.dL_dcolor).max()
    assert np.abs(g - ref.dL_dcolor).max() <= 1e-4 * scale, np.abs(g - ref.dL_dcolor).max() / scale
    assert np.allclose(out.pix_err[:n].cpu().numpy(), ref.pix_err, rtol=1e-6, atol=1e-7)
    st = out.tile_stats[:k].cpu().numpy().astype(np.float64)
    assert np.allclose(st[:, 0], ref.tile_stats[:, 0], rtol=2e-5)
    assert np.allclose(st[:, 1], ref.tile_stats[:, 1], rtol=1e-4, atol=1e-5)
    assert np.allclose(st[:, 2], ref.tile_stats[:, 2], rtol=1e-4, atol=1e-6)
    assert np.allclose(out.loss.cpu().numpy(), ref.loss, rtol=1e-4, atol=1e-7)


@pytest.mark.parametrize("name", ["cfg1", "small_d1", "cfg2"])
def test_loss_sparse_parity_on_rendered_colours(name, orc32, orc64, tgs, torch):
    """The loss on the forward's own output (sparse pixel lists of the scene, seeded target image)."""
    r = oracle_run(name, orc32, orc64)
    sc = r.sc
    rng = np.random.default_rng(5)
    target = np.clip(rng.normal(0.5, 0.25, (sc.cam.height, sc.cam.width, 3)), 0, 1).astype(np.float32)
    color = r.fwd.color.astype(np.float32)
    ref = orc64.loss_sparse(sc.cam, r.samp, color, target)
    samp = SimpleNamespace(k=r.samp.k, n=r.samp.n, tile_pix_offsets=dev(r.samp.tile_pix_offsets.astype(np.int32), torch),
                           pix=dev(r.samp.pix.astype(np.int32), torch))
    out = tgs.loss_sparse(sc.cam, samp, dev(color, torch), dev(target, torch))
    torch.cuda.synchronize()
    _check_loss(out, ref, r.samp.n, r.samp.k, torch)


@pytest.mark.parametrize("mode,pct,rate", [(0, (100, 100), (1, 1)), (1, (40, 100), (1, 3)), (1, (100, 100), (1, 200))])
def test_loss_sparse_modes_and_edge_tiles(mode, pct, rate, orc32, orc64, tgs, torch):
    """Ragged image (edge tiles), Bernoulli lists down to one pixel per tile, low-contrast renders (lambda < 1),
    a render equal to the target (zero residual)."""
    W, H = 203, 117
    cam = workloads.Camera(W, H, 100.0, 100.0, W / 2, H / 2, np.eye(3, dtype=np.float32), np.zeros(3, np.float32))
    rng = np.random.default_rng(21)
    s = orc32.sample(cam, pct, mode, rate, 9, err=workloads.blob_error_map(rng, W, H, 6))
    target = rng.random((H, W, 3)).astype(np.float32)
    samp = SimpleNamespace(k=s.k, n=s.n, tile_pix_offsets=dev(s.tile_pix_offsets.astype(np.int32), torch),
                           pix=dev(s.pix.astype(np.int32), torch))
    cases = [rng.random((s.n, 3)).astype(np.float32),
             (0.5 + 0.02 * (rng.random((s.n, 3)) - 0.5)).astype(np.float32),
             target.reshape(-1, 3)[s.pix].copy()]
    lam_inside = False
    for color in cases:
        ref = orc64.loss_sparse(cam, s, color, target)
        out = tgs.loss_sparse(cam, samp, dev(color, torch), dev(target, torch))
        torch.cuda.synchronize()
        _check_loss(out, ref, s.n, s.k, torch)
        lam_inside |= bool((ref.tile_stats[:, 2] < 0.999).any())
    assert lam_inside


def test_loss_sparse_empty_tiles_in_the_list(orc32, orc64, tgs, torch):
    """A list with EMPTY tiles (m = 0), which the library's samplers never produce but the ABI accepts: an empty tile
    contributes nothing (tile_stats = 0, no NaN in loss), also as the last tile (no read past the list); the other
    tiles are unaffected (the oracle skips empty tiles)."""
    W, H = 96, 64
    cam = workloads.Camera(W, H, 100.0, 100.0, W / 2, H / 2, np.eye(3, dtype=np.float32), np.zeros(3, np.float32))
    rng = np.random.default_rng(33)
    s = orc32.sample(cam, (50, 100), 1, (1, 2), 4, err=workloads.blob_error_map(rng, W, H, 4))   # 12 of 24 tiles: k + 2 <= T
    tpo = s.tile_pix_offsets.astype(np.int64)
    # insert an empty tile after the second tile, and one at the end
    tpo2 = np.concatenate([tpo[:3], [tpo[2]], tpo[3:], [tpo[-1]]]).astype(np.uint32)
    s2 = SimpleNamespace(k=s.k + 2, n=s.n, tile_pix_offsets=tpo2, pix=s.pix)
    target = rng.random((H, W, 3)).astype(np.float32)
    color = rng.random((s.n, 3)).astype(np.float32)
    ref = orc64.loss_sparse(cam, s, color, target)          # without the empty tiles
    samp = SimpleNamespace(k=s2.k, n=s2.n, tile_pix_offsets=dev(tpo2.astype(np.int32), torch), pix=dev(s.pix.astype(np.int32), torch))
    out = tgs.loss_sparse(cam, samp, dev(color, torch), dev(target, torch))
    torch.cuda.synchronize()
    ts = out.tile_stats.cpu().numpy()
    assert not ts[2].any() and not ts[-1].any()
    keep = np.ones(s2.k, bool)
    keep[2] = keep[-1] = False
    assert np.isfinite(out.loss.cpu().numpy()).all()
    np.testing.assert_allclose(ts[keep], ref.tile_stats, rtol=2e-4, atol=1e-6)
    np.testing.assert_allclose(out.loss.cpu().numpy(), ref.loss, rtol=1e-4, atol=1e-7)
    g = out.dL_dcolor.cpu().numpy()[:s.n]
    assert np.abs(g - ref.dL_dcolor).max() <= 1e-4 * np.abs(ref.dL_dcolor).max()


def test_loss_feeds_the_backward(orc32, orc64, tgs, torch):
    """End of the chain: forward colours -> tgs_loss_sparse -> tgs_raster_bwd_sparse, all on the GPU.  The loss
    kernel's dL/dcolor is held to the loss test's bar against the oracle's O7; the backward is then compared with the
    oracle's backward of that SAME upstream gradient (rows of threshold-fragile pixels zeroed on both sides)."""
    r = oracle_run("small_rot", orc32, orc64)
    sc = r.sc
    rng = np.random.default_rng(2)
    target = rng.random((sc.cam.height, sc.cam.width, 3)).astype(np.float32)
    ref_l = orc64.loss_sparse(sc.cam, r.samp, r.fwd.color, target)
    import paper_2606_15924_b200 as pk
    d = scene_dev(sc, torch)
    step = pk.SparseRasterStep(tgs, sc.cam, sc.N, sc.sh_degree, r.binned.P + 8)
    fw = step.forward(d.means3D, d.scales, d.quats, d.opacities, d.sh, sc.tile_pct, sc.pixel_mode, sc.pix_rate,
                      sc.sample_seed, err=dev(sc.err, torch))
    P, k, n = step.counts()
    assert (k, n) == (r.samp.k, r.samp.n)
    samp = SimpleNamespace(k=k, n=n, tile_pix_offsets=step.samp.tile_pix_offsets, pix=step.samp.pix)
    lo = tgs.loss_sparse(sc.cam, samp, fw.color, dev(target, torch), n_capacity=sc.cam.width * sc.cam.height)
    g_gpu = lo.dL_dcolor[:n].cpu().numpy()
    ok = r.fwd.margin[:, 0] > MARGIN  # (a fragile pixel's colour, hence its loss gradient, may differ by a flipped Gaussian)
    assert np.abs(g_gpu - ref_l.dL_dcolor)[ok].max() <= 1e-4 * np.abs(ref_l.dL_dcolor).max()
    ref = SimpleNamespace(pre=r.pre, binned=r.binned, samp=r.samp, fwd=r.fwd)
    oracle_backward(orc32, orc64, sc, ref, g_gpu)
    lo.dL_dcolor[:n] = dev(ref.g, torch)  # = g_gpu with the fragile rows zeroed
    bw = step.backward(lo.dL_dcolor)
    torch.cuda.synchronize()
    rep = check_raster_grads(bw.dL_dsplats.cpu().numpy(), ref.rbwd)
    rep.update(check_chain_grads(bw, ref.pbwd, ref.rbwd, ref.scale))
    print("loss -> backward", rep)


# ---- f3: tgs_raster_stats_sparse against the oracle's O8 (Eq. 12) ------------------------------
# Same bar as the gradients (fp32 atomics reorder the per-Gaussian sums): 1e-3 rel / 1e-5 abs with the block rule,
# Gaussians reachable from a threshold-fragile pixel held to the loose bound; expected depth like the forward.
@pytest.mark.parametrize("name", SCENES)
def test_raster_stats_parity(name, orc32, orc64, tgs, torch):
    r = oracle_run(name, orc32, orc64)
    sc = r.sc
    # the statistics are sums of positive terms (no cancellation): the plain 1e-3 / 1e-5 bar on every element.  The
    # threshold-fragile pixels are taken out of the lists on both sides (their walk may differ by one Gaussian).
    samp = drop_pixels(r.samp, ~(r.fwd.margin[:, 0] > MARGIN))
    assert samp.n >= 0.99 * r.samp.n
    fw = orc32.raster_fwd(sc.cam, r.binned, r.pre, samp)
    e = np.random.default_rng(3).random(samp.n).astype(np.float32)
    ref = orc32.raster_stats(sc.cam, r.binned, r.pre, samp, e)
    out = tgs.raster_stats_sparse(sc.cam, dev(pack_splats(r.pre), torch), binned_dev(r.binned, torch, sc.cam.num_tiles),
                                  samp_dev(samp, torch), dev(e, torch))
    torch.cuda.synchronize()
    st = out.stats.cpu().numpy()
    assert (st[:, 3] == 0).all()
    rep = check_grad("stats(E,D,W)", st[:, :3], ref.stats)
    assert ref.stats[:, 2].sum() > 0
    # sum_i W_i = sum_p (1 - T_final): the statistics walk is the forward's walk
    assert np.isclose(st[:, 2].sum(dtype=np.float64), (1.0 - fw.T.astype(np.float64)).sum(), rtol=1e-4)
    d = out.depth[:samp.n].cpu().numpy()
    assert np.allclose(d, ref.depth, rtol=1e-4, atol=1e-5), np.abs(d - ref.depth).max()
    print(name, rep)


def test_raster_stats_partial_tiles_and_empty(orc32, tgs, torch):
    """Bernoulli pixel lists (partial units), error == 1 gives E == W, an empty selection gives zeros."""
    sc = workloads.small_random_scene(23, 2500, 180, 120, sh_degree=0, spread=1.2, log_scale=(-2.6, 0.6))
    pre = orc32.preprocess(sc.cam, 0, sc.means3D, sc.scales, sc.quats, sc.opacities, sc.sh)
    b = orc32.bin_sort(sc.cam, pre)
    s = orc32.sample(sc.cam, (60, 100), 1, (1, 3), 4, err=workloads.blob_error_map(np.random.default_rng(3), 180, 120, 5))
    s = drop_pixels(s, ~(orc32.raster_fwd(sc.cam, b, pre, s).margin[:, 0] > MARGIN))
    ones = np.ones(s.n, np.float32)
    ref = orc32.raster_stats(sc.cam, b, pre, s, ones)
    splats = dev(pack_splats(pre), torch)
    out = tgs.raster_stats_sparse(sc.cam, splats, binned_dev(b, torch, sc.cam.num_tiles), samp_dev(s, torch), dev(ones, torch))
    torch.cuda.synchronize()
    st = out.stats.cpu().numpy()
    check_grad("stats partial", st[:, :3], ref.stats)
    assert np.allclose(st[:, 0], st[:, 2], rtol=1e-5, atol=1e-6)
    # k = 0: nothing sampled
    empty = SimpleNamespace(k=0, n=0, tiles=torch.zeros(1, dtype=torch.int32, device="cuda"),
                            tile_pix_offsets=torch.zeros(1, dtype=torch.int32, device="cuda"),
                            pix=torch.zeros(1, dtype=torch.int32, device="cuda"))
    out0 = tgs.raster_stats_sparse(sc.cam, splats, binned_dev(b, torch, sc.cam.num_tiles), empty, dev(ones[:1], torch))
    torch.cuda.synchronize()
    assert (out0.stats.cpu().numpy() == 0).all()


# ---- f2: tgs_sample_paper / tgs_maps_update against the oracle's O9 (Eq. 3-4, 7-8): bit exact ----
def _maps(rng, W, H, zero_frac=0.0):
    e = (rng.random((H, W)) ** 3 * 4).astype(np.float32)
    e[rng.random((H, W)) < zero_frac] = 0
    E = e.astype(np.float16).view(np.uint16)
    A = rng.integers(0, 40, (H, W)).astype(np.uint16)
    return E, A


@pytest.mark.parametrize("W,H,n_pix,n_hard,n_stable", [(128, 128, 25, 10, 10), (203, 117, 64, 40, 24), (75, 41, 256, 100, 100),
                                                      (980, 545, 25, 12, 8), (64, 48, 1, 0, 0), (333, 77, 85, 85, 0)])
def test_sample_paper_bit_exact(W, H, n_pix, n_hard, n_stable, orc32, tgs, torch):
    cam = workloads.Camera(W, H, 100.0, 100.0, W / 2, H / 2, np.eye(3, dtype=np.float32), np.zeros(3, np.float32))
    rng = np.random.default_rng(W + H)
    E, A = _maps(rng, W, H, zero_frac=0.3)
    ref = orc32.sample_paper(cam, E, A, n_pix, n_hard, n_stable, seed=77)
    Ed, Ad = dev(E.view(np.int16), torch), dev(A.view(np.int16), torch)
    out = tgs.sample_paper(cam, Ed, Ad, n_pix, n_hard, n_stable, seed=77)
    assert (out.k, out.n) == (ref.k, ref.n)
    assert np.array_equal(u32(out.tiles)[:ref.k], ref.tiles)
    assert np.array_equal(u32(out.tile_pix_offsets)[:ref.k + 1], ref.tile_pix_offsets)
    assert np.array_equal(u32(out.pix)[:ref.n], ref.pix)
    # maps: Eq. 3-4 in place
    e = (rng.random(ref.n) * 3).astype(np.float32)
    E2, A2 = orc32.maps_update(cam, E, A, ref.pix, e, 0.2)
    tgs.maps_update(cam, Ed, Ad, out, dev(e, torch), 0.2)
    torch.cuda.synchronize()
    assert np.array_equal(Ed.cpu().numpy().view(np.uint16), E2)
    assert np.array_equal(Ad.cpu().numpy().view(np.uint16), A2)


def test_sample_paper_degenerate_maps(orc32, tgs, torch):
    """All-zero error map (uniform draws), saturated and equal ages (ties by index), NaN / inf / negative errors."""
    W, H = 90, 50
    cam = workloads.Camera(W, H, 100.0, 100.0, W / 2, H / 2, np.eye(3, dtype=np.float32), np.zeros(3, np.float32))
    rng = np.random.default_rng(1)
    cases = []
    cases.append((np.zeros((H, W), np.uint16), np.full((H, W), 65535, np.uint16)))
    e = rng.random((H, W)).astype(np.float32)
    e[::3, ::2] = np.nan; e[1::4, 1::3] = np.inf; e[2::5, :] = -1.0; e[0, 0] = 65504.0
    cases.append((e.astype(np.float16).view(np.uint16), np.zeros((H, W), np.uint16)))
    for E, A in cases:
        ref = orc32.sample_paper(cam, E, A, 40, 15, 15, seed=3)
        out = tgs.sample_paper(cam, dev(E.view(np.int16), torch), dev(A.view(np.int16), torch), 40, 15, 15, seed=3)
        assert out.n == ref.n and np.array_equal(u32(out.pix)[:ref.n], ref.pix)
        Ed, Ad = dev(E.view(np.int16), torch), dev(A.view(np.int16), torch)
        pe = rng.random(ref.n).astype(np.float32)
        E2, A2 = orc32.maps_update(cam, E, A, ref.pix, pe, 0.5)
        tgs.maps_update(cam, Ed, Ad, out, dev(pe, torch), 0.5)
        torch.cuda.synchronize()
        assert np.array_equal(Ad.cpu().numpy().view(np.uint16), A2)
        got, want = Ed.cpu().numpy().view(np.uint16), E2
        nan = lambda b: (b & 0x7c00) == 0x7c00  # NaN payloads may differ; NaN / inf class and everything else must agree
        assert np.array_equal(nan(got), nan(want)) and np.array_equal(got[~nan(got)], want[~nan(want)])


def test_paper_sampler_drives_the_raster(orc32, orc64, tgs, torch):
    """The paper's pixel lists (few pixels in every tile: all units partial) through forward and backward."""
    r = oracle_run("small_rot", orc32, orc64)
    sc = r.sc
    W, H = sc.cam.width, sc.cam.height
    E, A = _maps(np.random.default_rng(8), W, H)
    s = orc32.sample_paper(sc.cam, E, A, 25, 10, 10, seed=4)
    b = orc32.bin_sort(sc.cam, r.pre)
    fw = orc32.raster_fwd(sc.cam, b, r.pre, s)
    g, _ = zero_fragile(workloads.dl_dcolor(3, s.n), fw)
    rb = orc32.raster_bwd(sc.cam, b, r.pre, s, fw, g, want_abs=True)
    splats = dev(pack_splats(r.pre), torch)
    sd = tgs.sample_paper(sc.cam, dev(E.view(np.int16), torch), dev(A.view(np.int16), torch), 25, 10, 10, seed=4)
    assert sd.n == s.n and np.array_equal(u32(sd.pix)[:s.n], s.pix)
    bd = binned_dev(b, torch, sc.cam.num_tiles)
    out = tgs.raster_fwd_sparse(sc.cam, splats, bd, sd)
    torch.cuda.synchronize()
    check_forward(out.color[:s.n].cpu().numpy(), out.T[:s.n].cpu().numpy(), u32(out.n_contrib)[:s.n], fw, r.cmax)
    bw = tgs.raster_bwd_sparse(sc.cam, sc.sh_degree, splats, bd, sd, out, dev(g, torch), project=False)
    torch.cuda.synchronize()
    print("paper lists", check_raster_grads(bw.dL_dsplats.cpu().numpy(), rb))


def test_step_replays_in_a_cuda_graph(orc32, orc64, tgs, torch):
    """The five calls enqueue only (sizes are read on the device), including the fork / join onto the context's
    side stream: a whole step is captured in a CUDA graph and replayed on new inputs, bit-identical lists and the
    same gradients as the eager step."""
    import paper_2606_15924_b200 as pk
    r = oracle_run("small_rot", orc32, orc64)
    sc = r.sc
    d = scene_dev(sc, torch)
    err = dev(sc.err, torch)
    step = pk.SparseRasterStep(tgs, sc.cam, sc.N, sc.sh_degree, r.binned.P + 64)
    g = torch.zeros((sc.cam.width * sc.cam.height, 3), device="cuda")
    g[:r.samp.n] = dev(r.g, torch)

    def run():
        step.forward(d.means3D, d.scales, d.quats, d.opacities, d.sh, sc.tile_pct, sc.pixel_mode, sc.pix_rate,
                     sc.sample_seed, err=err)
        step.backward(g)

    run()  # eager: also sets the kernels' shared-memory attributes before the capture
    torch.cuda.synchronize()
    P, k, n = step.counts()
    eager = {k_: getattr(step.bwd, k_).clone() for k_ in ("dL_dmeans3D", "dL_dscales", "dL_dquats", "dL_dsh")}
    eager_pix = step.samp.pix[:n].clone()
    eager_gid = step.binned.gid_sorted[:P].clone()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        with torch.cuda.graph(graph, stream=s):
            run()
    for t_ in eager:
        getattr(step.bwd, t_).zero_()
    step.samp.pix.zero_()
    step.binned.gid_sorted.zero_()
    graph.replay()
    torch.cuda.synchronize()
    assert step.counts() == (P, k, n)
    assert torch.equal(step.samp.pix[:n], eager_pix) and torch.equal(step.binned.gid_sorted[:P], eager_gid)
    # two runs of the same step differ only by the order of the atomics: twice the summation-order allowance
    for t_, ref in eager.items():
        check_grad(t_ + " (graph vs eager)", getattr(step.bwd, t_).cpu().numpy(), ref.cpu().numpy(), r.scale[t_], c=16.0)
    check_grad("dL_dmeans3D (graph vs oracle)", step.bwd.dL_dmeans3D.cpu().numpy(), r.pbwd.dL_dmeans3D, r.scale["dL_dmeans3D"])
    # replay on changed inputs: move the Gaussians, the graph must follow (nothing was baked in)
    d.means3D.add_(0.01)
    graph.replay()
    torch.cuda.synchronize()
    moved = step.bwd.dL_dmeans3D.clone()
    run()
    torch.cuda.synchronize()
    # (moved scene: the unmoved scene's scale is the right order of magnitude for the same sums)
    check_grad("dL_dmeans3D (graph vs eager, moved)", moved.cpu().numpy(), step.bwd.dL_dmeans3D.cpu().numpy(),
               r.scale["dL_dmeans3D"], c=32.0)
