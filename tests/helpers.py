"""Shared helpers of the GPU parity tests: moving oracle results to the device, packing oracle
outputs into the library's record layout, fragile-pixel bookkeeping and tolerance checks.

Tolerances (BASELINE.json north_star): forward 1e-5 relative / 1e-6 absolute; gradients 1e-3
relative / 1e-5 absolute; integer / index work bit exact.
"""
from types import SimpleNamespace

import numpy as np

FWD_RTOL, FWD_ATOL = 1e-5, 1e-6
GRAD_RTOL, GRAD_ATOL = 1e-3, 1e-5
# a pixel whose walk came within this relative distance of a skip / stop threshold may take the
# other branch on the GPU (exp differs in the last ulps); DESIGN.md "threshold fragility"
MARGIN = 2e-6


def pack_splats(pre):
    """Oracle preprocess outputs -> [N,12] fp32 records in the layout of include/tgs.h."""
    N = pre.means2D.shape[0]
    s = np.zeros((N, 12), np.float32)
    s[:, 0:2] = pre.means2D
    s[:, 2:5] = pre.conic_opacity[:, 0:3]
    s[:, 5] = pre.conic_opacity[:, 3]
    s[:, 6:9] = pre.rgb
    s[:, 9] = pre.depths
    r = pre.rect.astype(np.uint32)
    su = s.view(np.uint32)
    su[:, 10] = r[:, 0] | (r[:, 2] << 16)
    su[:, 11] = r[:, 1] | (r[:, 3] << 16)
    vis = pre.radii > 0
    s[~vis] = 0
    return s


def unpack_splats(s):
    """[N,12] records (numpy) -> namespace with the oracle's field names."""
    su = s.view(np.uint32)
    rect = np.stack([su[:, 10] & 0xffff, su[:, 11] & 0xffff, su[:, 10] >> 16, su[:, 11] >> 16], 1).astype(np.int32)
    return SimpleNamespace(means2D=s[:, 0:2], conic_opacity=np.concatenate([s[:, 2:5], s[:, 5:6]], 1), rgb=s[:, 6:9],
                           depths=s[:, 9], rect=rect,
                           tiles_touched=((rect[:, 2] - rect[:, 0]) * (rect[:, 3] - rect[:, 1])).astype(np.uint32))


def dev(a, torch, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def scene_dev(sc, torch):
    return SimpleNamespace(means3D=dev(sc.means3D, torch), scales=dev(sc.scales, torch), quats=dev(sc.quats, torch),
                           opacities=dev(sc.opacities, torch), sh=dev(sc.sh, torch))


def binned_dev(b, torch, T):
    return SimpleNamespace(gid_sorted=dev(b.gid_sorted.astype(np.int64), torch, torch.int32) if b.P else
                           torch.zeros(1, dtype=torch.int32, device="cuda"),
                           tile_offsets=dev(b.tile_offsets.astype(np.int64), torch, torch.int32))


def samp_dev(s, torch):
    return SimpleNamespace(k=s.k, n=s.n, tiles=dev(s.tiles.astype(np.int64), torch, torch.int32),
                           tile_pix_offsets=dev(s.tile_pix_offsets.astype(np.int64), torch, torch.int32),
                           pix=dev(s.pix.astype(np.int64), torch, torch.int32))


def u32(t):
    """int32 device tensor -> numpy uint32"""
    return t.cpu().numpy().view(np.uint32)


def check_forward(gpu_color, gpu_T, gpu_nc, ofwd, max_fragile_frac=2e-3):
    """Element-by-element forward comparison; returns a small report dict."""
    ok = ofwd.margin[:, 0] > MARGIN
    n = len(ok)
    frag = int((~ok).sum())
    assert frag <= max(3, max_fragile_frac * n), f"{frag}/{n} fragile pixels"
    ref = ofwd.color.astype(np.float64)
    d = np.abs(gpu_color.astype(np.float64) - ref)
    tol = FWD_ATOL + FWD_RTOL * np.abs(ref)
    bad = (d > tol) & ok[:, None]
    assert not bad.any(), f"{bad.sum()} colour values out of tolerance, worst {d[ok].max():.3e}"
    dT = np.abs(gpu_T.astype(np.float64) - ofwd.T)
    assert not ((dT > FWD_ATOL + FWD_RTOL * np.abs(ofwd.T)) & ok).any(), f"T_final worst {dT[ok].max():.3e}"
    assert np.array_equal(gpu_nc[ok], ofwd.n_contrib[ok]), "n_contrib differs on non-fragile pixels"
    # fragile pixels: one decision may flip; the result moves by at most one Gaussian's contribution
    if frag:
        assert d[~ok].max() < 2e-2, f"fragile pixel moved by {d[~ok].max():.3e}"
    return dict(n=n, fragile=frag, worst=float(d[ok].max()) if ok.any() else 0.0,
                worst_rel=float((d / (np.abs(ref) + 1e-1))[ok].max()) if ok.any() else 0.0)


def tainted_gaussians(N, binned, samp, ofwd, margin=MARGIN):
    """Gaussians whose gradient may legitimately differ because a pixel that reaches them sits on a
    decision threshold (its replay may include / exclude one Gaussian)."""
    bad = np.zeros(N, bool)
    frag = np.nonzero(~(ofwd.margin[:, 1] > margin))[0]
    if len(frag) == 0:
        return bad
    tile_of_pix = np.searchsorted(samp.tile_pix_offsets, frag, side="right") - 1
    for ip, it in zip(frag, tile_of_pix):
        t = int(samp.tiles[it])
        s0 = int(binned.tile_offsets[t])
        bad[binned.gid_sorted[s0:s0 + max(int(ofwd.n_walked[ip]), int(ofwd.n_contrib[ip]))]] = True
    return bad


def check_grad(name, got, ref, tainted=None, rtol=GRAD_RTOL, atol=GRAD_ATOL):
    """Gradient comparison, rows = Gaussians, columns = the components of one parameter block.

    1. Elementwise bar (north_star): |got - ref| <= atol + rtol * |ref|.
    2. An element that misses (1) must be a cancelling sum: it has to pass the same bar measured
       against the largest component of its own block, |got - ref| <= atol + rtol * max_row|ref|
       (fp32 accumulation-order noise scales with the summed terms, not with a result that cancelled),
       and such elements must be rare (<= 2 + 1e-4 of all elements).  Their count is returned.
    3. Rows in `tainted` (a pixel that reaches the Gaussian sits on a decision threshold, so the
       GPU may legitimately have replayed one Gaussian more or less) are held to the loose bound
       atol + rtol * max|ref| over the whole array instead.
    """
    ref2 = np.asarray(ref, np.float64).reshape(len(ref), -1)
    got2 = np.asarray(got, np.float64).reshape(len(ref), -1)
    assert np.isfinite(got2).all(), f"{name}: non-finite values"
    d = np.abs(got2 - ref2)
    tol = atol + rtol * np.abs(ref2)
    viol = d > tol
    taint = np.zeros(len(ref2), bool) if tainted is None else np.asarray(tainted, bool)
    block = np.abs(ref2).max(axis=1, keepdims=True)
    v = viol & ~taint[:, None]
    over = d > atol + rtol * np.broadcast_to(block, d.shape)
    assert not (v & over).any(), (f"{name}: {int((v & over).sum())} elements out of tolerance even against their block "
                                  f"norm; worst abs {d[v & over].max():.3e}")
    assert v.sum() <= 2 + 1e-4 * v.size, f"{name}: {int(v.sum())}/{v.size} elements miss the elementwise bar"
    vt = viol & taint[:, None]
    if vt.any():
        assert d[vt].max() <= atol + rtol * np.abs(ref2).max(), f"{name}: tainted row off by {d[vt].max():.3e}"
    return dict(miss=int(v.sum()), miss_tainted=int(vt.sum()), worst_ratio=float((d / tol)[~taint].max()) if (~taint).any() else 0.0)
