"""Shared helpers of the GPU parity tests: moving oracle results to the device, packing oracle
outputs into the library's record layout, fragile-pixel bookkeeping and tolerance checks.

Tolerances (BASELINE.json north_star; derivations in DESIGN.md "Tolerances"):
  forward   |got - ref| <= 1e-6 + 1e-5 |ref|                      on every non-fragile pixel; a fragile pixel
            (a skip / stop decision within MARGIN of its threshold) may move by the weight that decision
            carries, 2 cmax flip_w(p), which the oracle computes per pixel;
  gradients |got - ref| <= 1e-5 + 1e-3 |ref| + GRAD_C 2^-24 S     on EVERY element, S = sum of |term| over the
            (pixel, Gaussian) terms behind the element (the oracle accumulates it in fp64 next to the sum): fp32
            atomics reorder a sum whose terms cancel, and that error scales with S, not with the cancelled result.
            Fragile pixels never enter a gradient comparison: their upstream gradient is zeroed on both sides
            (`zero_fragile`), so no Gaussian needs a looser bar.
  integer / index work: bit exact.
Every check returns how many elements needed the third term and the largest multiple of 2^-24 S any element
needed (`c_needed`); the tests print them so they show in the GPU test log.
"""
from types import SimpleNamespace

import numpy as np

FWD_RTOL, FWD_ATOL = 1e-5, 1e-6
GRAD_RTOL, GRAD_ATOL = 1e-3, 1e-5
# a pixel whose walk came within this relative distance of a skip / stop threshold may take the
# other branch on the GPU (exp differs in the last ulps); DESIGN.md "threshold fragility"
MARGIN = 2e-6
# multiples of 2^-24 * S granted to a gradient element on top of the north_star bar.  Each
# term of a per-Gaussian sum is good to ~1e-5 relative on its own (exp 2 ulp, the T_k recurrence ~2 ulp per replayed
# Gaussian, random in sign) -- that is inside the 1e-3 |ref| part; what is NOT is the rounding of the fp32 partial sums
# (16 pixels in registers, then one atomic add per (warp, tile)): n additions of terms with |term| <= S cost at most
# (n - 1) 2^-24 S, ~sqrt(n) 2^-24 S when the signs are random.  Measured on the B200 over the whole suite (1.28e9
# elements at full size): 1.7 at most (profiles/r2_parity.md); 4 grants a little over twice that (round 2 granted 8).
GRAD_C = 4.0
U24 = 2.0 ** -24


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


def colour_max(pre, cam):
    """Largest colour any composited term can carry: max over splat colours and the background."""
    return float(max(np.abs(np.asarray(pre.rgb)).max(initial=0.0), np.abs(np.asarray(cam.bg, np.float64)).max()))


def check_forward(gpu_color, gpu_T, gpu_nc, ofwd, cmax, max_fragile_frac=2e-3):
    """Element-by-element forward comparison; returns a small report dict.

    Non-fragile pixels: north_star's bar on colour and T_final, n_contrib exact.  Fragile pixels (a decision within
    MARGIN of its threshold): one decision may flip; the oracle's flip_w(p) is the compositing weight that then moves
    (alpha T of a Gaussian skipped or kept at alpha ~ 1/255, or the unspent transmittance T at a stop taken or not), so
    colour moves by at most 2 cmax flip_w and T_final by at most flip_w."""
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
    tolT = FWD_ATOL + FWD_RTOL * np.abs(ofwd.T)
    assert not ((dT > tolT) & ok).any(), f"T_final worst {dT[ok].max():.3e}"
    assert np.array_equal(gpu_nc[ok], ofwd.n_contrib[ok]), "n_contrib differs on non-fragile pixels"
    flipped = 0
    if frag:
        fw = ofwd.flip_w.astype(np.float64)[~ok]
        assert (fw > 0).all(), "a fragile pixel must carry a flip weight"
        over = d[~ok] > tol[~ok] + 2.0 * cmax * fw[:, None] * (1 + 1e-3)
        assert not over.any(), f"fragile pixel moved by {d[~ok].max():.3e}, more than the flipped weight allows"
        assert not (dT[~ok] > tolT[~ok] + fw * (1 + 1e-3)).any(), "fragile pixel: T_final moved by more than the flipped weight"
        flipped = int(((d[~ok] > tol[~ok]).any(axis=1)).sum())
    return dict(n=n, fragile=frag, flipped=flipped, worst=float(d[ok].max()) if ok.any() else 0.0,
                worst_rel=float((d / (np.abs(ref) + 1e-1))[ok].max()) if ok.any() else 0.0)


def zero_fragile(g, ofwd, margin=MARGIN):
    """Upstream gradient with the rows of threshold-fragile pixels zeroed (both sides get the same array): a pixel
    whose replay may include / exclude one Gaussian then contributes exactly nothing on either side."""
    g = np.array(g, copy=True)
    frag = ~(ofwd.margin[:, 1] > margin)
    g[frag] = 0
    return g, int(frag.sum())


def drop_pixels(samp, drop):
    """The sampled lists without the pixels flagged in `drop` (bool [n]); tiles left empty are removed."""
    keep = ~np.asarray(drop, bool)
    tpo = samp.tile_pix_offsets.astype(np.int64)
    cnt = np.array([keep[tpo[i]:tpo[i + 1]].sum() for i in range(samp.k)], np.int64)
    live = cnt > 0
    return SimpleNamespace(k=int(live.sum()), n=int(keep.sum()), tiles=samp.tiles[live].copy(),
                           tile_pix_offsets=np.concatenate([[0], np.cumsum(cnt[live])]).astype(np.uint32),
                           pix=samp.pix[keep].copy())


def check_grad(name, got, ref, sum_abs=None, c=GRAD_C, rtol=GRAD_RTOL, atol=GRAD_ATOL):
    """Elementwise gradient comparison on EVERY element:

        |got - ref| <= atol + rtol |ref| + c 2^-24 S

    S = `sum_abs`, the sum of |term| behind the element (same shape as ref once flattened per row; None = no third term).
    Returns {third: elements that needed the third term, c_needed: largest multiple of 2^-24 S any element needed,
    worst_ratio: max |d| / tol}."""
    ref2 = np.asarray(ref, np.float64).reshape(len(ref), -1)
    got2 = np.asarray(got, np.float64).reshape(len(ref), -1)
    assert np.isfinite(got2).all(), f"{name}: non-finite values"
    d = np.abs(got2 - ref2)
    base = atol + rtol * np.abs(ref2)
    if sum_abs is None:
        S = np.zeros_like(d)
    else:
        S = np.asarray(sum_abs, np.float64).reshape(len(ref), -1)
        assert S.shape == d.shape, (name, S.shape, d.shape)
    tol = base + c * U24 * S
    miss = d > tol
    need = d > base
    c_needed = float(((d - base)[need] / np.maximum(U24 * S[need], 1e-300)).max()) if need.any() else 0.0
    assert not miss.any(), (f"{name}: {int(miss.sum())}/{miss.size} elements out of tolerance; worst |d| {d[miss].max():.3e}, "
                            f"needs c = {c_needed:.1f} (granted {c})")
    return dict(third=int(need.sum()), of=int(need.size), c_needed=round(c_needed, 2), worst_ratio=float((d / tol).max()))


RASTER_COLS = dict(mean2D=slice(0, 2), conic=slice(2, 5), opacity=slice(5, 6), rgb=slice(6, 9))


def check_raster_grads(ds, rbwd, label=""):
    """The raster half's [N,12] gradient records against the oracle's four arrays, each element with its own S."""
    rep = {}
    S = rbwd.sum_abs
    rep["mean2D"] = check_grad(label + "dL_dmean2D", ds[:, 0:2], rbwd.dL_dmeans2D, S[:, 0:2])
    rep["conic"] = check_grad(label + "dL_dconic", ds[:, 2:5], rbwd.dL_dconic, S[:, 2:5])
    rep["opacity"] = check_grad(label + "dL_dopacity", ds[:, 5:6], rbwd.dL_dopacity.reshape(-1, 1), S[:, 5:6])
    rep["rgb"] = check_grad(label + "dL_drgb", ds[:, 6:9], rbwd.dL_drgb, S[:, 6:9])
    assert not ds[:, 9:].any(), "gradient record words 9..11 must stay zero"
    return rep


def chain_scale(orc64, cam, sh_degree, means3D, scales, quats, sh, pre, sum_abs, rows=None, grads=None, n_pert=4):
    """S for the projection chain's outputs (O6), two parts, both from the fp64 oracle:

    1. input noise.  The chain is LINEAR in the eight raster gradients it consumes, out_i = sum_j M_ij g_j; a
       perturbation of g_j of size s_j (the raster sum's own S, `sum_abs`) moves out_i by at most sum_j |M_ij| s_j.
       M's columns come from the oracle run on unit inputs (one pass per column).  The three conic columns are
       scaled by kappa = A C / (A C - B^2) >= 1, the condition number of the 2x2 inverse (cov2D -> conic) the chain
       starts from: an fp32 conic carries a relative error of kappa 2^-24 (det = a c - b^2 cancels), and so does
       conic * v for a projected axis v of a needle-shaped splat (project_bwd.cu forms it axis by axis so that the
       loss is kappa and not kappa^2).
    2. conditioning of the rest.  An fp32 evaluation of the chain rounds every intermediate; to first order that is a relative
       perturbation of 2^-24 of its inputs, amplified by the componentwise condition number of out_i (large where
       the chain cancels: an axis of the splat seen end on, a nearly singular 2x2 covariance).  It is measured, not
       guessed: the oracle is re-run on (mu, s, q) with every component multiplied by (1 +- 2^-24), random signs,
       `n_pert` times on the raster gradients `grads` (default: unit-free -- see below), and the largest change of
       out_i, divided by 2^-24, is added to S.  `grads` = (dL_dmean2D, dL_dconic, dL_drgb) the chain is evaluated on.
    rows: optional index array; the bound is then computed for those Gaussians only (others get 0)."""
    N = len(means3D)
    idx = np.arange(N) if rows is None else np.asarray(rows)
    sub = lambda a: np.ascontiguousarray(np.asarray(a)[idx])
    K = (sh_degree + 1) ** 2
    out = dict(dL_dmeans3D=np.zeros((N, 3)), dL_dscales=np.zeros((N, 3)), dL_dquats=np.zeros((N, 4)),
               dL_dsh=np.zeros((N, K, 3)))
    if len(idx) == 0:
        return out
    s9 = np.asarray(sum_abs, np.float64)[idx]
    mu, sc, qt, shc = (sub(a).astype(np.float64) for a in (means3D, scales, quats, sh))
    rad, clp = sub(pre.radii), sub(pre.clamped)
    A, B, C = (np.asarray(pre.conic_opacity, np.float64)[idx, j] for j in range(3))
    det = A * C - B * B
    kappa = np.where(det > 0, A * C / np.where(det > 0, det, 1.0), 1.0)
    cols = [("m", 0, 0), ("m", 1, 1), ("c", 0, 2), ("c", 1, 3), ("c", 2, 4), ("r", 0, 6), ("r", 1, 7), ("r", 2, 8)]
    for kind, j, col in cols:
        gm, gc, gr = np.zeros((len(idx), 2)), np.zeros((len(idx), 3)), np.zeros((len(idx), 3))
        {"m": gm, "c": gc, "r": gr}[kind][:, j] = 1.0
        o = orc64.project_bwd(cam, sh_degree, mu, sc, qt, shc, rad, clp, gm, gc, gr)
        wgt = s9[:, col] * (kappa if kind == "c" else 1.0)
        for nm in out:
            a = np.abs(np.asarray(getattr(o, nm), np.float64))
            out[nm][idx] += a * wgt.reshape((-1,) + (1,) * (a.ndim - 1))
    if grads is not None and n_pert > 0:
        gm, gc, gr = (sub(a).astype(np.float64) for a in grads)
        base = orc64.project_bwd(cam, sh_degree, mu, sc, qt, shc, rad, clp, gm, gc, gr)
        rng = np.random.default_rng(12345)
        pert = lambda a: a * (1.0 + U24 * rng.choice([-1.0, 1.0], size=a.shape))
        worst = {nm: np.zeros_like(np.asarray(getattr(base, nm), np.float64)) for nm in out}
        for _ in range(n_pert):
            o = orc64.project_bwd(cam, sh_degree, pert(mu), pert(sc), pert(qt), shc, rad, clp, gm, gc, gr)
            for nm in out:
                np.maximum(worst[nm], np.abs(np.asarray(getattr(o, nm), np.float64) - getattr(base, nm)), out=worst[nm])
        for nm in out:
            out[nm][idx] += worst[nm] / U24
    return out


def check_chain_grads(bw, pbwd, rbwd, scale, label=""):
    """Projection-chain outputs (GPU namespace with torch tensors) against the oracle's, elementwise, with the
    propagated S of `chain_scale`; dL_dopacities passes through the chain unchanged."""
    rep = {}
    for nm in ("dL_dmeans3D", "dL_dscales", "dL_dquats", "dL_dsh"):
        rep[nm[3:]] = check_grad(label + nm, getattr(bw, nm).cpu().numpy(), getattr(pbwd, nm), scale[nm])
    rep["opacities"] = check_grad(label + "dL_dopacities", bw.dL_dopacities.cpu().numpy().reshape(-1, 1),
                                  rbwd.dL_dopacity.reshape(-1, 1), rbwd.sum_abs[:, 5:6])
    return rep
