"""GPU parity of tgs_lm_solve against oracle/lm.py (numpy fp64), element by element, through the C ABI.

Bars (f4).  LM blocks: the kernel forms the moment sums, J^T J and the Cholesky solve in fp64
from the same fp32 inputs, so Delta, m, v and the applied parameters of the geometry / appearance blocks are the
oracle's values rounded to fp32: 1e-6 relative (a few fp32 ulp).  Adam branch (higher SH coefficients): fp32
arithmetic.  gbar = sum of V fp32 gradients that may cancel, so with u = 2^-24
    |m - ref| <= 1e-6 |ref| + (V + 1) u S_m,   S_m = beta1 |m_old| + (1 - beta1) sum_i |g_i|
    |v - ref| <= 1e-6 |ref| + (2 V + 2) u S_v, S_v = beta2 v_old + (1 - beta2) (sum_i |g_i|)^2
and Delta = -eta m_hat / (sqrt(v_hat) + eps) carries those two errors to first order plus 1e-5 relative of its own
(IEEE fp32 sqrt and division, the two bias-correction factors rounded to fp32).
Masked Gaussians: exactly zero / exactly unchanged.
"""
from types import SimpleNamespace

import numpy as np
import pytest

import workloads
from oracle import lm

pytestmark = pytest.mark.gpu

# scalars of the call are fp32 on the ABI: both sides get the fp32-representable values
B1, B2, EPS, ETA = (float(np.float32(x)) for x in (0.9, 0.999, 1e-8, 1.25e-4))
KEYS = workloads.LM_KEYS


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available(), "GPU tests need a CUDA device"
    return t


@pytest.fixture(scope="module")
def tgs(torch):
    import paper_2606_15924_b200 as pk
    return pk.TGS(0)


def _dev(ps, torch):
    return {k: torch.from_numpy(np.ascontiguousarray(a)).cuda() for k, a in ps.items()}


def _close(got, ref, rtol, what, atol=0.0):
    got = np.asarray(got, np.float64)
    err = np.abs(got - ref)
    bar = atol + rtol * np.abs(ref)
    bad = err > bar
    assert not bad.any(), f"{what}: {bad.sum()} of {bad.size} off, worst {err[bad].max():.3e} vs ref {np.abs(ref[bad]).max():.3e}"
    with np.errstate(divide="ignore", invalid="ignore"):
        rel = np.where(ref != 0, err / np.abs(ref), 0.0)
    return float(rel.max()) if rel.size else 0.0


U = 2.0 ** -24


def _adam_bars(grads, m, v, m_ref, v_ref, d_ref, V, t):
    """Absolute error bars of the Adam branch (sh[:, 1:, :]) for m, v and Delta; see the module docstring."""
    sabs = np.abs(np.asarray(grads["sh"], np.float64)[:, :, 1:, :]).sum(0)
    S_m = B1 * np.abs(np.asarray(m["sh"], np.float64)[:, 1:, :]) + (1 - B1) * sabs
    S_v = B2 * np.asarray(v["sh"], np.float64)[:, 1:, :] + (1 - B2) * sabs ** 2
    Em = 1e-6 * np.abs(m_ref["sh"][:, 1:, :]) + (V + 1) * U * S_m
    Ev = 1e-6 * np.abs(v_ref["sh"][:, 1:, :]) + (2 * V + 2) * U * S_v
    bc1, bc2 = 1 - B1 ** t, 1 - B2 ** t
    mh, vh = m_ref["sh"][:, 1:, :] / bc1, v_ref["sh"][:, 1:, :] / bc2
    den = np.sqrt(vh) + EPS
    with np.errstate(divide="ignore", invalid="ignore"):
        dd_dv = np.where(vh > 0, ETA * np.abs(mh) / (2 * np.sqrt(vh) * den ** 2 * bc2), 0.0)
    Ed = 1e-5 * np.abs(d_ref["sh"][:, 1:, :]) + ETA / (bc1 * den) * Em + dd_dv * Ev + 1e-30
    return Em, Ev, Ed


def _within(got, ref, bar, what):
    err = np.abs(np.asarray(got, np.float64) - ref)
    bad = err > bar
    assert not bad.any(), f"{what}: {bad.sum()} of {bad.size} outside the bar, worst ratio {(err[bad] / bar[bad]).max():.2f}"
    rel = 1e-6 * np.abs(ref) if "delta" not in what else 1e-5 * np.abs(ref)
    return int((err > rel + 1e-37).sum())


def _run(tgs, torch, seed, n, D, V, t, use_mask, with_params, p_update=0.7, warm=True):
    grads, m, v, upd = workloads.lm_state(seed, n, D, views=V, p_update=p_update, warm=warm)
    rng = np.random.default_rng(777 + seed)
    params = {k: rng.standard_normal(m[k].shape).astype(np.float32) for k in KEYS} if with_params else None
    d_ref, m_ref, v_ref, p_ref = lm.lm_solve(grads, m, v, upd if use_mask else None, B1, B2, EPS, ETA, t=t, params=params)
    gd, md, vd = _dev(grads, torch), _dev(m, torch), _dev(v, torch)
    pd = _dev(params, torch) if with_params else None
    ud = torch.from_numpy(upd).cuda() if use_mask else None
    dd = tgs.lm_solve(D, gd, md, vd, update=ud, beta1=B1, beta2=B2, eps=EPS, eta_sh=ETA, t=t, params=pd)
    torch.cuda.synchronize()
    worst = {}
    for k in KEYS:
        got = dd[k].cpu().numpy()
        if k == "sh":
            worst["d_dc"] = _close(got[:, 0, :], d_ref[k][:, 0, :], 1e-6, "delta sh DC", atol=1e-30)
            worst["m_dc"] = _close(md[k].cpu().numpy()[:, 0, :], m_ref[k][:, 0, :], 1e-6, "m sh DC", atol=1e-37)
            worst["v_dc"] = _close(vd[k].cpu().numpy()[:, 0, :], v_ref[k][:, 0, :], 1e-6, "v sh DC", atol=1e-37)
            if got.shape[1] > 1:
                Em, Ev, Ed = _adam_bars(grads, m, v, m_ref, v_ref, d_ref, V, t)
                worst["n_adam_S_term"] = (_within(got[:, 1:, :], d_ref[k][:, 1:, :], Ed, "delta sh (Adam)")
                                          + _within(md[k].cpu().numpy()[:, 1:, :], m_ref[k][:, 1:, :], Em, "m sh (Adam)")
                                          + _within(vd[k].cpu().numpy()[:, 1:, :], v_ref[k][:, 1:, :], Ev, "v sh (Adam)"))
        else:
            worst["d_" + k] = _close(got, d_ref[k], 1e-6, "delta " + k, atol=1e-30)
            worst["m_" + k] = _close(md[k].cpu().numpy(), m_ref[k], 1e-6, "m " + k, atol=1e-37)
            worst["v_" + k] = _close(vd[k].cpu().numpy(), v_ref[k], 1e-6, "v " + k, atol=1e-37)
        if with_params and k == "sh":
            worst["p_dc"] = _close(pd[k].cpu().numpy()[:, 0, :], p_ref[k][:, 0, :], 1e-6, "params sh DC", atol=1e-7)
            if got.shape[1] > 1:   # p + Delta in fp32: half an ulp of p on top of Delta's own bar
                _within(pd[k].cpu().numpy()[:, 1:, :], p_ref[k][:, 1:, :], Ed + U * np.abs(p_ref[k][:, 1:, :]), "params sh (Adam)")
        elif with_params:
            worst["p_" + k] = _close(pd[k].cpu().numpy(), p_ref[k], 1e-6, "params " + k, atol=1e-7)
        if use_mask:
            off = upd == 0
            assert not got[off].any()
            assert np.array_equal(md[k].cpu().numpy()[off], m[k][off]) and np.array_equal(vd[k].cpu().numpy()[off], v[k][off])
            if with_params:
                assert np.array_equal(pd[k].cpu().numpy()[off], params[k][off])
    return worst


@pytest.mark.parametrize("D", [0, 1, 2, 3])
@pytest.mark.parametrize("V", [1, 3, 7])
def test_lm_solve_parity(tgs, torch, D, V):
    # sizes spanning several blocks of 128 and a ragged tail
    w = _run(tgs, torch, 10 * D + V, 1000 + 37 * D, D, V, t=5, use_mask=True, with_params=(V == 3))
    print(f"lm parity D={D} V={V}: Adam elements that needed the S term: {w.get('n_adam_S_term', 0)}; worst relative errors "
          + ", ".join(f"{k} {x:.1e}" for k, x in w.items() if k[0] != "n" and x > 2e-7))


def test_lm_solve_no_mask_first_iteration(tgs, torch):
    """t = 1 from zero moments (cold start): v = (1 - beta2) gbar^2 is tiny, the damping nearly vanishes and the
    systems are at their worst conditioned."""
    _run(tgs, torch, 50, 4099, 3, 2, t=1, use_mask=False, with_params=True, warm=False, p_update=1.0)


def test_lm_solve_large_t_and_sizes(tgs, torch):
    _run(tgs, torch, 51, 1, 3, 1, t=1000, use_mask=False, with_params=False)
    _run(tgs, torch, 52, 127, 3, 4, t=30000, use_mask=True, with_params=True)
    _run(tgs, torch, 53, 129, 1, 10, t=2, use_mask=True, with_params=False, p_update=0.1)


def test_lm_solve_params_only_and_errors(tgs, torch):
    """delta == NULL with params given is allowed (steps 9 and 10 fused); neither is an error; so are V = 0, eps = 0."""
    import paper_2606_15924_b200 as pk
    grads, m, v, upd = workloads.lm_state(60, 300, 3, views=2)
    params = {k: np.ones_like(a) for k, a in m.items()}
    _, _, _, p_ref = lm.lm_solve(grads, m, v, upd, B1, B2, EPS, ETA, t=3, params=params)
    gd, md, vd, pd = _dev(grads, torch), _dev(m, torch), _dev(v, torch), _dev(params, torch)
    out = tgs.lm_solve(3, gd, md, vd, update=torch.from_numpy(upd).cuda(), beta1=B1, beta2=B2, eps=EPS, eta_sh=ETA, t=3,
                       want_delta=False, params=pd)
    assert out is None
    for k in KEYS:   # params ~ 1, Delta ~ 1e-4: the fp32 Adam error is far below an ulp of the parameter
        _close(pd[k].cpu().numpy(), p_ref[k], 1e-6, "params " + k, atol=1e-7)
    with pytest.raises(pk.TgsError):
        tgs.lm_solve(3, gd, md, vd, want_delta=False, params=None)
    with pytest.raises(pk.TgsError):
        tgs.lm_solve(3, gd, md, vd, eps=0.0)
    with pytest.raises(pk.TgsError):
        tgs.lm_solve(3, gd, md, vd, t=0)
    with pytest.raises(pk.TgsError):
        tgs.lm_solve(4, gd, md, vd)


def test_lm_solve_follows_the_backward(tgs, torch):
    """The call as the step uses it: the per-view gradients are the outputs of tgs_raster_bwd_sparse for V views of one
    scene (written into slices of one [V, N, ...] buffer), update = Gaussians visible in any view."""
    import oracle
    V = 2
    scs = [workloads.small_random_scene(7 + i, 1200, 120, 88, sh_degree=3, spread=1.3, log_scale=(-2.8, 0.6)) for i in range(V)]
    sc0 = scs[0]
    N, K = sc0.N, 16
    o = oracle.Oracle("f32")
    g_np = {k: np.zeros((V,) + s, np.float32) for k, s in
            (("means3D", (N, 3)), ("scales", (N, 3)), ("quats", (N, 4)), ("opacities", (N,)), ("sh", (N, K, 3)))}
    vis = np.zeros(N, bool)
    for i, sc in enumerate(scs):
        sc.means3D, sc.scales, sc.quats, sc.opacities, sc.sh = sc0.means3D, sc0.scales, sc0.quats, sc0.opacities, sc0.sh
        r = o.pipeline(sc, backward=False, restrict=True)
        g = workloads.dl_dcolor(i, r.samp.n)
        rb = o.raster_bwd(sc.cam, r.binned, r.pre, r.samp, r.fwd, g)
        pb = o.project_bwd(sc.cam, sc.sh_degree, sc.means3D, sc.scales, sc.quats, sc.sh, r.pre.radii, r.pre.clamped,
                           rb.dL_dmeans2D, rb.dL_dconic, rb.dL_drgb)
        g_np["means3D"][i], g_np["scales"][i], g_np["quats"][i] = pb.dL_dmeans3D, pb.dL_dscales, pb.dL_dquats
        g_np["opacities"][i], g_np["sh"][i] = rb.dL_dopacity, pb.dL_dsh
        vis |= r.pre.radii > 0
    _, m, v, _ = workloads.lm_state(70, N, 3, views=1)
    upd = vis.astype(np.int32)
    d_ref, m_ref, v_ref, _ = lm.lm_solve(g_np, m, v, upd, B1, B2, EPS, ETA, t=4)
    gd, md, vd = _dev(g_np, torch), _dev(m, torch), _dev(v, torch)
    dd = tgs.lm_solve(3, gd, md, vd, update=torch.from_numpy(upd).cuda(), beta1=B1, beta2=B2, eps=EPS, eta_sh=ETA, t=4)
    torch.cuda.synchronize()
    for k in KEYS:
        got = dd[k].cpu().numpy()
        if k == "sh":
            _close(got[:, 0], d_ref[k][:, 0], 1e-6, "delta DC", atol=1e-30)
            Em, Ev, Ed = _adam_bars(g_np, m, v, m_ref, v_ref, d_ref, V, 4)
            _within(got[:, 1:], d_ref[k][:, 1:], Ed, "delta sh (Adam)")
            _within(md[k].cpu().numpy()[:, 1:], m_ref[k][:, 1:], Em, "m sh (Adam)")
            _close(md[k].cpu().numpy()[:, 0], m_ref[k][:, 0], 1e-6, "m DC", atol=1e-37)
        else:
            _close(got, d_ref[k], 1e-6, "delta " + k, atol=1e-30)
            _close(md[k].cpu().numpy(), m_ref[k], 1e-6, "m " + k, atol=1e-37)


def test_lm_solve_full_size_sampled(tgs, torch):
    """N = 1 M Gaussians, degree 3, V = 3 (the launch configuration bench.py times, a third of its N): the whole call on
    the GPU, then the oracle on a seeded sample of 20 000 Gaussians (blocks and the SH sweep are per Gaussian, so a sample
    is a full check of those rows) plus whole-array properties: masked rows untouched, everything finite."""
    N, D, V, t = 1_000_000, 3, 3, 9
    grads, m, v, upd = workloads.lm_state(99, N, D, views=V)
    gd, md, vd = _dev(grads, torch), _dev(m, torch), _dev(v, torch)
    dd = tgs.lm_solve(D, gd, md, vd, update=torch.from_numpy(upd).cuda(), beta1=B1, beta2=B2, eps=EPS, eta_sh=ETA, t=t)
    torch.cuda.synchronize()
    sel = np.sort(np.random.default_rng(5).choice(N, 20_000, replace=False))
    sub = lambda ps, lead=False: {k: np.ascontiguousarray(a[:, sel] if lead else a[sel]) for k, a in ps.items()}
    d_ref, m_ref, v_ref, _ = lm.lm_solve(sub(grads, True), sub(m), sub(v), upd[sel], B1, B2, EPS, ETA, t=t)
    Em, Ev, Ed = _adam_bars(sub(grads, True), sub(m), sub(v), m_ref, v_ref, d_ref, V, t)
    off = upd == 0
    for k in KEYS:
        got, gm, gv = dd[k].cpu().numpy(), md[k].cpu().numpy(), vd[k].cpu().numpy()
        assert np.isfinite(got).all() and np.isfinite(gm).all() and np.isfinite(gv).all()
        assert not got[off].any() and np.array_equal(gm[off], m[k][off]) and np.array_equal(gv[off], v[k][off])
        if k == "sh":
            _close(got[sel][:, 0], d_ref[k][:, 0], 1e-6, "delta DC", atol=1e-30)
            _within(got[sel][:, 1:], d_ref[k][:, 1:], Ed, "delta sh (Adam)")
            _within(gm[sel][:, 1:], m_ref[k][:, 1:], Em, "m sh (Adam)")
            _within(gv[sel][:, 1:], v_ref[k][:, 1:], Ev, "v sh (Adam)")
        else:
            _close(got[sel], d_ref[k], 1e-6, "delta " + k, atol=1e-30)
            _close(gm[sel], m_ref[k], 1e-6, "m " + k, atol=1e-37)
            _close(gv[sel], v_ref[k], 1e-6, "v " + k, atol=1e-37)


@pytest.mark.parametrize("D,V", [(3, 3), (2, 5), (0, 2)])
def test_lm_solve_per_view_masks(tgs, torch, D, V):
    """view_touched [V, N] (tgs.h): rows of a view's gradient are read only where its mask is set -- NaN sits in every
    masked row here, and a Gaussian touched in no view keeps its moments (oracle R36)."""
    n = 2000 + 13 * D
    grads, m, v, _ = workloads.lm_state(80 + D, n, D, views=V, p_update=1.0)
    rng = np.random.default_rng(81)
    vt = (rng.random((V, n)) < 0.5).astype(np.int32)
    vt[:, :7] = 0
    garbage = {k: np.where(vt.reshape(vt.shape + (1,) * (a.ndim - 2)) != 0, a, np.nan).astype(np.float32) for k, a in grads.items()}
    d_ref, m_ref, v_ref, _ = lm.lm_solve(garbage, m, v, None, B1, B2, EPS, ETA, t=6, view_touched=vt)
    zeroed = {k: np.nan_to_num(a, nan=0.0) for k, a in garbage.items()}
    gd, md, vd = _dev(garbage, torch), _dev(m, torch), _dev(v, torch)
    dd = tgs.lm_solve(D, gd, md, vd, view_touched=torch.from_numpy(vt).cuda(), beta1=B1, beta2=B2, eps=EPS, eta_sh=ETA, t=6)
    torch.cuda.synchronize()
    off = ~(vt.any(0))
    assert off[:7].all()
    for k in KEYS:
        got, gm, gv = dd[k].cpu().numpy(), md[k].cpu().numpy(), vd[k].cpu().numpy()
        assert np.isfinite(got).all() and np.isfinite(gm).all() and np.isfinite(gv).all(), k + ": a masked row was read"
        assert not got[off].any() and np.array_equal(gm[off], m[k][off]) and np.array_equal(gv[off], v[k][off])
        if k == "sh":
            _close(got[:, 0], d_ref[k][:, 0], 1e-6, "delta DC", atol=1e-30)
            if got.shape[1] > 1:
                Em, Ev, Ed = _adam_bars(zeroed, m, v, m_ref, v_ref, d_ref, V, 6)
                _within(got[:, 1:], d_ref[k][:, 1:], Ed, "delta sh (Adam)")
                _within(gm[:, 1:], m_ref[k][:, 1:], Em, "m sh (Adam)")
        else:
            _close(got, d_ref[k], 1e-6, "delta " + k, atol=1e-30)
            _close(gm, m_ref[k], 1e-6, "m " + k, atol=1e-37)
            _close(gv, v_ref[k], 1e-6, "v " + k, atol=1e-37)


def test_sparse_iteration_equals_its_calls(tgs, torch):
    """pipeline.SparseIteration (Alg. 1 steps 3-10 for V views: step, loss, sparse backward into view-major slices, one
    tgs_lm_solve with the per-view touched masks) against the same calls made one by one with DENSE gradients and an
    explicit update mask.  Every call has its own oracle parity test; this one holds the plumbing: camera per view,
    slices, masks, in-place parameter update.  (Atomics reorder the gradient sums from run to run: 1e-4.)"""
    import paper_2606_15924_b200 as pk
    from helpers import dev, scene_dev
    V, D = 3, 3
    sc = workloads.small_random_scene(7, 3000, 200, 136, sh_degree=D, bg=(0.1, 0.3, 0.2), spread=1.3, log_scale=(-2.8, 0.6))
    cams = [workloads.orbit_view(sc, i).cam for i in range(V)]
    N, W, H = sc.N, sc.cam.width, sc.cam.height
    rng = np.random.default_rng(17)
    targets = [dev(rng.random((H, W, 3)).astype(np.float32), torch) for _ in range(V)]
    errs = [dev(workloads.blob_error_map(rng, W, H, 6), torch) for _ in range(V)]
    _, m_np, v_np, _ = workloads.lm_state(71, N, D, views=1)
    d = scene_dev(sc, torch)
    base = {"means3D": d.means3D, "scales": d.scales, "quats": d.quats, "opacities": d.opacities, "sh": d.sh}
    clone = lambda ps: {k: a.clone() for k, a in ps.items()}
    P_cap = 200_000

    it = pk.SparseIteration(tgs, cams, N, D, P_cap)
    p1, m1, v1 = clone(base), _dev(m_np, torch), _dev(v_np, torch)
    it.run(p1, targets, errs, m1, v1, t=3, tile_pct=(50, 100), pixel_mode=pk.PIXELS_ALL, seed=5, apply=True)
    torch.cuda.synchronize()
    touched = it.touched.cpu().numpy()
    assert set(np.unique(touched)) <= {0, 1} and 0 < touched.sum() < touched.size

    # the same iteration, call by call, dense gradients
    step = pk.SparseRasterStep(tgs, cams[0], N, D, P_cap)
    K = (D + 1) ** 2
    G = {"means3D": torch.zeros((V, N, 3), device="cuda"), "scales": torch.zeros((V, N, 3), device="cuda"),
         "quats": torch.zeros((V, N, 4), device="cuda"), "opacities": torch.zeros((V, N), device="cuda"),
         "sh": torch.zeros((V, N, K, 3), device="cuda")}
    for i, cam in enumerate(cams):
        fw = step.forward(base["means3D"], base["scales"], base["quats"], base["opacities"], base["sh"], (50, 100),
                          pk.PIXELS_ALL, (1, 1), 5 + i, err=errs[i], cam=cam)
        samp = SimpleNamespace(k=step.samp.k, n=None, tile_pix_offsets=step.samp.tile_pix_offsets, pix=step.samp.pix)
        lo = tgs.loss_sparse(cam, samp, fw.color, targets[i])
        bw = step.backward(lo.dL_dcolor)
        G["means3D"][i], G["scales"][i], G["quats"][i] = bw.dL_dmeans3D, bw.dL_dscales, bw.dL_dquats
        G["opacities"][i], G["sh"][i] = bw.dL_dopacities, bw.dL_dsh
        rec = bw.dL_dsplats.cpu().numpy()[:, :9]
        assert np.array_equal(touched[i] == 1, (rec != 0).any(axis=1)), "touched mask of view %d" % i
    p2, m2, v2 = clone(base), _dev(m_np, torch), _dev(v_np, torch)
    upd = torch.from_numpy(touched.any(0).astype(np.int32)).cuda()
    tgs.lm_solve(D, G, m2, v2, update=upd, t=3, want_delta=False, params=p2)
    torch.cuda.synchronize()
    moved = 0
    for k in KEYS:
        a, b, b0 = p1[k].cpu().numpy().astype(np.float64), p2[k].cpu().numpy().astype(np.float64), base[k].cpu().numpy()
        step_size = np.abs(b - b0)
        assert np.abs(a - b).max() <= 1e-4 * step_size.max() + 1e-7, (k, np.abs(a - b).max(), step_size.max())
        assert np.array_equal(a[upd.cpu().numpy() == 0], b0[upd.cpu().numpy() == 0])     # untouched Gaussians do not move
        np.testing.assert_allclose(m1[k].cpu().numpy(), m2[k].cpu().numpy(), rtol=1e-3, atol=1e-9)
        moved += int((step_size > 0).sum())
    assert moved > 1000


def test_paper_iteration_equals_its_calls_and_replays_in_a_graph(tgs, torch):
    """SparseIteration.run_paper (the paper's sampler from persistent maps, all tiles binned, loss, map update, sparse
    backward, LM solve) against the same calls made one by one with dense gradients; the maps are integer work and must
    agree bit for bit.  Then the whole iteration captured in ONE CUDA graph and replayed: nothing in it synchronises."""
    import paper_2606_15924_b200 as pk
    from helpers import dev, scene_dev
    V, D = 2, 3
    sc = workloads.small_random_scene(7, 3000, 200, 136, sh_degree=D, bg=(0.1, 0.3, 0.2), spread=1.3, log_scale=(-2.8, 0.6))
    cams = [workloads.orbit_view(sc, i).cam for i in range(V)]
    N, W, H = sc.N, sc.cam.width, sc.cam.height
    rng = np.random.default_rng(23)
    targets = [dev(rng.random((H, W, 3)).astype(np.float32), torch) for _ in range(V)]
    E0 = [(4.0 * rng.random((H, W)) ** 3).astype(np.float16).view(np.int16) for _ in range(V)]
    A0 = [rng.integers(0, 40, (H, W)).astype(np.int16) for _ in range(V)]
    _, m_np, v_np, _ = workloads.lm_state(72, N, D, views=1)
    d = scene_dev(sc, torch)
    base = {"means3D": d.means3D, "scales": d.scales, "quats": d.quats, "opacities": d.opacities, "sh": d.sh}
    clone = lambda ps: {k: a.clone() for k, a in ps.items()}
    P_cap = 400_000
    kw = dict(n_pix=25, n_hard=10, n_stable=8, beta=0.4, seed=9, apply=True)

    it = pk.SparseIteration(tgs, cams, N, D, P_cap)
    p1, m1, v1 = clone(base), _dev(m_np, torch), _dev(v_np, torch)
    E1, A1 = [dev(e, torch) for e in E0], [dev(a, torch) for a in A0]
    it.run_paper(p1, targets, E1, A1, m1, v1, t=2, **kw)
    torch.cuda.synchronize()
    P = int(it.step.binned.P_dev.cpu()[0])
    assert 0 < P <= P_cap and int(it.step.binned.P_dev.cpu()[1]) == 0

    # call by call, dense gradients
    step = pk.SparseRasterStep(tgs, cams[0], N, D, P_cap)
    K = (D + 1) ** 2
    G = {"means3D": torch.zeros((V, N, 3), device="cuda"), "scales": torch.zeros((V, N, 3), device="cuda"),
         "quats": torch.zeros((V, N, 4), device="cuda"), "opacities": torch.zeros((V, N), device="cuda"),
         "sh": torch.zeros((V, N, K, 3), device="cuda")}
    E2, A2 = [dev(e, torch) for e in E0], [dev(a, torch) for a in A0]
    touched = np.zeros((V, N), bool)
    for i, cam in enumerate(cams):
        pre = tgs.preprocess(cam, D, base["means3D"], base["scales"], base["quats"], base["opacities"], base["sh"])
        sp = tgs.sample_paper(cam, E2[i], A2[i], 25, 10, 8, seed=9 + i)
        b = tgs.bin_sort(cam, pre.splats, P_cap)
        fw = tgs.raster_fwd_sparse(cam, pre.splats, b, sp)
        lo = tgs.loss_sparse(cam, sp, fw.color, targets[i])
        tgs.maps_update(cam, E2[i], A2[i], sp, lo.pix_err, 0.4)
        bw = tgs.raster_bwd_sparse(cam, D, pre.splats, b, sp, fw, lo.dL_dcolor, base["means3D"], base["scales"],
                                   base["quats"], base["sh"], pre.radii, pre.clamped)
        G["means3D"][i], G["scales"][i], G["quats"][i] = bw.dL_dmeans3D, bw.dL_dscales, bw.dL_dquats
        G["opacities"][i], G["sh"][i] = bw.dL_dopacities, bw.dL_dsh
        touched[i] = (bw.dL_dsplats.cpu().numpy()[:, :9] != 0).any(axis=1)
        # the maps: integer / fixed-rounding work, deterministic given the same pix_err... which is (forward + loss are)
        assert torch.equal(E1[i], E2[i]) and torch.equal(A1[i], A2[i]), "maps of view %d" % i
    assert np.array_equal(it.touched.cpu().numpy() == 1, touched)
    p2, m2, v2 = clone(base), _dev(m_np, torch), _dev(v_np, torch)
    upd = torch.from_numpy(touched.any(0).astype(np.int32)).cuda()
    tgs.lm_solve(D, G, m2, v2, update=upd, t=2, want_delta=False, params=p2)
    torch.cuda.synchronize()
    for k in KEYS:
        a, b_, b0 = p1[k].cpu().numpy().astype(np.float64), p2[k].cpu().numpy().astype(np.float64), base[k].cpu().numpy()
        assert np.abs(a - b_).max() <= 1e-4 * np.abs(b_ - b0).max() + 1e-7, k
    assert np.abs(p2["means3D"].cpu().numpy() - base["means3D"].cpu().numpy()).max() > 0

    # one CUDA graph for the whole iteration, replayed on fresh state: same result as the eager run above
    p3, m3, v3 = clone(base), _dev(m_np, torch), _dev(v_np, torch)
    E3, A3 = [dev(e, torch) for e in E0], [dev(a, torch) for a in A0]
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        it.run_paper(p3, targets, E3, A3, m3, v3, t=2, **kw)      # warm-up on the capture stream
        s.synchronize()
        for dst, src in ((p3, base), (m3, _dev(m_np, torch)), (v3, _dev(v_np, torch))):
            for k in KEYS:
                dst[k].copy_(src[k])
        for i in range(V):
            E3[i].copy_(dev(E0[i], torch)); A3[i].copy_(dev(A0[i], torch))
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            it.run_paper(p3, targets, E3, A3, m3, v3, t=2, **kw)
    g.replay()
    torch.cuda.synchronize()
    for i in range(V):
        assert torch.equal(E3[i], E1[i]) and torch.equal(A3[i], A1[i])
    for k in KEYS:
        a, b_, b0 = p3[k].cpu().numpy().astype(np.float64), p1[k].cpu().numpy().astype(np.float64), base[k].cpu().numpy()
        assert np.abs(a - b_).max() <= 1e-4 * np.abs(b_ - b0).max() + 1e-7, k

    # a SECOND replay: t and the sampler seeds are host scalars baked into the captured launches (tgs.h, tgs_lm_solve),
    # so the replay is the eager call with the SAME t = 2 and seed = 9 on the state the first iteration left -- not an
    # iteration with t = 3.  Both start from identical state (the eager run's), in the buffers the graph points at.
    for dst, src in ((p3, p1), (m3, m1), (v3, v1)):
        for k in KEYS:
            dst[k].copy_(src[k])
    for i in range(V):
        E3[i].copy_(E1[i]); A3[i].copy_(A1[i])
    before = {k: p1[k].clone() for k in KEYS}
    it.run_paper(p1, targets, E1, A1, m1, v1, t=2, **kw)
    torch.cuda.synchronize()
    g.replay()
    torch.cuda.synchronize()
    for i in range(V):
        assert torch.equal(E3[i], E1[i]) and torch.equal(A3[i], A1[i]), "maps of view %d after the second replay" % i
    for k in KEYS:
        a, b_, b0 = p3[k].cpu().numpy().astype(np.float64), p1[k].cpu().numpy().astype(np.float64), before[k].cpu().numpy()
        assert np.abs(a - b_).max() <= 1e-4 * np.abs(b_ - b0).max() + 1e-7, k
        np.testing.assert_allclose(m3[k].cpu().numpy(), m1[k].cpu().numpy(), rtol=1e-3, atol=1e-9)
    assert np.abs(p1["means3D"].cpu().numpy() - before["means3D"].cpu().numpy()).max() > 0
