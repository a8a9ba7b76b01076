"""One sparse-raster training step (the five C-ABI calls in order) on pre-allocated buffers.

Host logic only: buffer ownership and call order.  Nothing here synchronises, so a step can be
captured in a CUDA graph; ``counts()`` reads the data-dependent sizes back (one sync).
"""
from __future__ import annotations

from types import SimpleNamespace

import torch

from .binding import Camera, SPLAT_WORDS, TGS


class SparseRasterStep:
    def __init__(self, tgs: TGS, cam, N: int, sh_degree: int, P_capacity: int, want_keys: bool = False,
                 want_walked: bool = False):
        self.tgs, self.cam, self.N, self.D = tgs, Camera.of(cam), int(N), int(sh_degree)
        self.P_capacity = int(P_capacity)
        dev = tgs.device
        T = self.cam.num_tiles
        npx = self.cam.width * self.cam.height
        K = (sh_degree + 1) ** 2
        f32, i32, i64, u8 = torch.float32, torch.int32, torch.int64, torch.uint8
        e = lambda shape, dt: torch.empty(shape, dtype=dt, device=dev)
        self.pre = SimpleNamespace(splats=e((N, SPLAT_WORDS), f32), radii=e(N, i32), clamped=e(N, u8))
        self.binned = SimpleNamespace(keys_sorted=e(max(P_capacity, 1), i64) if want_keys else None,
                                      gid_sorted=e(max(P_capacity, 1), i32), tile_offsets=e(T + 1, i32),
                                      P_dev=torch.zeros(2, dtype=i64, device=dev), P=None)
        self.samp = SimpleNamespace(tile_score=e(T, i64), tiles=e(T, i32), tile_pix_offsets=e(T + 1, i32),
                                    pix=e(npx, i32), tile_select=e(T, i32),
                                    kn_dev=torch.zeros(2, dtype=i32, device=dev), k=None, n=None)
        self.fwd = SimpleNamespace(color=e((npx, 3), f32), T=e(npx, f32), n_contrib=e(npx, i32),
                                   n_walked=e(npx, i32) if want_walked else None,
                                   n_blended=e(npx, i32) if want_walked else None)
        self.bwd = SimpleNamespace(dL_dsplats=e((N, SPLAT_WORDS), f32), dL_dmeans3D=e((N, 3), f32),
                                   dL_dscales=e((N, 3), f32), dL_dquats=e((N, 4), f32), dL_dopacities=e(N, f32),
                                   dL_dsh=e((N, K, 3), f32), touched=e(N, i32))
        self.ws_sort = e(tgs.bin_sort_workspace_bytes(N, P_capacity, T), u8)
        self.ws_sample = e(tgs.sample_workspace_bytes(self.cam), u8)
        self._side = torch.cuda.Stream(device=dev)
        self._ev_fork, self._ev_join = torch.cuda.Event(), torch.cuda.Event()

    def forward(self, means3D, scales, quats, opacities, sh, tile_pct, pixel_mode, pix_rate=(1, 1), seed=0,
                err=None, render=None, target=None, stream=None, restrict=True, cam=None):
        """restrict=True: sample first and bin only the selected tiles (tgs_bin_sort's tile_select;
        DESIGN.md R14).  restrict=False: bin every tile, then sample (the call order of north_star).
        cam: another view of the same image size (the buffers are sized by the image, not by the pose)."""
        t = self.tgs
        if cam is not None:
            cam = Camera.of(cam)
            assert (cam.width, cam.height) == (self.cam.width, self.cam.height), "a step's views share the image size"
            self.cam = cam
        if restrict:
            # projection and sampling do not depend on each other: the sampler runs on a side stream (fork / join by
            # events, also under graph capture) while the projection runs on the caller's stream
            main = stream if stream is not None else torch.cuda.current_stream()
            self._ev_fork.record(main)
            self._side.wait_event(self._ev_fork)
            t.sample(self.cam, tile_pct, pixel_mode, pix_rate, seed, err=err, render=render, target=target,
                     out=self.samp, workspace=self.ws_sample, sync=False, stream=self._side)
            self._ev_join.record(self._side)
            t.preprocess(self.cam, self.D, means3D, scales, quats, opacities, sh, out=self.pre, stream=stream)
            main.wait_event(self._ev_join)
            t.bin_sort(self.cam, self.pre.splats, self.P_capacity, out=self.binned, workspace=self.ws_sort, sync=False,
                       stream=stream, tile_select=self.samp.tile_select)
        else:
            t.preprocess(self.cam, self.D, means3D, scales, quats, opacities, sh, out=self.pre, stream=stream)
            t.bin_sort(self.cam, self.pre.splats, self.P_capacity, out=self.binned, workspace=self.ws_sort, sync=False,
                       stream=stream)
            t.sample(self.cam, tile_pct, pixel_mode, pix_rate, seed, err=err, render=render, target=target,
                     out=self.samp, workspace=self.ws_sample, sync=False, stream=stream)
        t.raster_fwd_sparse(self.cam, self.pre.splats, self.binned, self.samp, out=self.fwd, stream=stream)
        self._inputs = (means3D, scales, quats, sh)
        return self.fwd

    def backward(self, dL_dcolor, project=True, stream=None, sparse=False, out=None):
        """sparse=True: gradients as (touched mask, rows of the touched Gaussians); see tgs.h.
        out: where the gradients go (default: the step's own buffers), e.g. one view's slices of [V, N, ...] buffers."""
        means3D, scales, quats, sh = self._inputs
        out = out if out is not None else self.bwd
        self.tgs.raster_bwd_sparse(self.cam, self.D, self.pre.splats, self.binned, self.samp, self.fwd, dL_dcolor,
                                   means3D, scales, quats, sh, self.pre.radii, self.pre.clamped, project=project,
                                   out=out, stream=stream, sparse=sparse)
        return out

    def counts(self):
        """(P, k, n) -- synchronises."""
        P, ovf = (int(v) for v in self.binned.P_dev.tolist())
        k, n = (int(v) for v in self.samp.kn_dev.tolist())
        if ovf:
            raise RuntimeError(f"P = {P} exceeds P_capacity = {self.P_capacity}")
        self.binned.P, self.samp.k, self.samp.n = P, k, n
        return P, k, n


class SparseIteration:
    """Alg. 1 steps 3-10 for the V views of one iteration, all on the device: per view the five-call
    step, the fused sparse loss and the sparse backward -- its gradients written view-major into [V, N, ...] buffers
    with one `touched` mask per view -- then ONE tgs_lm_solve over the V views that updates the moments and the
    parameters in place.  Host logic only: buffer ownership and call order; nothing synchronises."""

    def __init__(self, tgs: TGS, cams, N: int, sh_degree: int, P_capacity: int):
        self.tgs, self.cams, self.N, self.D = tgs, [Camera.of(c) for c in cams], int(N), int(sh_degree)
        V, K, dev = len(self.cams), (sh_degree + 1) ** 2, tgs.device
        # view i's SH gradients are the slice grads["sh"][i] of one [V, N, K, 3] buffer, and the kernels read and write SH
        # rows as float4: the per-view stride N*K*3 floats must be a multiple of 4 (only sh_degree 2, K = 9, with N % 4 != 0
        # breaks it).  Refused here, at construction, rather than by tgs_raster_bwd_sparse in the middle of an iteration.
        if V > 1 and (self.N * K * 3) % 4 != 0:
            raise ValueError(f"SparseIteration: with sh_degree = {sh_degree} the per-view SH gradient slice is "
                             f"{self.N * K * 3} floats, not a multiple of 4 (16-byte alignment of every view's slice): "
                             f"make N = {self.N} a multiple of 4")
        self.step = SparseRasterStep(tgs, self.cams[0], N, sh_degree, P_capacity)
        f = dict(dtype=torch.float32, device=dev)
        self.grads = {"means3D": torch.empty((V, N, 3), **f), "scales": torch.empty((V, N, 3), **f),
                      "quats": torch.empty((V, N, 4), **f), "opacities": torch.empty((V, N), **f),
                      "sh": torch.empty((V, N, K, 3), **f)}
        self.touched = torch.empty((V, N), dtype=torch.int32, device=dev)
        g = self.grads
        self.views = [SimpleNamespace(dL_dsplats=self.step.bwd.dL_dsplats, dL_dmeans3D=g["means3D"][i],
                                      dL_dscales=g["scales"][i], dL_dquats=g["quats"][i], dL_dopacities=g["opacities"][i],
                                      dL_dsh=g["sh"][i], touched=self.touched[i]) for i in range(V)]
        self.losses = [None] * V
        self.delta = None

    def _solve(self, params, m, v, t, beta1, beta2, eps, eta_sh, apply, stream):
        """Alg. 1 steps 9-10.  apply=False (the default of run / run_paper): the update goes to self.delta and the
        parameters are left alone.  Eq. 14 prints no step size: with small gradients it degenerates to a unit-rate Adam
        step, and three such steps blow the scales up on configs[3] (R37) -- so the step as printed is only
        applied when the caller asks for it with apply=True; a caller that wants a trust region scales Delta itself."""
        if not apply and self.delta is None:
            self.delta = {k: torch.empty_like(a) for k, a in params.items()}
        self.tgs.lm_solve(self.D, self.grads, m, v, view_touched=self.touched, beta1=beta1, beta2=beta2, eps=eps,
                          eta_sh=eta_sh, t=t, want_delta=not apply, delta=None if apply else self.delta,
                          params=params if apply else None, stream=stream)

    def run(self, params, targets, errs, m, v, t, tile_pct, pixel_mode, pix_rate=(1, 1), seed=0, beta1=0.9, beta2=0.999,
            eps=1e-8, eta_sh=1.25e-4, stream=None, apply=False):
        """params, m, v: parameter sets (dicts of device tensors); m and v are updated in place, params only with
        apply=True (Alg. 1 step 10 as printed, no step size: DESIGN.md R37), otherwise Delta is left in self.delta;
        targets[i]: [H, W, 3] image of view i; errs[i]: [H, W] error map that drives view i's sampling.  Returns the
        per-view loss namespaces.
        CUDA graphs: t (the bias correction of Eq. 19) and the per-view sampler seeds seed + i are HOST scalars that go
        into the launch arguments, so a captured iteration replays with the t and the seeds it was captured with:
        re-capture (or update the kernel-node parameters) every iteration that needs new ones."""
        st, tg = self.step, self.tgs
        for i, cam in enumerate(self.cams):
            fw = st.forward(params["means3D"], params["scales"], params["quats"], params["opacities"], params["sh"],
                            tile_pct, pixel_mode, pix_rate, seed + i, err=errs[i], stream=stream, cam=cam)
            samp = SimpleNamespace(k=tg.sample_num_tiles(cam, tile_pct[0], tile_pct[1]), n=None,
                                   tile_pix_offsets=st.samp.tile_pix_offsets, pix=st.samp.pix)
            lo = tg.loss_sparse(cam, samp, fw.color, targets[i], out=self.losses[i], stream=stream)
            self.losses[i] = lo
            st.samp.k = samp.k
            st.backward(lo.dL_dcolor, sparse=True, out=self.views[i], stream=stream)
        self._solve(params, m, v, t, beta1, beta2, eps, eta_sh, apply, stream)
        return self.losses

    def run_paper(self, params, targets, E_maps, ages, m, v, t, n_pix=25, n_hard=10, n_stable=8, beta=0.4, seed=0,
                  beta1=0.9, beta2=0.999, eps=1e-8, eta_sh=1.25e-4, stream=None, apply=False):
        """The same iteration with the paper's own sampler: per view, n_pix pixels in EVERY tile from the
        view's persistent maps -- E_maps[i] (fp16 bits, [H, W]) and ages[i] (uint16 bits) --, all tiles binned, sparse
        forward, fused loss, map update with the loss kernel's per-pixel error (Eq. 3-4), sparse backward; then the LM
        solve.  m, v and the maps are updated in place; params only with apply=True (see run), else Delta is in
        self.delta.  A captured graph of this call replays with the t and seeds of the capture (see run)."""
        st, tg, D = self.step, self.tgs, self.D
        p = params
        for i, cam in enumerate(self.cams):
            st.cam = cam
            tg.preprocess(cam, D, p["means3D"], p["scales"], p["quats"], p["opacities"], p["sh"], out=st.pre, stream=stream)
            sp = tg.sample_paper(cam, E_maps[i], ages[i], n_pix, n_hard, n_stable, seed=seed + i, out=st.samp,
                                 workspace=st.ws_sample, sync=False, stream=stream)
            tg.bin_sort(cam, st.pre.splats, st.P_capacity, out=st.binned, workspace=st.ws_sort, sync=False, stream=stream)
            fw = tg.raster_fwd_sparse(cam, st.pre.splats, st.binned, sp, out=st.fwd, stream=stream)
            lo = tg.loss_sparse(cam, sp, fw.color, targets[i], out=self.losses[i], stream=stream)
            self.losses[i] = lo
            tg.maps_update(cam, E_maps[i], ages[i], sp, lo.pix_err, beta, stream=stream)
            tg.raster_bwd_sparse(cam, D, st.pre.splats, st.binned, sp, st.fwd, lo.dL_dcolor, p["means3D"], p["scales"],
                                 p["quats"], p["sh"], st.pre.radii, st.pre.clamped, out=self.views[i], stream=stream,
                                 sparse=True)
        self._solve(params, m, v, t, beta1, beta2, eps, eta_sh, apply, stream)
        return self.losses
