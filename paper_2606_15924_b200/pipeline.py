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
                err=None, render=None, target=None, stream=None, restrict=True):
        """restrict=True: sample first and bin only the selected tiles (tgs_bin_sort's tile_select;
        DESIGN.md R14).  restrict=False: bin every tile, then sample (the call order of north_star)."""
        t = self.tgs
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

    def backward(self, dL_dcolor, project=True, stream=None, sparse=False):
        """sparse=True: gradients as (touched mask, rows of the touched Gaussians); see tgs.h."""
        means3D, scales, quats, sh = self._inputs
        self.tgs.raster_bwd_sparse(self.cam, self.D, self.pre.splats, self.binned, self.samp, self.fwd, dL_dcolor,
                                   means3D, scales, quats, sh, self.pre.radii, self.pre.clamped, project=project,
                                   out=self.bwd, stream=stream, sparse=sparse)
        return self.bwd

    def counts(self):
        """(P, k, n) -- synchronises."""
        P, ovf = (int(v) for v in self.binned.P_dev.tolist())
        k, n = (int(v) for v in self.samp.kn_dev.tolist())
        if ovf:
            raise RuntimeError(f"P = {P} exceeds P_capacity = {self.P_capacity}")
        self.binned.P, self.samp.k, self.samp.n = P, k, n
        return P, k, n
