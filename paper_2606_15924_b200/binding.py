"""Thin ctypes binding of libtgs.so (include/tgs.h).  Argument marshalling only: every step of
the hot path runs in the CUDA kernels; torch is used for device memory and streams.

There is no fallback: importing this module without the built library, or creating a context
without a CUDA device, raises.
"""
from __future__ import annotations

import ctypes as C
import os
from types import SimpleNamespace

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtgs.so")

SPLAT_WORDS = 12
PIXELS_ALL = 0
PIXELS_BERNOULLI_ERR = 1

ERR_NAMES = {0: "TGS_OK", 1: "TGS_ERR_INVALID_ARG", 2: "TGS_ERR_CAPACITY", 3: "TGS_ERR_CUDA",
             4: "TGS_ERR_UNSUPPORTED"}

# every symbol include/tgs.h declares (tests check the library exports them all)
SYMBOLS = ["tgs_create", "tgs_destroy", "tgs_last_error", "tgs_version", "tgs_launch_count", "tgs_fp32_peak", "tgs_preprocess",
           "tgs_bin_sort_workspace_bytes", "tgs_bin_sort", "tgs_sample_num_tiles",
           "tgs_sample_workspace_bytes", "tgs_sample", "tgs_sample_static", "tgs_raster_fwd_sparse", "tgs_raster_bwd_sparse", "tgs_loss_sparse", "tgs_raster_stats_sparse", "tgs_sample_paper",
           "tgs_maps_update", "tgs_lm_solve"]
PARAM_KEYS = ("means3D", "scales", "quats", "opacities", "sh")


class TgsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{ERR_NAMES.get(code, code)}: {msg}")
        self.code = code


class Camera(C.Structure):
    _fields_ = [("width", C.c_int32), ("height", C.c_int32), ("fx", C.c_float), ("fy", C.c_float),
                ("cx", C.c_float), ("cy", C.c_float), ("R", C.c_float * 9), ("t", C.c_float * 3),
                ("znear", C.c_float), ("bg", C.c_float * 3)]

    @staticmethod
    def of(cam) -> "Camera":
        """From any object with width height fx fy cx cy R t znear bg (e.g. workloads.Camera)."""
        if isinstance(cam, Camera):
            return cam
        c = Camera()
        c.width, c.height = int(cam.width), int(cam.height)
        c.fx, c.fy, c.cx, c.cy, c.znear = float(cam.fx), float(cam.fy), float(cam.cx), float(cam.cy), float(cam.znear)
        R = [float(v) for v in list(getattr(cam.R, "reshape", lambda *_: cam.R)(-1))]
        for i in range(9):
            c.R[i] = R[i]
        for i in range(3):
            c.t[i] = float(cam.t[i])
            c.bg[i] = float(cam.bg[i])
        return c

    @property
    def grid(self):
        return ((self.width + 15) // 16, (self.height + 15) // 16)

    @property
    def num_tiles(self):
        gx, gy = self.grid
        return gx * gy


class Params(C.Structure):
    """tgs_params: five device pointers in the parameter layouts."""
    _fields_ = [(k, C.c_void_p) for k in ("means3D", "scales", "quats", "opacities", "sh")]

    @staticmethod
    def of(ps) -> "Params":
        """From a dict (or any object) holding the five device tensors under PARAM_KEYS."""
        get = ps.__getitem__ if isinstance(ps, dict) else (lambda k: getattr(ps, k))
        q = Params()
        for k in PARAM_KEYS:
            t = get(k)
            assert t.is_cuda and t.is_contiguous() and t.dtype == torch.float32, "device, contiguous, fp32 tensors only"
            setattr(q, k, t.data_ptr())
        return q


def load_library() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_15924_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i32, i64, u64 = C.c_void_p, C.c_int, C.c_int64, C.c_uint64
    lib.tgs_create.argtypes = [C.POINTER(vp), i32]
    lib.tgs_destroy.argtypes = [vp]
    lib.tgs_last_error.argtypes = [vp]
    lib.tgs_last_error.restype = C.c_char_p
    lib.tgs_version.restype = C.c_char_p
    lib.tgs_launch_count.restype = C.c_uint64
    lib.tgs_fp32_peak.argtypes = [vp, i32, C.POINTER(C.c_double), vp]
    cam = C.POINTER(Camera)
    lib.tgs_preprocess.argtypes = [vp, cam, i32, i32] + [vp] * 5 + [vp] * 3 + [vp]
    lib.tgs_bin_sort_workspace_bytes.argtypes = [i32, i64, i32, C.POINTER(C.c_size_t)]
    lib.tgs_bin_sort.argtypes = [vp, cam, i32, vp, vp, i64, vp, vp, vp, vp, C.POINTER(i64), vp, C.c_size_t, vp]
    lib.tgs_sample_num_tiles.argtypes = [cam, i32, i32]
    lib.tgs_sample_workspace_bytes.argtypes = [cam, C.POINTER(C.c_size_t)]
    lib.tgs_sample.argtypes = [vp, cam, vp, vp, vp, i32, i32, i32, i32, i32, u64, vp, vp, vp, vp, vp, vp,
                               C.POINTER(C.c_int32), vp, C.c_size_t, vp]
    lib.tgs_sample_static.argtypes = [i32, cam, vp, vp, vp, i32, i32, i32, i32, i32, u64, vp, vp, vp, vp, vp, vp,
                                      C.POINTER(C.c_int32), C.c_char_p, C.c_size_t, vp]
    lib.tgs_raster_fwd_sparse.argtypes = [vp, cam, i32, vp, vp, vp, i32, vp, vp, vp, vp, vp, vp, vp, vp, vp]
    lib.tgs_raster_bwd_sparse.argtypes = [vp, cam, i32, i32, vp, vp, vp, i32, vp, vp, vp, vp, vp, vp] + [vp] * 6 + \
                                         [vp] + [vp] * 5 + [vp, vp]
    f32 = C.c_float
    lib.tgs_loss_sparse.argtypes = [vp, cam, i32, vp, vp, vp, vp, f32, f32, f32, vp, vp, vp, vp, vp]
    lib.tgs_raster_stats_sparse.argtypes = [vp, cam, i32, vp, vp, vp, i32, vp, vp, vp, vp, vp, vp, vp]
    lib.tgs_sample_paper.argtypes = [vp, cam, vp, vp, i32, i32, i32, u64, vp, vp, vp, vp, C.POINTER(C.c_int32), vp,
                                     C.c_size_t, vp]
    lib.tgs_maps_update.argtypes = [vp, cam, vp, vp, vp, vp, vp, f32, vp]
    ps = C.POINTER(Params)
    lib.tgs_lm_solve.argtypes = [vp, i32, i32, i32, ps, vp, vp, f32, f32, f32, f32, i32, ps, ps, ps, ps, vp]
    return lib


def _p(t):
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device, contiguous tensors only"
    return C.c_void_p(t.data_ptr())


def _stream(stream=None):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


SAMPLE_STATIC_MAX_TILES = 16384  # TGS_SAMPLE_STATIC_MAX_TILES of include/tgs.h


def sample_static(device, cam, tile_pct, pixel_mode, out, pix_rate=(1, 1), seed=0, err=None, render=None, target=None,
                  sync=True, stream=None, lib=None):
    """tgs_sample_static: what `TGS.sample` computes, for a caller that may not allocate device memory.

    Some programs that embed this library are handed their GPU buffers and are not allowed (or not able) to get more:
    a plug-in under a host application's memory budget, a step in a loop that cannot afford cudaMalloc's device-wide
    synchronisation, a process whose framework allocator already owns all of HBM.  This call needs no `TGS` context
    and no workspace: its scratch is a fixed 640 KiB array inside the loaded library, good for images of up to
    SAMPLE_STATIC_MAX_TILES = 16384 tiles (2048 x 2048); a larger image raises TgsError (TGS_ERR_CAPACITY).

    `out` is REQUIRED and is the caller's: a namespace with device tensors tile_score[T] (int64), tiles[T],
    tile_pix_offsets[T+1], pix[W*H], kn_dev[2] (int32) and optionally tile_select[T] -- the fields `TGS.sample`
    returns.  This wrapper allocates no tensor either.  The first call on a device resolves the scratch address
    (it may load the library's device code): make it during start-up, before capturing any stream.  All calls on
    one GPU share the one scratch array: issue them on one stream, or order them with events -- calls that overlap
    on the GPU corrupt each other's pixel lists."""
    lib = lib if lib is not None else load_library()
    cam = Camera.of(cam)
    kn = (C.c_int32 * 2)(-1, -1)
    msg = C.create_string_buffer(512)
    rc = lib.tgs_sample_static(int(device), C.byref(cam), _p(err), _p(render), _p(target), int(tile_pct[0]),
                               int(tile_pct[1]), int(pixel_mode), int(pix_rate[0]), int(pix_rate[1]), C.c_uint64(seed),
                               _p(out.tile_score), _p(out.tiles), _p(out.tile_pix_offsets), _p(out.pix),
                               _p(getattr(out, "tile_select", None)), _p(out.kn_dev), kn if sync else None,
                               msg, len(msg), _stream(stream))
    if rc != 0:
        raise TgsError(rc, msg.value.decode())
    out.k = lib.tgs_sample_num_tiles(C.byref(cam), int(tile_pct[0]), int(tile_pct[1]))
    if sync:
        assert kn[0] == out.k
        out.n = int(kn[1])
    return out


class TGS:
    """One library context on one CUDA device.  Method names are the C-ABI names without `tgs_`."""

    def __init__(self, device: int = 0):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_15924_b200 needs a CUDA device (no CPU fallback)")
        self.lib = load_library()
        self.device = torch.device("cuda", device)
        torch.cuda.set_device(self.device)
        torch.cuda.current_stream()  # make sure the primary context exists
        h = C.c_void_p()
        rc = self.lib.tgs_create(C.byref(h), device)
        if rc != 0:
            raise TgsError(rc, "tgs_create failed")
        self._h = h

    def __del__(self):
        h = getattr(self, "_h", None)
        if h:
            self.lib.tgs_destroy(h)
            self._h = None

    def launch_count(self) -> int:
        return int(self.lib.tgs_launch_count())

    def fp32_peak(self, reps: int = 10, stream=None) -> float:
        """Measured FFMA-only peak in TFLOP/s (tgs_fp32_peak)."""
        v = C.c_double()
        self._check(self.lib.tgs_fp32_peak(self._h, reps, C.byref(v), _stream(stream)))
        return float(v.value)

    def _check(self, rc):
        if rc != 0:
            raise TgsError(rc, self.lib.tgs_last_error(self._h).decode())

    # ---- a1 ----
    def preprocess(self, cam, sh_degree, means3D, scales, quats, opacities, sh, out=None, stream=None):
        cam = Camera.of(cam)
        N = means3D.shape[0]
        if out is None:
            out = SimpleNamespace(splats=torch.empty((N, SPLAT_WORDS), dtype=torch.float32, device=self.device),
                                  radii=torch.empty(N, dtype=torch.int32, device=self.device),
                                  clamped=torch.empty(N, dtype=torch.uint8, device=self.device))
        self._check(self.lib.tgs_preprocess(self._h, C.byref(cam), N, sh_degree, _p(means3D), _p(scales), _p(quats),
                                            _p(opacities), _p(sh), _p(out.splats), _p(out.radii), _p(out.clamped),
                                            _stream(stream)))
        return out

    # ---- a2 ----
    def bin_sort_workspace_bytes(self, N, P_capacity, num_tiles):
        b = C.c_size_t()
        rc = self.lib.tgs_bin_sort_workspace_bytes(N, P_capacity, num_tiles, C.byref(b))
        if rc != 0:
            raise TgsError(rc, "tgs_bin_sort_workspace_bytes")
        return b.value

    def bin_sort(self, cam, splats, P_capacity, want_keys=False, out=None, workspace=None, sync=True, stream=None,
                 tile_select=None):
        cam = Camera.of(cam)
        N = splats.shape[0]
        T = cam.num_tiles
        if out is None:
            out = SimpleNamespace(
                keys_sorted=torch.empty(max(P_capacity, 1), dtype=torch.int64, device=self.device) if want_keys else None,
                gid_sorted=torch.empty(max(P_capacity, 1), dtype=torch.int32, device=self.device),
                tile_offsets=torch.empty(T + 1, dtype=torch.int32, device=self.device),
                P_dev=torch.zeros(2, dtype=torch.int64, device=self.device), P=None)
        need = self.bin_sort_workspace_bytes(N, P_capacity, T)
        if workspace is None:
            workspace = torch.empty(need, dtype=torch.uint8, device=self.device)
        ph = C.c_int64(-1)
        rc = self.lib.tgs_bin_sort(self._h, C.byref(cam), N, _p(splats), _p(tile_select), P_capacity, _p(out.keys_sorted),
                                   _p(out.gid_sorted), _p(out.tile_offsets), _p(out.P_dev),
                                   C.byref(ph) if sync else None, _p(workspace), workspace.numel(), _stream(stream))
        if sync:
            out.P = ph.value
        self._check(rc)
        return out

    # ---- a3 ----
    def sample_num_tiles(self, cam, num, den):
        cam = Camera.of(cam)
        return self.lib.tgs_sample_num_tiles(C.byref(cam), num, den)

    def sample_workspace_bytes(self, cam):
        cam = Camera.of(cam)
        b = C.c_size_t()
        rc = self.lib.tgs_sample_workspace_bytes(C.byref(cam), C.byref(b))
        if rc != 0:
            raise TgsError(rc, "tgs_sample_workspace_bytes")
        return b.value

    def sample(self, cam, tile_pct, pixel_mode, pix_rate=(1, 1), seed=0, err=None, render=None, target=None,
               out=None, workspace=None, sync=True, stream=None):
        cam = Camera.of(cam)
        T = cam.num_tiles
        if out is None:
            out = SimpleNamespace(tile_score=torch.empty(T, dtype=torch.int64, device=self.device),
                                  tiles=torch.empty(T, dtype=torch.int32, device=self.device),
                                  tile_pix_offsets=torch.empty(T + 1, dtype=torch.int32, device=self.device),
                                  pix=torch.empty(cam.width * cam.height, dtype=torch.int32, device=self.device),
                                  tile_select=torch.empty(T, dtype=torch.int32, device=self.device),
                                  kn_dev=torch.zeros(2, dtype=torch.int32, device=self.device), k=None, n=None)
        if workspace is None:
            workspace = torch.empty(self.sample_workspace_bytes(cam), dtype=torch.uint8, device=self.device)
        kn = (C.c_int32 * 2)(-1, -1)
        self._check(self.lib.tgs_sample(self._h, C.byref(cam), _p(err), _p(render), _p(target), int(tile_pct[0]),
                                        int(tile_pct[1]), int(pixel_mode), int(pix_rate[0]), int(pix_rate[1]),
                                        C.c_uint64(seed), _p(out.tile_score), _p(out.tiles), _p(out.tile_pix_offsets),
                                        _p(out.pix), _p(getattr(out, "tile_select", None)), _p(out.kn_dev),
                                        kn if sync else None, _p(workspace),
                                        workspace.numel(), _stream(stream)))
        out.k = self.sample_num_tiles(cam, tile_pct[0], tile_pct[1])
        if sync:
            assert kn[0] == out.k
            out.n = int(kn[1])
        return out

    # ---- f2: the paper's own sampler (every tile, N_pix pixels each) and its maps ----
    def sample_paper(self, cam, E_half, age, n_pix, n_hard, n_stable, seed=0, out=None, workspace=None, sync=True,
                     stream=None):
        """E_half: int16/uint16 device tensor [H,W] holding fp16 bit patterns (or a float16 tensor); age: int16 [H,W]."""
        cam = Camera.of(cam)
        T = cam.num_tiles
        if out is None:
            i32t = dict(dtype=torch.int32, device=self.device)
            out = SimpleNamespace(tiles=torch.empty(T, **i32t), tile_pix_offsets=torch.empty(T + 1, **i32t),
                                  pix=torch.empty(cam.width * cam.height, **i32t), kn_dev=torch.zeros(2, **i32t),
                                  k=None, n=None)
        if workspace is None:
            workspace = torch.empty(self.sample_workspace_bytes(cam), dtype=torch.uint8, device=self.device)
        kn = (C.c_int32 * 2)(-1, -1)
        self._check(self.lib.tgs_sample_paper(self._h, C.byref(cam), _p(E_half), _p(age), int(n_pix), int(n_hard),
                                              int(n_stable), C.c_uint64(seed), _p(out.tiles), _p(out.tile_pix_offsets),
                                              _p(out.pix), _p(out.kn_dev), kn if sync else None, _p(workspace),
                                              workspace.numel(), _stream(stream)))
        out.k = T
        if sync:
            assert kn[0] == T
            out.n = int(kn[1])
        return out

    def maps_update(self, cam, E_half, age, samp, pix_err, beta, stream=None):
        """In place: Eq. 4 on age, Eq. 3 on E_half at the pixels of `samp` (its kn_dev gives n)."""
        cam = Camera.of(cam)
        self._check(self.lib.tgs_maps_update(self._h, C.byref(cam), _p(E_half), _p(age), _p(samp.kn_dev), _p(samp.pix),
                                             _p(pix_err), float(beta), _stream(stream)))

    # ---- a4 ----
    def raster_fwd_sparse(self, cam, splats, binned, samp, n_capacity=None, want_walked=False, out=None, stream=None):
        cam = Camera.of(cam)
        n = n_capacity if n_capacity is not None else (samp.n if samp.n is not None else samp.pix.numel())
        if out is None:
            out = SimpleNamespace(color=torch.empty((n, 3), dtype=torch.float32, device=self.device),
                                  T=torch.empty(n, dtype=torch.float32, device=self.device),
                                  n_contrib=torch.empty(n, dtype=torch.int32, device=self.device),
                                  n_walked=torch.empty(n, dtype=torch.int32, device=self.device) if want_walked else None,
                                  n_blended=torch.empty(n, dtype=torch.int32, device=self.device) if want_walked else None)
        self._check(self.lib.tgs_raster_fwd_sparse(self._h, C.byref(cam), splats.shape[0], _p(splats),
                                                   _p(binned.tile_offsets), _p(binned.gid_sorted), samp.k,
                                                   _p(samp.tiles), _p(samp.tile_pix_offsets), _p(samp.pix),
                                                   _p(out.color), _p(out.T), _p(out.n_contrib), _p(out.n_walked),
                                                   _p(getattr(out, "n_blended", None)), _stream(stream)))
        return out

    # ---- f1: sparse supervision between the forward and the backward ----
    def loss_sparse(self, cam, samp, color, target, eps_l1=1e-3, eps_ncc=1e-6, eps_lambda=1e-8, n_capacity=None,
                    want_loss=True, out=None, stream=None):
        cam = Camera.of(cam)
        n = n_capacity if n_capacity is not None else (samp.n if samp.n is not None else samp.pix.numel())
        if out is None:
            f = dict(dtype=torch.float32, device=self.device)
            out = SimpleNamespace(dL_dcolor=torch.empty((n, 3), **f), pix_err=torch.empty(n, **f),
                                  tile_stats=torch.empty((max(samp.k, 1), 3), **f),
                                  loss=torch.zeros(2, **f) if want_loss else None)
        self._check(self.lib.tgs_loss_sparse(self._h, C.byref(cam), samp.k, _p(samp.tile_pix_offsets), _p(samp.pix),
                                             _p(color), _p(target), eps_l1, eps_ncc, eps_lambda, _p(out.dL_dcolor),
                                             _p(out.pix_err), _p(out.tile_stats), _p(out.loss), _stream(stream)))
        return out

    # ---- f3: statistics forward (E_i, D_i, W_i per Gaussian, expected depth per sampled pixel) ----
    def raster_stats_sparse(self, cam, splats, binned, samp, pix_err, n_capacity=None, want_depth=True, out=None,
                            stream=None):
        cam = Camera.of(cam)
        n = n_capacity if n_capacity is not None else (samp.n if samp.n is not None else samp.pix.numel())
        N = splats.shape[0]
        if out is None:
            f = dict(dtype=torch.float32, device=self.device)
            out = SimpleNamespace(stats=torch.empty((max(N, 1), 4), **f), depth=torch.empty(max(n, 1), **f) if want_depth else None)
        self._check(self.lib.tgs_raster_stats_sparse(self._h, C.byref(cam), N, _p(splats), _p(binned.tile_offsets),
                                                     _p(binned.gid_sorted), samp.k, _p(samp.tiles),
                                                     _p(samp.tile_pix_offsets), _p(samp.pix), _p(pix_err), _p(out.stats),
                                                     _p(out.depth), _stream(stream)))
        return out

    # ---- f4: moment-damped LM solve (Alg. 1 steps 9-10) ----
    def lm_solve(self, sh_degree, grads, m, v, update=None, view_touched=None, beta1=0.9, beta2=0.999, eps=1e-8, eta_sh=1.25e-4, t=1,
                 want_delta=True, delta=None, params=None, stream=None):
        """grads: parameter set with a leading view axis [V,N,...]; m, v (and params, if given) are updated in place.
        view_touched: [V,N] int32, the `touched` masks of the V backward calls (rows of grads are read only where set).
        Returns the delta parameter set (allocated here unless given; None if want_delta is False)."""
        V, N = grads["opacities"].shape
        K = (sh_degree + 1) ** 2
        if not 1 <= V <= 64:
            raise ValueError(f"lm_solve: V = {V} views, the kernels take 1..64")
        # the kernels index raw pointers with these extents: a wrong dtype or shape is misread silently (a bool mask
        # even out of bounds), so it is refused here
        shapes = {"means3D": (N, 3), "scales": (N, 3), "quats": (N, 4), "opacities": (N,), "sh": (N, K, 3)}
        for name, ps, lead in (("grads", grads, (V,)), ("m", m, ()), ("v", v, ()), ("delta", delta, ()), ("params", params, ())):
            if ps is None or not 0 <= sh_degree <= 3:   # an unsupported degree is the library's to refuse (TGS_ERR_UNSUPPORTED)
                continue
            for k in PARAM_KEYS:
                if tuple(ps[k].shape) != lead + shapes[k]:
                    raise ValueError(f"lm_solve: {name}[{k!r}] has shape {tuple(ps[k].shape)}, expected {lead + shapes[k]}")
        for name, mask, shape in (("update", update, (N,)), ("view_touched", view_touched, (V, N))):
            if mask is not None and (mask.dtype != torch.int32 or tuple(mask.shape) != shape):
                raise ValueError(f"lm_solve: {name} must be an int32 tensor of shape {shape}, got {mask.dtype} "
                                 f"{tuple(mask.shape)}")
        if delta is None and want_delta:
            delta = {k: torch.empty_like(m[k]) for k in PARAM_KEYS}
        pg, pm, pv = Params.of(grads), Params.of(m), Params.of(v)
        pd = Params.of(delta) if delta is not None else None
        pp = Params.of(params) if params is not None else None
        self._check(self.lib.tgs_lm_solve(self._h, N, sh_degree, V, C.byref(pg), _p(update), _p(view_touched), beta1, beta2, eps, eta_sh, int(t),
                                          C.byref(pm), C.byref(pv), C.byref(pd) if pd is not None else None,
                                          C.byref(pp) if pp is not None else None, _stream(stream)))
        return delta

    # ---- a5 + a6 ----
    def raster_bwd_sparse(self, cam, sh_degree, splats, binned, samp, fwd, dL_dcolor, means3D=None, scales=None,
                          quats=None, sh=None, radii=None, clamped=None, project=True, out=None, stream=None,
                          sparse=False):
        """sparse=True: out.touched[N] (int32) marks the Gaussians with a non-zero gradient; the rows of the others are
        left unwritten (tgs.h: sparse gradients)."""
        cam = Camera.of(cam)
        N = splats.shape[0]
        if out is None:
            out = SimpleNamespace(dL_dsplats=torch.empty((N, SPLAT_WORDS), dtype=torch.float32, device=self.device))
            if project:
                K = (sh_degree + 1) ** 2
                out.dL_dmeans3D = torch.empty((N, 3), dtype=torch.float32, device=self.device)
                out.dL_dscales = torch.empty((N, 3), dtype=torch.float32, device=self.device)
                out.dL_dquats = torch.empty((N, 4), dtype=torch.float32, device=self.device)
                out.dL_dopacities = torch.empty(N, dtype=torch.float32, device=self.device)
                out.dL_dsh = torch.empty((N, K, 3), dtype=torch.float32, device=self.device)
        if sparse and getattr(out, "touched", None) is None:
            out.touched = torch.empty(N, dtype=torch.int32, device=self.device)
        g = lambda name: _p(getattr(out, name)) if project else None
        self._check(self.lib.tgs_raster_bwd_sparse(
            self._h, C.byref(cam), N, sh_degree, _p(splats), _p(binned.tile_offsets), _p(binned.gid_sorted), samp.k,
            _p(samp.tiles), _p(samp.tile_pix_offsets), _p(samp.pix), _p(fwd.T), _p(fwd.n_contrib), _p(dL_dcolor),
            _p(means3D), _p(scales), _p(quats), _p(sh), _p(radii), _p(clamped), _p(out.dL_dsplats),
            g("dL_dmeans3D"), g("dL_dscales"), g("dL_dquats"), g("dL_dopacities"), g("dL_dsh"),
            _p(out.touched) if (sparse and project) else None, _stream(stream)))
        return out
