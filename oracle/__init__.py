"""CPU ORACLE (test infrastructure, NOT the product) -- ctypes front end of tgs_oracle.c.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports the CUDA package
``paper_2606_15924_b200`` and shares no code with it; cameras are duck-typed (any object
with ``width height fx fy cx cy R t znear bg``), scenes come from ``workloads``.

Two builds of the same C source: ``Oracle("f32")`` (the parity referee, discrete decisions in
the kernel's precision) and ``Oracle("f64")`` (finite differences, cross-checks).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from types import SimpleNamespace

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tgs_oracle.c")


# ORACLE_SANITIZE=1: a second build with -fsanitize=address,undefined; run the CPU suite as
#   ORACLE_SANITIZE=1 LD_PRELOAD="$(gcc -print-file-name=libasan.so) $(gcc -print-file-name=libubsan.so)" \
#   ASAN_OPTIONS=detect_leaks=0 python -m pytest tests -q -m "not gpu"
_SANITIZE = os.environ.get("ORACLE_SANITIZE", "") not in ("", "0")


def _lib_path(prec: str) -> str:
    return os.path.join(_HERE, f"liboracle_{prec}{'_san' if _SANITIZE else ''}.so")


def build(force: bool = False) -> None:
    """Compile both precisions with gcc.  -ffp-contract=off: no implicit FMA contraction;
    -mfma only lets the explicit fma()/fmaf() calls inline (the result is the same either way,
    fma is exactly specified)."""
    has_fma = False
    try:
        with open("/proc/cpuinfo") as f:
            has_fma = " fma " in f.read().replace("\n", " ")
    except OSError:
        pass
    for prec, define in (("f32", []), ("f64", ["-DORC_F64"])):
        out = _lib_path(prec)
        if not force and os.path.exists(out) and os.path.getmtime(out) >= os.path.getmtime(_SRC):
            continue
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
               "-Wall", "-Wno-unused-function"] + (["-mfma"] if has_fma else []) + define + \
              (["-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined"]
               if _SANITIZE else []) + \
              [_SRC, "-o", out + ".tmp", "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(out + ".tmp", out)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class Oracle:
    def __init__(self, precision: str = "f32"):
        assert precision in ("f32", "f64")
        build()
        self.precision = precision
        self.real = np.float32 if precision == "f32" else np.float64
        self._creal = C.c_float if precision == "f32" else C.c_double
        self.lib = C.CDLL(_lib_path(precision))
        assert self.lib.orc_real_bytes() == np.dtype(self.real).itemsize
        self.lib.orc_bin_sort.restype = C.c_int64
        self.lib.orc_mix64.restype = C.c_uint64
        self.lib.orc_mix64.argtypes = [C.c_uint64, C.c_uint64]

        class Cam(C.Structure):
            _fields_ = [("W", C.c_int32), ("H", C.c_int32), ("fx", self._creal), ("fy", self._creal),
                        ("cx", self._creal), ("cy", self._creal), ("Rcw", self._creal * 9),
                        ("tau", self._creal * 3), ("znear", self._creal), ("bg", self._creal * 3)]
        self._Cam = Cam

    # ---- helpers -------------------------------------------------------------------------
    def r(self, a):
        return np.ascontiguousarray(np.asarray(a), dtype=self.real)

    def cam(self, cam):
        c = self._Cam()
        c.W, c.H = int(cam.width), int(cam.height)
        # every camera scalar is first rounded to fp32 (the boundary type of the CUDA library)
        f = lambda v: float(np.float32(v))
        c.fx, c.fy, c.cx, c.cy, c.znear = f(cam.fx), f(cam.fy), f(cam.cx), f(cam.cy), f(cam.znear)
        R = np.asarray(cam.R, dtype=np.float32).reshape(9)
        t = np.asarray(cam.t, dtype=np.float32).reshape(3)
        bg = np.asarray(cam.bg, dtype=np.float32).reshape(3)
        for i in range(9):
            c.Rcw[i] = float(R[i])
        for i in range(3):
            c.tau[i] = float(t[i])
            c.bg[i] = float(bg[i])
        return c

    @staticmethod
    def grid(cam):
        return ((cam.width + 15) // 16, (cam.height + 15) // 16)

    # ---- O1 ------------------------------------------------------------------------------
    def preprocess(self, cam, sh_degree, means3D, scales, quats, opacities, sh):
        N = int(np.asarray(means3D).shape[0])
        K = (sh_degree + 1) ** 2
        mu, sc, q, op = self.r(means3D), self.r(scales), self.r(quats), self.r(opacities)
        shc = self.r(sh).reshape(N, K, 3)
        o = SimpleNamespace(
            means2D=np.zeros((N, 2), self.real), depths=np.zeros(N, self.real),
            conic_opacity=np.zeros((N, 4), self.real), rgb=np.zeros((N, 3), self.real),
            radii=np.zeros(N, np.int32), rect=np.zeros((N, 4), np.int32),
            tiles_touched=np.zeros(N, np.uint32), clamped=np.zeros(N, np.uint8))
        c = self.cam(cam)
        self.lib.orc_preprocess(C.byref(c), N, sh_degree, _ptr(mu), _ptr(sc), _ptr(q), _ptr(op), _ptr(shc),
                                _ptr(o.means2D), _ptr(o.depths), _ptr(o.conic_opacity), _ptr(o.rgb),
                                _ptr(o.radii), _ptr(o.rect), _ptr(o.tiles_touched), _ptr(o.clamped))
        return o

    # ---- O2 ------------------------------------------------------------------------------
    def bin_sort(self, cam, pre, tile_select=None):
        """tile_select: optional [T] mask (nonzero = bin this tile); None bins every tile."""
        N = pre.depths.shape[0]
        gx, gy = self.grid(cam)
        cap = int(pre.tiles_touched.astype(np.int64).sum())
        keys = np.zeros(max(cap, 1), np.uint64)
        gid = np.zeros(max(cap, 1), np.uint32)
        offs = np.zeros(gx * gy + 1, np.uint32)
        sel = None if tile_select is None else np.ascontiguousarray(tile_select, dtype=np.uint32)
        assert sel is None or sel.shape == (gx * gy,)
        c = self.cam(cam)
        P = int(self.lib.orc_bin_sort(C.byref(c), N, _ptr(self.r(pre.depths)), _ptr(pre.rect),
                                      _ptr(pre.tiles_touched), _ptr(sel), _ptr(keys), _ptr(gid), _ptr(offs)))
        assert P <= cap and (sel is not None or P == cap)
        return SimpleNamespace(P=P, keys_sorted=keys[:P].copy(), gid_sorted=gid[:P].copy(), tile_offsets=offs)

    # ---- O3 ------------------------------------------------------------------------------
    def sample(self, cam, tile_pct, pixel_mode, pix_rate=(1, 1), seed=0, err=None, render=None, target=None):
        H, W = cam.height, cam.width
        gx, gy = self.grid(cam)
        T = gx * gy
        qerr = np.zeros(H * W, np.uint32)
        score = np.zeros(T, np.uint64)
        tiles = np.zeros(T, np.uint32)
        tpo = np.zeros(T + 1, np.uint32)
        pix = np.zeros(H * W, np.uint32)
        kn = np.zeros(2, np.int32)
        e = None if err is None else self.r(err).reshape(H, W)
        rd = None if render is None else self.r(render).reshape(H, W, 3)
        tg = None if target is None else self.r(target).reshape(H, W, 3)
        assert e is not None or (rd is not None and tg is not None)
        c = self.cam(cam)
        self.lib.orc_sample(C.byref(c), _ptr(e), _ptr(rd), _ptr(tg), int(tile_pct[0]), int(tile_pct[1]),
                            int(pixel_mode), int(pix_rate[0]), int(pix_rate[1]), C.c_uint64(seed),
                            _ptr(qerr), _ptr(score), _ptr(tiles), _ptr(tpo), _ptr(pix), _ptr(kn))
        k, n = int(kn[0]), int(kn[1])
        return SimpleNamespace(k=k, n=n, qerr=qerr.reshape(H, W), tile_score=score, tiles=tiles[:k].copy(),
                               tile_pix_offsets=tpo[:k + 1].copy(), pix=pix[:n].copy())

    # ---- O4 ------------------------------------------------------------------------------
    def raster_fwd(self, cam, binned, pre, samp, margin_thr=2e-6):
        """margin[n,2]: smallest relative distance of a tested quantity to its threshold along the walk (forward
        decisions; forward + the 0.99 clamp that only the derivative sees).  flip_w[n]: the compositing weight that
        moves if every decision closer than margin_thr to its threshold is taken the other way."""
        n = samp.n
        o = SimpleNamespace(color=np.zeros((n, 3), self.real), T=np.zeros(n, self.real),
                            n_contrib=np.zeros(n, np.uint32), n_walked=np.zeros(n, np.uint32),
                            margin=np.ones((n, 2), self.real), flip_w=np.zeros(n, self.real))
        c = self.cam(cam)
        self.lib.orc_raster_fwd(C.byref(c), _ptr(binned.tile_offsets), _ptr(binned.gid_sorted),
                                _ptr(self.r(pre.means2D)), _ptr(self.r(pre.conic_opacity)), _ptr(self.r(pre.rgb)),
                                samp.k, _ptr(samp.tiles), _ptr(samp.tile_pix_offsets), _ptr(samp.pix),
                                _ptr(o.color), _ptr(o.T), _ptr(o.n_contrib), _ptr(o.n_walked), _ptr(o.margin),
                                self._creal(margin_thr), _ptr(o.flip_w))
        return o

    # ---- O5 ------------------------------------------------------------------------------
    def raster_bwd(self, cam, binned, pre, samp, fwd, dL_dcolor, want_abs=False):
        """want_abs: also return sum_abs[N,9] (fp64), the sum of |term| behind every gradient element in the
        order mean2D[2], conic[3], opacity, rgb[3]."""
        N = pre.means2D.shape[0]
        g = self.r(dL_dcolor).reshape(samp.n, 3)
        o = SimpleNamespace(dL_dmeans2D=np.zeros((N, 2), self.real), dL_dconic=np.zeros((N, 3), self.real),
                            dL_dopacity=np.zeros(N, self.real), dL_drgb=np.zeros((N, 3), self.real),
                            sum_abs=np.zeros((N, 9), np.float64) if want_abs else None)
        c = self.cam(cam)
        self.lib.orc_raster_bwd(C.byref(c), N, _ptr(binned.tile_offsets), _ptr(binned.gid_sorted),
                                _ptr(self.r(pre.means2D)), _ptr(self.r(pre.conic_opacity)), _ptr(self.r(pre.rgb)),
                                samp.k, _ptr(samp.tiles), _ptr(samp.tile_pix_offsets), _ptr(samp.pix),
                                _ptr(self.r(fwd.T)), _ptr(fwd.n_contrib), _ptr(g),
                                _ptr(o.dL_dmeans2D), _ptr(o.dL_dconic), _ptr(o.dL_dopacity), _ptr(o.dL_drgb),
                                _ptr(o.sum_abs))
        return o

    # ---- O6 ------------------------------------------------------------------------------
    def project_bwd(self, cam, sh_degree, means3D, scales, quats, sh, radii, clamped,
                    dL_dmeans2D, dL_dconic, dL_drgb):
        N = int(np.asarray(means3D).shape[0])
        K = (sh_degree + 1) ** 2
        o = SimpleNamespace(dL_dmeans3D=np.zeros((N, 3), self.real), dL_dscales=np.zeros((N, 3), self.real),
                            dL_dquats=np.zeros((N, 4), self.real), dL_dsh=np.zeros((N, K, 3), self.real))
        c = self.cam(cam)
        self.lib.orc_project_bwd(C.byref(c), N, sh_degree, _ptr(self.r(means3D)), _ptr(self.r(scales)),
                                 _ptr(self.r(quats)), _ptr(self.r(sh).reshape(N, K, 3)),
                                 _ptr(np.ascontiguousarray(radii, np.int32)),
                                 _ptr(np.ascontiguousarray(clamped, np.uint8)),
                                 _ptr(self.r(dL_dmeans2D)), _ptr(self.r(dL_dconic)), _ptr(self.r(dL_drgb)),
                                 _ptr(o.dL_dmeans3D), _ptr(o.dL_dscales), _ptr(o.dL_dquats), _ptr(o.dL_dsh))
        return o

    def render_dense(self, cam, binned, pre):
        img = np.zeros((cam.height, cam.width, 3), self.real)
        c = self.cam(cam)
        self.lib.orc_render_dense(C.byref(c), _ptr(binned.tile_offsets), _ptr(binned.gid_sorted),
                                  _ptr(self.r(pre.means2D)), _ptr(self.r(pre.conic_opacity)), _ptr(self.r(pre.rgb)),
                                  _ptr(img))
        return img

    # ---- O7: sparse supervision, Eq. 9-11, 472-481 Eq. 17-18 ----
    def loss_sparse(self, cam, samp, color, target, eps_l1=1e-3, eps_ncc=1e-6, eps_lam=1e-8):
        n, k = samp.n, samp.k
        col = self.r(color).reshape(n, 3)
        tg = self.r(target).reshape(cam.height, cam.width, 3)
        o = SimpleNamespace(dL_dcolor=np.zeros((n, 3), self.real), pix_err=np.zeros(n, self.real),
                            tile_stats=np.zeros((k, 3), self.real), loss=np.zeros(2, self.real))
        c = self.cam(cam)
        R = self._creal
        self.lib.orc_loss_sparse(C.byref(c), C.c_int(k), _ptr(samp.tile_pix_offsets), _ptr(samp.pix), _ptr(col), _ptr(tg),
                                 R(eps_l1), R(eps_ncc), R(eps_lam), _ptr(o.dL_dcolor), _ptr(o.pix_err),
                                 _ptr(o.tile_stats), _ptr(o.loss))
        return o

    # ---- O8: statistics forward, Eq. 12 ----
    def raster_stats(self, cam, binned, pre, samp, pix_err):
        N = pre.means2D.shape[0]
        o = SimpleNamespace(stats=np.zeros((N, 3), self.real), depth=np.zeros(samp.n, self.real))
        c = self.cam(cam)
        self.lib.orc_raster_stats(C.byref(c), C.c_int(N), _ptr(binned.tile_offsets), _ptr(binned.gid_sorted),
                                  _ptr(self.r(pre.means2D)), _ptr(self.r(pre.conic_opacity)), _ptr(self.r(pre.depths)),
                                  C.c_int(samp.k), _ptr(samp.tiles), _ptr(samp.tile_pix_offsets), _ptr(samp.pix),
                                  _ptr(self.r(pix_err)), _ptr(o.stats), _ptr(o.depth))
        return o

    # ---- O9: the paper's sampler and its maps, Eq. 3-4, 128-150 Eq. 7-8 ----
    def sample_paper(self, cam, E_half, age, n_pix, n_hard, n_stable, seed=0):
        """E_half: uint16 [H,W] fp16 bit patterns of the error map; age: uint16 [H,W]."""
        H, W = cam.height, cam.width
        gx, gy = self.grid(cam)
        T = gx * gy
        E = np.ascontiguousarray(E_half, np.uint16).reshape(H, W)
        A = np.ascontiguousarray(age, np.uint16).reshape(H, W)
        tiles = np.zeros(T, np.uint32)
        tpo = np.zeros(T + 1, np.uint32)
        pix = np.zeros(H * W, np.uint32)
        kn = np.zeros(2, np.int32)
        c = self.cam(cam)
        self.lib.orc_sample_paper(C.byref(c), _ptr(E), _ptr(A), C.c_int(n_pix), C.c_int(n_hard), C.c_int(n_stable),
                                  C.c_uint64(seed), _ptr(tiles), _ptr(tpo), _ptr(pix), _ptr(kn))
        k, n = int(kn[0]), int(kn[1])
        return SimpleNamespace(k=k, n=n, tiles=tiles[:k].copy(), tile_pix_offsets=tpo[:k + 1].copy(), pix=pix[:n].copy())

    def maps_update(self, cam, E_half, age, pix, pix_err, beta):
        """Returns the updated (E_half, age) copies (Eq. 3-4)."""
        E = np.ascontiguousarray(E_half, np.uint16).copy()
        A = np.ascontiguousarray(age, np.uint16).copy()
        px = np.ascontiguousarray(pix, np.uint32)
        er = np.ascontiguousarray(pix_err, np.float32)
        c = self.cam(cam)
        self.lib.orc_maps_update(C.byref(c), _ptr(E), _ptr(A), C.c_int(len(px)), _ptr(px), _ptr(er), C.c_float(beta))
        return E, A

    def float_to_half(self, f):
        self.lib.orc_float_to_half.restype = C.c_uint16
        return int(self.lib.orc_float_to_half(C.c_float(f)))

    # ---- small exported helpers (pinned individually) ---------------------------------------
    def quat_to_R(self, q):
        R = np.zeros(9, self.real)
        self.lib.orc_quat_to_R(_ptr(self.r(q)), _ptr(R))
        return R.reshape(3, 3)

    def cov3d(self, s, q):
        S = np.zeros(9, self.real)
        self.lib.orc_cov3d(_ptr(self.r(s)), _ptr(self.r(q)), _ptr(S))
        return S.reshape(3, 3)

    def sh_basis(self, d):
        B = np.zeros(16, self.real)
        self.lib.orc_sh_basis(_ptr(self.r(d)), _ptr(B))
        return B

    def mix64(self, seed, idx):
        return int(self.lib.orc_mix64(seed, idx))

    # ---- whole path --------------------------------------------------------------------------
    def pipeline(self, scene, dL_dcolor=None, backward=True, restrict=False):
        """preprocess -> bin_sort -> sample -> fwd -> (bwd) on a ``workloads.Scene``.  restrict=True
        (needs an error map): sample first, then bin only the selected tiles (R14)."""
        cam = scene.cam
        pre = self.preprocess(cam, scene.sh_degree, scene.means3D, scene.scales, scene.quats,
                              scene.opacities, scene.sh)
        if restrict and scene.err is not None:
            samp = self.sample(cam, scene.tile_pct, scene.pixel_mode, scene.pix_rate, scene.sample_seed,
                               err=scene.err)
            gx, gy = self.grid(cam)
            sel = np.zeros(gx * gy, np.uint32)
            sel[samp.tiles] = 1
            samp.tile_select = sel
            binned = self.bin_sort(cam, pre, tile_select=sel)
        else:
            binned = self.bin_sort(cam, pre)
            if scene.err is not None:
                samp = self.sample(cam, scene.tile_pct, scene.pixel_mode, scene.pix_rate, scene.sample_seed,
                                   err=scene.err)
            else:
                render = self.render_dense(cam, binned, pre)
                samp = self.sample(cam, scene.tile_pct, scene.pixel_mode, scene.pix_rate, scene.sample_seed,
                                   render=render, target=scene.target)
        fwd = self.raster_fwd(cam, binned, pre, samp)
        out = SimpleNamespace(pre=pre, binned=binned, samp=samp, fwd=fwd, rbwd=None, pbwd=None)
        if backward:
            g = dL_dcolor if dL_dcolor is not None else np.ones((samp.n, 3), np.float32)
            out.rbwd = self.raster_bwd(cam, binned, pre, samp, fwd, g)
            out.pbwd = self.project_bwd(cam, scene.sh_degree, scene.means3D, scene.scales, scene.quats, scene.sh,
                                        pre.radii, pre.clamped, out.rbwd.dL_dmeans2D, out.rbwd.dL_dconic,
                                        out.rbwd.dL_drgb)
        return out
