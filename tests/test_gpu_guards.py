"""Memory-safety checks of our own (compute-sanitizer is closed on this GPU pool, profiles/r2_sanitizers.md):

* out-of-bounds WRITES: every buffer the library writes (outputs, workspaces) is carved out of a larger allocation
  with 4 KiB canary zones on both sides, at the TIGHTEST capacities the ABI accepts (P_capacity = P exactly); the
  canaries must be intact after a whole step (projection, sampling, binning, forward, loss, statistics, backward,
  map update, LM solve);
* reads of UNINITIALISED memory: the same step is run with every buffer pre-filled with 0x00, 0xFF and 0x5A bytes
  (0xFF: NaN as fp32, 0xffffffff as an index); every deterministic output must be bit-identical across the three
  fills and equal to the oracle's, the atomically accumulated ones equal within the parity bars.
"""
import numpy as np
import pytest

import workloads
from helpers import dev, scene_dev, u32

pytestmark = pytest.mark.gpu

GUARD = 4096


class GuardedAllocator:
    """Stands in for torch.empty / torch.zeros: each tensor is the middle of a byte buffer whose first and last GUARD
    bytes (and, for `empty`, the payload too) hold `fill`."""

    def __init__(self, torch, fill):
        self.torch, self.fill, self.bufs = torch, fill, []
        self._empty, self._zeros = torch.empty, torch.zeros

    def _alloc(self, shape, dtype, device, zero):
        t = self.torch
        shape = (shape,) if isinstance(shape, int) else tuple(shape)
        item = t.empty((), dtype=dtype).element_size()
        nbytes = int(np.prod(shape, dtype=np.int64)) * item
        pad = (-nbytes) % 256
        raw = self._empty(GUARD + nbytes + pad + GUARD, dtype=t.uint8, device=device)
        raw.fill_(self.fill)
        body = raw[GUARD:GUARD + nbytes]
        if zero:
            body.zero_()
        self.bufs.append((raw, nbytes))
        return body.view(dtype).view(shape)

    def empty(self, *shape, dtype=None, device=None, **kw):
        shape = shape[0] if len(shape) == 1 else shape
        if device is None or self.torch.device(device).type != "cuda":
            return self._empty(shape, dtype=dtype, device=device, **kw)
        return self._alloc(shape, dtype or self.torch.float32, device, zero=False)

    def zeros(self, *shape, dtype=None, device=None, **kw):
        shape = shape[0] if len(shape) == 1 else shape
        if device is None or self.torch.device(device).type != "cuda":
            return self._zeros(shape, dtype=dtype, device=device, **kw)
        return self._alloc(shape, dtype or self.torch.float32, device, zero=True)

    def check(self):
        self.torch.cuda.synchronize()
        for i, (raw, nbytes) in enumerate(self.bufs):
            lo, hi = raw[:GUARD], raw[GUARD + nbytes:]
            assert bool((lo == self.fill).all()), f"buffer {i} ({nbytes} B): bytes written BEFORE its start"
            assert bool((hi == self.fill).all()), f"buffer {i} ({nbytes} B): bytes written PAST its end"
        return len(self.bufs)


def _step(torch, tgs, pk, sc, orc, fill, monkeypatch):
    """One whole step with guarded buffers pre-filled with `fill`; returns the outputs as numpy arrays."""
    ga = GuardedAllocator(torch, fill)
    with monkeypatch.context() as mp:
        mp.setattr(torch, "empty", ga.empty)
        mp.setattr(torch, "zeros", ga.zeros)
        step = pk.SparseRasterStep(tgs, sc.cam, sc.N, sc.sh_degree, orc.binned.P, want_keys=True)   # P_capacity = P exactly
        d = scene_dev(sc, torch)
        fw = step.forward(d.means3D, d.scales, d.quats, d.opacities, d.sh, sc.tile_pct, sc.pixel_mode, sc.pix_rate,
                          sc.sample_seed, err=dev(sc.err, torch))
        P, k, n = step.counts()
        npx = sc.cam.width * sc.cam.height
        target = dev(workloads.dl_dcolor(5, npx).reshape(sc.cam.height, sc.cam.width, 3) * 0.1 + 0.5, torch)
        lo = tgs.loss_sparse(sc.cam, step.samp, fw.color, target, n_capacity=n)
        so = tgs.raster_stats_sparse(sc.cam, step.pre.splats, step.binned, step.samp, lo.pix_err, n_capacity=n)
        bw = step.backward(lo.dL_dcolor)
        # the paper's sampler + maps on the same image, the LM solve on the step's gradients
        E = ga.empty((sc.cam.height, sc.cam.width), dtype=torch.int16, device="cuda")
        E.copy_((dev(np.abs(workloads.dl_dcolor(6, npx)[:, 0]).reshape(sc.cam.height, sc.cam.width), torch)).to(torch.float16).view(torch.int16))
        age = ga.zeros((sc.cam.height, sc.cam.width), dtype=torch.int16, device="cuda")
        sp = tgs.sample_paper(sc.cam, E, age, 25, 10, 8, seed=3)
        perr = ga.empty(sp.n, dtype=torch.float32, device="cuda")
        perr.copy_(dev(np.abs(workloads.dl_dcolor(7, sp.n)[:, 0]), torch))
        tgs.maps_update(sc.cam, E, age, sp, perr, 0.4)
        grads = {"means3D": bw.dL_dmeans3D[None], "scales": bw.dL_dscales[None], "quats": bw.dL_dquats[None],
                 "opacities": bw.dL_dopacities[None], "sh": bw.dL_dsh[None]}
        m = {k_: ga.zeros(tuple(g.shape[1:]), dtype=torch.float32, device="cuda") for k_, g in grads.items()}
        v = {k_: ga.zeros(tuple(g.shape[1:]), dtype=torch.float32, device="cuda") for k_, g in grads.items()}
        delta = tgs.lm_solve(sc.sh_degree, grads, m, v, t=1)
        nbuf = ga.check()
    out = dict(P=P, k=k, n=n, nbuf=nbuf,
               splats=step.pre.splats.cpu().numpy(), radii=step.pre.radii.cpu().numpy(),
               gid=u32(step.binned.gid_sorted)[:P], keys=step.binned.keys_sorted.cpu().numpy()[:P],
               offs=u32(step.binned.tile_offsets), tiles=u32(step.samp.tiles)[:k], pix=u32(step.samp.pix)[:n],
               color=fw.color[:n].cpu().numpy(), T=fw.T[:n].cpu().numpy(), nc=u32(fw.n_contrib)[:n],
               dLdc=lo.dL_dcolor[:n].cpu().numpy(), perr=lo.pix_err[:n].cpu().numpy(), loss=lo.loss.cpu().numpy(),
               E=E.cpu().numpy(), age=age.cpu().numpy(), ppix=u32(sp.pix)[:sp.n],
               stats=so.stats.cpu().numpy(), dsplats=bw.dL_dsplats.cpu().numpy(), dsh=bw.dL_dsh.cpu().numpy(),
               dmu=bw.dL_dmeans3D.cpu().numpy(), delta_mu=delta["means3D"].cpu().numpy(), delta_sh=delta["sh"].cpu().numpy())
    return out


@pytest.mark.parametrize("name", ["small_rot", "cfg2"])
def test_guards_and_uninitialised_memory(name, monkeypatch):
    import torch
    import oracle
    import paper_2606_15924_b200 as pk
    sc = {"small_rot": lambda: workloads.small_random_scene(7, 3000, 200, 136, sh_degree=3, bg=(0.1, 0.3, 0.2), spread=1.3,
                                                           log_scale=(-2.8, 0.6)),
          "cfg2": lambda: workloads.make(2)}[name]()
    orc = oracle.Oracle("f32").pipeline(sc, backward=False, restrict=True)
    tgs = pk.TGS(0)
    runs = [_step(torch, tgs, pk, sc, orc, fill, monkeypatch) for fill in (0x00, 0xFF, 0x5A)]
    a = runs[0]
    assert (a["P"], a["k"], a["n"]) == (orc.binned.P, orc.samp.k, orc.samp.n)
    assert np.array_equal(a["gid"], orc.binned.gid_sorted) and np.array_equal(a["pix"], orc.samp.pix)
    assert np.array_equal(a["offs"], orc.binned.tile_offsets)
    exact = ["P", "k", "n", "splats", "radii", "gid", "keys", "offs", "tiles", "pix", "color", "T", "nc", "dLdc", "perr", "loss",
             "E", "age", "ppix"]
    for b in runs[1:]:
        for key in exact:   # deterministic outputs: no dependence on what the buffers held before
            assert np.array_equal(np.asarray(a[key]), np.asarray(b[key]), equal_nan=True), f"{key} depends on uninitialised memory"
        for key in ("stats", "dsplats", "dsh", "dmu", "delta_mu", "delta_sh"):   # fp32 atomics: order differs run to run
            x, y = np.asarray(a[key], np.float64), np.asarray(b[key], np.float64)
            assert np.isfinite(y).all(), f"{key}: non-finite values with pre-filled buffers"
            scale = np.abs(x).max() + 1e-30
            assert np.abs(x - y).max() <= 2e-3 * scale, f"{key} depends on uninitialised memory"
    print(f"guards {name}: {a['nbuf']} guarded buffers intact under 3 fills, P = {a['P']} at P_capacity = P")
