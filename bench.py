#!/usr/bin/env python
"""bench.py -- one TurboGS sparse-raster step (all five C-ABI calls) on seeded synthetic scenes.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--pct P] [--impl tgs|reference]

A "step" is one pass of the whole hot path over one view: tgs_preprocess -> tgs_bin_sort ->
tgs_sample -> tgs_raster_fwd_sparse -> tgs_raster_bwd_sparse (raster + projection halves).

Headline workload (value / ms_per_step / roofline / e2e / cpu_baseline) = BASELINE.json configs[3], the largest
single-GPU configuration (3 M Gaussians, 1957x1091, dense mask).  The same run also times configs[0], [1], [2] and the
six points of the configs[4] sampling-rate sweep into `per_config` (N = 1 only).  `--config C` moves the headline.
Prints ONE JSON line (rank 0).  Multi-GPU = independent replicas, no data-path collective (DESIGN.md "Multi-GPU":
replicas only); the barrier / max-over-ranks timing uses NCCL.
"""
from __future__ import annotations

import argparse
import gc
import json
import os
import statistics
import sys
import threading
import time
from types import SimpleNamespace

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "sampled px/s fwd+bwd raster and Gaussian-px evals/s; % of HBM/FP32 roofline"
UNIT = "sampled_px/s"
HEADLINE_CONFIG = 4  # 1-based: BASELINE.json configs[3]

# Algorithmic FP32 flops per Gaussian-pixel evaluation, counted from the oracle's arithmetic
# (DESIGN.md "Roofline accounting"): every visited (pixel, Gaussian) costs the power / exp / alpha
# test; a composited one additionally the blend (forward) or the nine partial derivatives (backward).
FWD_FLOPS_WALK, FWD_FLOPS_BLEND = 15, 10
BWD_FLOPS_WALK, BWD_FLOPS_BLEND = 15, 64
SM_COUNT, FP32_LANES, SM_MAX_GHZ = 148, 128, 1.965
FP32_PEAK_TFLOPS = SM_COUNT * FP32_LANES * 2 * SM_MAX_GHZ / 1e3  # 74.4: FMA = 2 flop, nominal max clock
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r2_traffic.csv")  # dram bytes per launch from the committed ncu --set full captures


def load_scene(cfg: int, pct: int):
    import workloads
    return workloads.make(cfg, pct=pct) if cfg == 5 else workloads.make(cfg)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0}, "fallback"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.005):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.reasons = index, period_s, [], set()
        self.stop_flag = threading.Event()
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        while not self.stop_flag.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self):
        return {"sm_mhz": statistics.median(self.samples) if self.samples else None,
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# --------------------------------------------------------------------------------------------
# The CPU oracle, as it stands, on a BOUNDED sample of the workload (cpu_baseline and --impl reference).
class OracleSample:
    """One `step()` = the oracle's whole path over 1/den of the workload, single thread:
    projection (O1) and projection backward (O6) on the first N/den Gaussians, the sampler (O3) on the whole error
    map, and binning (O2) + sparse forward (O4) + backward (O5) on every den-th sampled tile.  Gaussians are i.i.d. and
    the tiles are taken at a fixed stride over the image, so a step costs ~1/den of the full step and processes ~n/den
    sampled pixels: the rate n_s / t is the oracle's rate on the workload.  den = 1 is the whole workload."""

    def __init__(self, scene, den: int):
        import oracle
        import workloads
        self.o, self.scene, self.den = oracle.Oracle("f32"), scene, max(1, int(den))
        o, sc, cam = self.o, scene, scene.cam
        if sc.err is None:  # config 1: mask from the residual of a dense render against the target
            pre = o.preprocess(cam, sc.sh_degree, sc.means3D, sc.scales, sc.quats, sc.opacities, sc.sh)
            sc.err = np.abs(o.render_dense(cam, o.bin_sort(cam, pre), pre) - sc.target).sum(axis=2).astype(np.float32)
        self.pre = o.preprocess(cam, sc.sh_degree, sc.means3D, sc.scales, sc.quats, sc.opacities, sc.sh)  # untimed set-up
        full = o.sample(cam, sc.tile_pct, sc.pixel_mode, sc.pix_rate, sc.sample_seed, err=sc.err)
        its = np.arange(0, full.k, self.den)
        off = full.tile_pix_offsets.astype(np.int64)
        cnt = (off[its + 1] - off[its])
        self.sub = SimpleNamespace(k=len(its), n=int(cnt.sum()), tiles=full.tiles[its].copy(),
                                   tile_pix_offsets=np.concatenate([[0], np.cumsum(cnt)]).astype(np.uint32),
                                   pix=np.concatenate([full.pix[off[i]:off[i + 1]] for i in its]).copy())
        self.sel = np.zeros(cam.num_tiles, np.uint32)
        self.sel[self.sub.tiles] = 1
        self.ng = max(1, sc.N // self.den)
        self.g = workloads.dl_dcolor(0, self.sub.n)
        self.n_full, self.k_full = full.n, full.k

    def step(self):
        o, sc, cam, m = self.o, self.scene, self.scene.cam, self.ng
        t0 = time.perf_counter()
        o.preprocess(cam, sc.sh_degree, sc.means3D[:m], sc.scales[:m], sc.quats[:m], sc.opacities[:m], sc.sh[:m])
        o.sample(cam, sc.tile_pct, sc.pixel_mode, sc.pix_rate, sc.sample_seed, err=sc.err)
        b = o.bin_sort(cam, self.pre, tile_select=self.sel)
        fw = o.raster_fwd(cam, b, self.pre, self.sub)
        rb = o.raster_bwd(cam, b, self.pre, self.sub, fw, self.g)
        o.project_bwd(cam, sc.sh_degree, sc.means3D[:m], sc.scales[:m], sc.quats[:m], sc.sh[:m], self.pre.radii[:m],
                      self.pre.clamped[:m], rb.dL_dmeans2D[:m], rb.dL_dconic[:m], rb.dL_drgb[:m])
        return time.perf_counter() - t0

    def describe(self, nsteps, total_s):
        return (f"{nsteps} step(s), each the oracle's whole path over 1/{self.den} of the workload ({self.sub.k} of {self.k_full} "
                f"sampled tiles at stride {self.den} = {self.sub.n} sampled pixels, {self.ng} of {self.scene.N} Gaussians through "
                f"projection and its backward), single thread, {total_s:.1f} s")


def oracle_den(scene, target_s: float) -> int:
    """Stride that makes one oracle step cost about target_s (measured rates of the oracle on these workloads:
    ~4e7 Gaussian-pixel evaluations/s; the dense config is ~1.8e9 evaluations fwd + bwd)."""
    est_full = {1: 0.05, 2: 1.1, 3: 3.0, 4: 52.0, 5: 30.0}.get(int(scene.extra.get("config", 0)), 10.0)
    if scene.extra.get("config") == 5:
        est_full = 4.0 + 26.0 * scene.tile_pct[0] / scene.tile_pct[1]
    return max(1, int(round(est_full / target_s)))


def run_reference(args):
    """--impl reference: the oracle timed on the host cores (this tier's reference arm), a bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    scene = load_scene(args.config, args.pct)
    scene.extra["config"] = args.config
    smp = OracleSample(scene, oracle_den(scene, 1.0))
    times = []
    for i in range(args.warmup + args.steps):
        dt = smp.step()
        if i >= args.warmup:
            times.append(dt)
    total = sum(times)
    val = smp.sub.n * len(times) / total
    cfg = workload_config(scene, args, None, smp.k_full, smp.n_full)
    cfg["l2"] = "n/a (CPU)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": cfg,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": smp.describe(len(times), total)},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_config(scene, args, P, k, n, cfg_index=None):
    c = (cfg_index if cfg_index is not None else args.config) - 1
    return {"workload": f"BASELINE.json configs[{c}] ({scene.name})", "gaussians": scene.N,
            "sh_degree": scene.sh_degree, "image": [scene.cam.width, scene.cam.height],
            "tiles": scene.cam.num_tiles, "tile_pct": list(scene.tile_pct), "binning": "sampled tiles only (tile_select)",
            "gradients": "sparse: touched mask + rows of the touched Gaussians (tgs_raster_bwd_sparse `touched`, the update mask of tgs_lm_solve)",
            "pixel_mode": "all" if scene.pixel_mode == 0 else "bernoulli_err", "pairs_P": None if P is None else int(P),
            "sampled_tiles_k": int(k), "sampled_pixels_n": int(n), "parallelism": f"replicas x{args.gpus}"}


# --------------------------------------------------------------------------------------------
class GpuWorkload:
    """One config resident on the device: pinned host inputs, device inputs, the pre-allocated step, work counts."""

    def __init__(self, tg, scene, dev):
        import torch
        import paper_2606_15924_b200 as pk
        import workloads
        self.tg, self.scene, self.dev, self.torch = tg, scene, dev, torch
        cam = scene.cam
        self.H = {k: torch.from_numpy(np.ascontiguousarray(getattr(scene, k))).pin_memory()
                  for k in ("means3D", "scales", "quats", "opacities", "sh")}
        if scene.err is None:  # config 1: its mask comes from the residual of a dense render; the bench uses a fixed seeded error map
            err_np = workloads.blob_error_map(np.random.default_rng(0), cam.width, cam.height, 8)
        else:
            err_np = scene.err
        self.H["err"] = torch.from_numpy(np.ascontiguousarray(err_np)).pin_memory()
        self.D = {k: v.to(dev) for k, v in self.H.items()}
        D = self.D
        # size the pair buffers: one preprocess, then P <= sum of tiles touched (plumbing, untimed)
        pre = tg.preprocess(cam, scene.sh_degree, D["means3D"], D["scales"], D["quats"], D["opacities"], D["sh"])
        rw = pre.splats[:, 10:12].contiguous().view(torch.int32)
        P_est = int((((rw[:, 0] >> 16) - (rw[:, 0] & 0xffff)).long() * ((rw[:, 1] >> 16) - (rw[:, 1] & 0xffff)).long()).sum())
        del pre, rw
        self.P_est = P_est
        self.step = pk.SparseRasterStep(tg, cam, scene.N, scene.sh_degree, P_est + 1024, want_walked=True)
        self.fwd()
        self.P, self.k, self.n = self.step.counts()
        n = self.n
        self.walked = int(self.step.fwd.n_walked[:n].long().sum())
        self.blended = int(self.step.fwd.n_blended[:n].long().sum())
        self.replayed = int(self.step.fwd.n_contrib[:n].long().sum())
        self.g_host = torch.from_numpy(workloads.dl_dcolor(0, n) / np.float32(max(n, 1))).pin_memory()
        self.g_dev = torch.zeros((cam.width * cam.height, 3), device=dev)
        self.g_dev[:n] = self.g_host.to(dev)
        self.step.fwd.n_walked = None   # work counters are not part of the timed step
        self.step.fwd.n_blended = None

    def fwd(self, D=None):
        D, sc = D or self.D, self.scene
        self.step.forward(D["means3D"], D["scales"], D["quats"], D["opacities"], D["sh"], sc.tile_pct, sc.pixel_mode,
                          sc.pix_rate, sc.sample_seed, err=D["err"])

    def full_step(self):
        # gradients as (touched mask, rows of the touched Gaussians): what tgs_lm_solve consumes (tgs.h, sparse gradients)
        self.fwd()
        self.step.backward(self.g_dev, sparse=True)

    # ---- the step, launched call by call, CUDA events around each step, L2 flushed between steps ----
    def time_eager(self, steps, warmup, flush, rep, sampler=None):
        torch = self.torch
        for _ in range(max(warmup, 3)):
            self.full_step()
        rep.barrier()
        if sampler is not None:
            sampler.start()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        l0 = self.tg.launch_count()
        rep.barrier()
        for s, e in ev:
            flush.fill_(1.0)
            s.record()
            self.full_step()
            e.record()
        rep.barrier()
        launches = self.tg.launch_count() - l0
        if sampler is not None:
            sampler.stop_flag.set()
            sampler.join()
        return rep.max_over_ranks(sum(s.elapsed_time(e) for s, e in ev)) / steps, launches

    # ---- the same step replayed from a CUDA graph (every call only enqueues; sizes are read on the device) ----
    def time_graph(self, steps, flush, rep):
        torch = self.torch
        try:
            gs = torch.cuda.Stream()
            gs.wait_stream(torch.cuda.current_stream())
            cg = torch.cuda.CUDAGraph()
            with torch.cuda.stream(gs):
                with torch.cuda.graph(cg, stream=gs):
                    self.full_step()
            torch.cuda.current_stream().wait_stream(gs)
            for _ in range(3):
                cg.replay()
            rep.barrier()
            gev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
            for s_, e_ in gev:
                flush.fill_(1.0)
                s_.record()
                cg.replay()
                e_.record()
            rep.barrier()
            ms = rep.max_over_ranks(sum(s_.elapsed_time(e_) for s_, e_ in gev)) / steps
            del cg
            return ms
        except Exception as ex:  # without a capture the eagerly launched step is the headline
            return f"capture failed: {ex}"

    # ---- per-call breakdown (separate pass; events between the calls) ----
    def time_calls(self, steps, flush):
        torch, tg, st, sc, D = self.torch, self.tg, self.step, self.scene, self.D
        cam = sc.cam
        names = ["preprocess", "sample", "bin_sort", "raster_fwd", "raster_bwd", "project_bwd"]
        acc = {k_: 0.0 for k_ in names}
        for _ in range(steps):
            flush.fill_(1.0)
            e_ = [torch.cuda.Event(enable_timing=True) for _ in range(7)]
            e_[0].record()
            tg.preprocess(cam, sc.sh_degree, D["means3D"], D["scales"], D["quats"], D["opacities"], D["sh"], out=st.pre)
            e_[1].record()
            tg.sample(cam, sc.tile_pct, sc.pixel_mode, sc.pix_rate, sc.sample_seed, err=D["err"], out=st.samp,
                      workspace=st.ws_sample, sync=False)
            e_[2].record()
            tg.bin_sort(cam, st.pre.splats, st.P_capacity, out=st.binned, workspace=st.ws_sort, sync=False,
                        tile_select=st.samp.tile_select)
            e_[3].record()
            tg.raster_fwd_sparse(cam, st.pre.splats, st.binned, st.samp, out=st.fwd)
            e_[4].record()
            tg.raster_bwd_sparse(cam, sc.sh_degree, st.pre.splats, st.binned, st.samp, st.fwd, self.g_dev, project=False,
                                 out=st.bwd)
            e_[5].record()
            tg.raster_bwd_sparse(cam, sc.sh_degree, st.pre.splats, st.binned, st.samp, st.fwd, self.g_dev, D["means3D"],
                                 D["scales"], D["quats"], D["sh"], st.pre.radii, st.pre.clamped, project=True, out=st.bwd,
                                 sparse=True)
            e_[6].record()
            torch.cuda.synchronize()
            d = [e_[i].elapsed_time(e_[i + 1]) for i in range(6)]
            for nm, v in zip(names[:5], d[:5]):
                acc[nm] += v
            acc["project_bwd"] += max(d[5] - d[4], 0.0)  # second call = raster + projection
        return {k_: v / steps for k_, v in acc.items()}

    def kernels(self, per_call_ms, fp32_peak, hbm_gbs):
        sc, cam = self.scene, self.scene.cam
        fwd_flops = FWD_FLOPS_WALK * self.walked + FWD_FLOPS_BLEND * self.blended
        bwd_flops = BWD_FLOPS_WALK * self.replayed + BWD_FLOPS_BLEND * self.blended
        K = (sc.sh_degree + 1) ** 2
        hbm_bytes = {"preprocess": sc.N * (4 * (11 + 3 * K) + 48 + 5),
                     "project_bwd": sc.N * (4 * (10 + 3 * K) + 48 + 5 + 4 * (11 + 3 * K)),
                     # rect/depth words of every record, then per emitted pair: segment write + read, gid_sorted write
                     "bin_sort": sc.N * 16 + self.P * (8 + 8 + 4) + cam.num_tiles * 12}
        kernels = {
            "raster_fwd": {"bound": "alu", "achieved": fwd_flops / (per_call_ms["raster_fwd"] * 1e-3) / 1e12,
                           "peak": fp32_peak, "unit": "TFLOP/s"},
            "raster_bwd": {"bound": "alu", "achieved": bwd_flops / (per_call_ms["raster_bwd"] * 1e-3) / 1e12,
                           "peak": fp32_peak, "unit": "TFLOP/s"},
        }
        for nm in ("preprocess", "project_bwd", "bin_sort"):
            kernels[nm] = {"bound": "hbm", "achieved": hbm_bytes[nm] / (per_call_ms[nm] * 1e-3) / 1e9,
                           "peak": hbm_gbs, "unit": "GB/s"}
        kernels["bin_sort"]["note"] = "a call of several dependent kernels (launch list in profiles/), not one kernel"
        for v in kernels.values():
            v["frac"] = v["achieved"] / v["peak"]
        return kernels

    def work(self, per_call_ms):
        return {"fwd_evals": self.walked, "bwd_evals": self.replayed, "blended": self.blended,
                "fwd_evals_per_s": self.walked / (per_call_ms["raster_fwd"] * 1e-3),
                "bwd_evals_per_s": self.replayed / (per_call_ms["raster_bwd"] * 1e-3),
                "raster_px_per_s": self.n / ((per_call_ms["raster_fwd"] + per_call_ms["raster_bwd"]) * 1e-3)}


def measure_side_config(tg, cfg, pct, args, dev, flush, rep, fp32_peak, hbm_gbs):
    """One entry of `per_config`: the step (graph replay and eager), the per-call split, work and roofline fractions."""
    scene = load_scene(cfg, pct)
    w = GpuWorkload(tg, scene, dev)
    steps = min(args.steps, 10)
    eager_ms, _ = w.time_eager(steps, 3, flush, rep)
    graph_ms = w.time_graph(steps, flush, rep)
    calls = w.time_calls(steps, flush)
    ms = graph_ms if isinstance(graph_ms, float) else eager_ms
    kern = w.kernels(calls, fp32_peak, hbm_gbs)
    out = {"workload": f"BASELINE.json configs[{cfg - 1}] ({scene.name})", "tile_pct": scene.tile_pct[0] * 100 // scene.tile_pct[1],
           "P": w.P, "k": w.k, "n": w.n, "ms_per_step": ms, "ms_per_step_eager": eager_ms, "px_per_s": w.n / (ms * 1e-3),
           "per_call_ms": {k_: round(v, 5) for k_, v in calls.items()},
           "raster_fwd_frac": kern["raster_fwd"]["frac"], "raster_bwd_frac": kern["raster_bwd"]["frac"],
           "bin_sort_hbm_frac": kern["bin_sort"]["frac"], "work": w.work(calls)}
    del w
    gc.collect()
    import torch
    torch.cuda.empty_cache()
    return out


def read_traffic(config, kernel):
    if not os.path.exists(TRAFFIC_CSV):
        return None
    with open(TRAFFIC_CSV) as f:
        for ln in f.read().splitlines()[1:]:
            c_, k_, b_ = ln.split(",")[:3]
            if int(c_) == config and k_ == kernel:
                return float(b_)
    return None


def run_tgs(args):
    import torch
    import paper_2606_15924_b200 as pk
    import workloads

    from paper_2606_15924_b200.replicas import Replicas
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    rep = Replicas("nccl", dev)  # replicas only: barrier + max / sum over ranks, no data-path collective
    world, rank = rep.world, rep.rank

    scene = workloads.orbit_view(load_scene(args.config, args.pct), rep.view_seed(0))  # one view per rank, rank 0: the config's own
    scene.extra["config"] = args.config
    cam = scene.cam
    tg = pk.TGS(local)
    w = GpuWorkload(tg, scene, dev)
    step, H, D, n, k, P = w.step, w.H, w.D, w.n, w.k, w.P
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)  # 256 MiB > 126 MB L2
    barrier = rep.barrier
    peaks, peak_src = measured_peaks()

    # measured FFMA-only peak (tgs_fp32_peak): the roofline denominator of the raster kernels
    fp32_peak_measured = tg.fp32_peak(5)

    # ---- timed region: K steps, each bracketed by CUDA events, L2 flushed between steps ----
    sampler = ClockSampler(local)
    eager_ms, launches = w.time_eager(args.steps, args.warmup, flush, rep, sampler)
    n_total = rep.sum_over_ranks(n)
    graph_ms = w.time_graph(args.steps, flush, rep)
    launch_mode = "eager launches"
    step_ms = eager_ms
    if isinstance(graph_ms, float):
        # the step a user runs in a training loop: the same kernels, launched by one graph replay
        launch_mode = "cuda graph replay of the five calls (eager launches timed beside it)"
        step_ms = graph_ms
    value = n_total / (step_ms * 1e-3)
    per_call_ms = w.time_calls(args.steps, flush)

    next_rows = None
    if not args.step_only:
        next_rows = measure_next_rows(tg, w, args, dev, flush, world, fp32_peak_measured, peaks)

    # ---- roofline of the dominant kernel ----
    kernels = w.kernels(per_call_ms, fp32_peak_measured, peaks["hbm_gbs"])
    # dominant KERNEL of the step (bin_sort and sample are calls of several shorter kernels; profiles/ has the
    # launch list that shows it; their call-level figures are in `kernels` / `per_call_ms`)
    dominant = max(("raster_fwd", "raster_bwd", "preprocess", "project_bwd"), key=lambda k_: per_call_ms[k_])
    roof = dict(kernels[dominant])
    roof.update({"kernel": dominant + "_kernel", "traffic": read_traffic(args.config, dominant), "ms": per_call_ms[dominant],
                 "peak_nominal": FP32_PEAK_TFLOPS if roof["bound"] == "alu" else None,
                 "peak_source": ("measured: tgs_fp32_peak (FFMA-only kernel, best of 5, CUDA events); nominal = 148 SM x 128 "
                                 "lanes x 2 flop x 1.965 GHz" if roof["bound"] == "alu"
                                 else f"MEASURED_PEAKS.json hbm_gbs ({peak_src})"),
                 "algorithmic_work": ("flops = 15 x walked + 10 x blended (fwd) / 15 x replayed + 64 x blended (bwd) "
                                      "(pixel, Gaussian) evaluations, DESIGN.md 'Roofline accounting'"
                                      if roof["bound"] == "alu" else "bytes per Gaussian, DESIGN.md 'Kernels'")})

    # ---- end to end: host buffers in, host gradients out, copies inside the timed region ----
    Hout = {k_: torch.empty(v.shape, dtype=v.dtype).pin_memory() for k_, v in
            (("dL_dmeans3D", step.bwd.dL_dmeans3D), ("dL_dscales", step.bwd.dL_dscales), ("dL_dquats", step.bwd.dL_dquats),
             ("dL_dopacities", step.bwd.dL_dopacities), ("dL_dsh", step.bwd.dL_dsh))}
    g_pin = torch.zeros((cam.width * cam.height, 3)).pin_memory()
    g_pin[:n] = w.g_host
    g_dev = w.g_dev
    h2d = sum(v.numel() * v.element_size() for v in H.values()) + n * 12
    d2h = sum(v.numel() * v.element_size() for v in Hout.values())

    def e2e_step():
        for k_, v in H.items():
            D[k_].copy_(v, non_blocking=True)
        g_dev[:n].copy_(g_pin[:n], non_blocking=True)
        w.fwd()
        step.backward(g_dev)   # dense gradients: every row is written, every row is copied back
        for k_, v in Hout.items():
            v.copy_(getattr(step.bwd, k_), non_blocking=True)

    for _ in range(3):
        e2e_step()
    barrier()
    es, ee = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    es.record()
    for _ in range(args.steps):
        e2e_step()
    ee.record()
    barrier()
    e2e_serial_ms = rep.max_over_ranks(es.elapsed_time(ee))

    # the same end-to-end step, pipelined the way a training loop would: the H2D copy of step i+1 (copy stream, second
    # set of device inputs) and the D2H copy of step i-1 (output stream, staged gradients) overlap the compute of step i.
    # Every step still copies all of its inputs in and all of its gradients out.
    comp, cs, os_ = torch.cuda.current_stream(), torch.cuda.Stream(), torch.cuda.Stream()
    Dsets = [D, {k_: torch.empty_like(v) for k_, v in D.items()}]
    gsets = [g_dev, torch.zeros_like(g_dev)]
    stage = [{k_: torch.empty_like(getattr(step.bwd, k_)) for k_ in Hout} for _ in range(2)]
    mk = lambda: [torch.cuda.Event(), torch.cuda.Event()]
    ev_in, ev_in_free, ev_out, ev_out_free = mk(), mk(), mk(), mk()

    def pipelined(nsteps):
        for i in range(nsteps):
            j = i & 1
            with torch.cuda.stream(cs):
                if i >= 2:
                    cs.wait_event(ev_in_free[j])
                for k_, v in H.items():
                    Dsets[j][k_].copy_(v, non_blocking=True)
                gsets[j][:n].copy_(g_pin[:n], non_blocking=True)
                ev_in[j].record(cs)
            comp.wait_event(ev_in[j])
            w.fwd(Dsets[j])
            step.backward(gsets[j])
            ev_in_free[j].record(comp)
            if i >= 2:
                comp.wait_event(ev_out_free[j])
            for k_ in Hout:
                stage[j][k_].copy_(getattr(step.bwd, k_), non_blocking=True)
            ev_out[j].record(comp)
            with torch.cuda.stream(os_):
                os_.wait_event(ev_out[j])
                for k_, v in Hout.items():
                    v.copy_(stage[j][k_], non_blocking=True)
                ev_out_free[j].record(os_)
        comp.wait_stream(os_)

    pipelined(4)
    barrier()
    es.record()
    pipelined(args.steps)
    ee.record()
    barrier()
    e2e_ms = rep.max_over_ranks(es.elapsed_time(ee))
    e2e_val = n_total * args.steps / (e2e_ms * 1e-3)
    # what arrived on the host is the last step's gradient (atomics reorder sums: compare with a tolerance)
    assert torch.allclose(Hout["dL_dsh"], step.bwd.dL_dsh.cpu(), rtol=1e-3, atol=1e-6), "pipelined e2e: host gradients differ"
    del Dsets, gsets, stage, Hout, g_pin

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": step_ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": dict(workload_config(scene, args, P, k, n), l2="flushed between steps (256 MiB write)", launch=launch_mode),
            "clocks": sampler.summary(),
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "ms_per_step_serial": e2e_serial_ms / args.steps,
                    "how": "pinned host -> device copies of all inputs and device -> pinned host copies of all gradients every step; "
                           "copies of neighbouring steps overlap the compute (3 streams, double-buffered); serial = one stream",
                    "ms_per_step": e2e_ms / args.steps},
            "gpu_launches": int(launches),
            "roofline": roof,
            "ms_per_step_cuda_graph": graph_ms, "ms_per_step_eager": eager_ms,
            "per_call_ms": per_call_ms,
            "next_rows": next_rows,
            "kernels": kernels,
            "work": w.work(per_call_ms)}

    # ---- the other BASELINE.json configs and the sampling-rate sweep, same run (N = 1 only) ----
    if world == 1 and not args.no_per_config:
        del w, step, H, D, g_dev
        gc.collect()
        torch.cuda.empty_cache()
        per = {}
        for cfg in (1, 2, 3, 4):
            if cfg != args.config:
                per[f"configs[{cfg - 1}]"] = measure_side_config(tg, cfg, 0, args, dev, flush, rep, fp32_peak_measured, peaks["hbm_gbs"])
        sweep = []
        for pct in workloads.SWEEP_PCTS:
            sweep.append(measure_side_config(tg, 5, pct, args, dev, flush, rep, fp32_peak_measured, peaks["hbm_gbs"]))
        xs = np.array([s_["tile_pct"] for s_ in sweep], np.float64)
        ys = np.array([s_["ms_per_step"] for s_ in sweep], np.float64)
        slope, icpt = np.polyfit(xs, ys, 1)
        per["configs[4] sweep"] = {"points": sweep,
                                   "fit_ms": {"intercept": float(icpt), "per_pct": float(slope),
                                              "note": "least-squares line through the six points; north_star wants time near-linear in the sampled-tile fraction"},
                                   "ratio_5pct_over_100pct": float(ys[0] / ys[-1])}
        line["per_config"] = per

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        smp = OracleSample(scene, oracle_den(scene, 4.0))
        times = [smp.step() for _ in range(4)]
        line["cpu_baseline"] = {"value": smp.sub.n * len(times) / sum(times), "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": smp.describe(len(times), sum(times)), "host_cores_available": os.cpu_count()}
    if rank == 0:
        print(json.dumps(line))
    rep.close()


def measure_next_rows(tg, w, args, dev, flush, world, fp32_peak_measured, peaks):
    """SURVEY.md 8f rows timed beside the five-call step (not part of `value`)."""
    import torch
    scene, st, cam, n, k = w.scene, w.step, w.scene.cam, w.n, w.k
    # f1: the fused sparse loss between forward and backward
    target_dev = torch.rand((cam.height, cam.width, 3), device=dev, generator=torch.Generator(device=dev).manual_seed(0))
    sn = SimpleNamespace(k=k, n=n, tile_pix_offsets=st.samp.tile_pix_offsets, pix=st.samp.pix)
    lo = tg.loss_sparse(cam, sn, st.fwd.color, target_dev, n_capacity=cam.width * cam.height)
    la, lb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    loss_ms = 0.0
    for _ in range(args.steps):
        flush.fill_(1.0)
        la.record()
        tg.loss_sparse(cam, sn, st.fwd.color, target_dev, out=lo)
        lb.record()
        torch.cuda.synchronize()
        loss_ms += la.elapsed_time(lb)
    loss_ms /= args.steps
    # f3: the statistics forward (E_i, D_i, W_i, expected depth), fed with the loss kernel's per-pixel error
    so = tg.raster_stats_sparse(cam, st.pre.splats, st.binned, st.samp, lo.pix_err, n_capacity=cam.width * cam.height)
    stats_ms = 0.0
    for _ in range(args.steps):
        flush.fill_(1.0)
        la.record()
        tg.raster_stats_sparse(cam, st.pre.splats, st.binned, st.samp, lo.pix_err, out=so)
        lb.record()
        torch.cuda.synchronize()
        stats_ms += la.elapsed_time(lb)
    stats_ms /= args.steps

    # f2: the paper's own regime -- N_pix = 25 pixels (r = 10 %) in EVERY tile with the settings of its
    # Tab. 6: r_hard = 0.4, r_stable = 0.3, 0.3 "mixed" remainder, beta = 0.4 -- sampler, binning of
    # all tiles, sparse forward / backward / statistics on those lists, map updates
    paper = None
    if world == 1:
        gE = torch.Generator(device=dev).manual_seed(1)
        E_half = (torch.rand((cam.height, cam.width), device=dev, generator=gE) ** 3).to(torch.float16).view(torch.int16)
        age = torch.randint(0, 50, (cam.height, cam.width), device=dev, generator=gE, dtype=torch.int32).to(torch.int16)
        sp = tg.sample_paper(cam, E_half, age, 25, 10, 8, seed=1)
        bp = tg.bin_sort(cam, st.pre.splats, w.P_est + 1024, workspace=st.ws_sort, sync=True)
        fp = tg.raster_fwd_sparse(cam, st.pre.splats, bp, sp)
        gp = torch.randn((sp.n, 3), device=dev, generator=gE) / sp.n
        sop = tg.raster_stats_sparse(cam, st.pre.splats, bp, sp, lo.pix_err)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(7)]
        accp = [0.0] * 6
        for _ in range(args.steps):
            flush.fill_(1.0)
            ev[0].record()
            tg.sample_paper(cam, E_half, age, 25, 10, 8, seed=1, out=sp, workspace=st.ws_sample, sync=False)
            ev[1].record()
            tg.bin_sort(cam, st.pre.splats, w.P_est + 1024, out=bp, workspace=st.ws_sort, sync=False)
            ev[2].record()
            tg.raster_fwd_sparse(cam, st.pre.splats, bp, sp, out=fp)
            ev[3].record()
            tg.raster_bwd_sparse(cam, scene.sh_degree, st.pre.splats, bp, sp, fp, gp, project=False, out=st.bwd)
            ev[4].record()
            tg.maps_update(cam, E_half, age, sp, lo.pix_err, 0.4)
            ev[5].record()
            tg.raster_stats_sparse(cam, st.pre.splats, bp, sp, lo.pix_err, out=sop)
            ev[6].record()
            torch.cuda.synchronize()
            for i_ in range(6):
                accp[i_] += ev[i_].elapsed_time(ev[i_ + 1])
        paper = {"n_pix_per_tile": 25, "n_hard": 10, "n_stable": 8, "beta": 0.4, "sampled_pixels_n": int(sp.n), "pairs_P_all_tiles": int(bp.P),
                 "sample_paper_ms": accp[0] / args.steps, "bin_sort_all_tiles_ms": accp[1] / args.steps,
                 "raster_fwd_ms": accp[2] / args.steps, "raster_bwd_ms": accp[3] / args.steps,
                 "maps_update_ms": accp[4] / args.steps, "raster_stats_ms": accp[5] / args.steps,
                 "raster_px_per_s": sp.n / ((accp[2] + accp[3]) / args.steps * 1e-3)}
        del E_half, age, sp, bp, fp, gp, sop
    # f4: the moment-damped LM solve on this scene's Gaussians, V = 3 views (the lower end of K_t in [3, 10])
    lm = None
    if world == 1:
        N, K, V = scene.N, (scene.sh_degree + 1) ** 2, 3
        shp = dict(means3D=(N, 3), scales=(N, 3), quats=(N, 4), opacities=(N,), sh=(N, K, 3))
        gL = torch.Generator(device=dev).manual_seed(2)
        rnd = lambda s_, sc_: torch.randn(s_, device=dev, generator=gL) * sc_
        lg = {k_: rnd((V,) + s_, 1e-3) for k_, s_ in shp.items()}
        lmm = {k_: rnd(s_, 1e-3) for k_, s_ in shp.items()}
        lv = {k_: torch.rand(s_, device=dev, generator=gL) * 1e-6 for k_, s_ in shp.items()}
        ld = {k_: torch.empty(s_, device=dev) for k_, s_ in shp.items()}
        tg.lm_solve(scene.sh_degree, lg, lmm, lv, t=5, delta=ld)
        lm_ms = 0.0
        for _ in range(args.steps):
            flush.fill_(1.0)
            la.record()
            tg.lm_solve(scene.sh_degree, lg, lmm, lv, t=5, delta=ld)
            lb.record()
            torch.cuda.synchronize()
            lm_ms += la.elapsed_time(lb)
        lm_ms /= args.steps
        row = 4 * (14 + 3 * K)                         # bytes of one parameter set per Gaussian (236 at degree 3)
        lm_bytes = N * row * ((V + 2) + 3)             # read V gradients + m + v, write m + v + Delta
        lm = {"views": V, "ms": lm_ms, "bytes_per_gaussian": row * (V + 5), "gbs": lm_bytes / (lm_ms * 1e-3) / 1e9,
              "hbm_frac": lm_bytes / (lm_ms * 1e-3) / 1e9 / peaks["hbm_gbs"], "kernels": ["lm_geo_kernel", "lm_app_sh_kernel"]}
        del lg, lmm, lv, ld
    # The whole of Alg. 1 steps 3-10 in the paper's regime (pipeline.SparseIteration.run_paper): V = 3 orbiting views of
    # this scene, per view projection, the paper's sampler from persistent maps, binning of all tiles, sparse forward,
    # fused loss, map update, sparse backward; then one LM solve with the per-view touched masks.  Eager launches.
    iteration = None
    if world == 1:
        import workloads
        import paper_2606_15924_b200 as pk
        V = 3
        cams = [workloads.orbit_view(scene, i).cam for i in range(V)]
        cap = int(1.5 * w.P_est) + 4096
        it_ = pk.SparseIteration(tg, cams, scene.N, scene.sh_degree, cap)
        gI = torch.Generator(device=dev).manual_seed(3)
        tgts = [torch.rand((cam.height, cam.width, 3), device=dev, generator=gI) for _ in range(V)]
        Em = [(torch.rand((cam.height, cam.width), device=dev, generator=gI) ** 3).to(torch.float16).view(torch.int16) for _ in range(V)]
        Ag = [torch.randint(0, 50, (cam.height, cam.width), device=dev, generator=gI, dtype=torch.int32).to(torch.int16) for _ in range(V)]
        K = (scene.sh_degree + 1) ** 2
        shp = dict(means3D=(scene.N, 3), scales=(scene.N, 3), quats=(scene.N, 4), opacities=(scene.N,), sh=(scene.N, K, 3))
        par = {k_: w.D[k_].clone() for k_ in shp}
        mI = {k_: torch.zeros(s_, device=dev) for k_, s_ in shp.items()}
        vI = {k_: torch.zeros(s_, device=dev) for k_, s_ in shp.items()}
        for t_ in (1, 2):
            it_.run_paper(par, tgts, Em, Ag, mI, vI, t=t_, n_pix=25, n_hard=10, n_stable=8, beta=0.4, seed=t_, apply=False)
        torch.cuda.synchronize()
        it_ms = 0.0
        nit = max(3, args.steps // 4)
        for r_ in range(nit):
            flush.fill_(1.0)
            la.record()
            it_.run_paper(par, tgts, Em, Ag, mI, vI, t=3 + r_, n_pix=25, n_hard=10, n_stable=8, beta=0.4, seed=3 + r_, apply=False)
            lb.record()
            torch.cuda.synchronize()
            it_ms += la.elapsed_time(lb)
        it_ms /= nit
        Pd = it_.step.binned.P_dev.tolist()
        n_it = int(it_.step.samp.kn_dev.tolist()[1])
        finite = bool(torch.isfinite(it_.delta["means3D"]).all())
        iteration = {"views": V, "n_pix_per_tile": 25, "ms_per_iteration": it_ms, "sampled_pixels_per_view": n_it,
                     "pairs_P_last_view": int(Pd[0]), "P_overflow": bool(Pd[1]), "delta_finite": finite,
                     "sampled_px_per_s": V * n_it / (it_ms * 1e-3),
                     "note": "Alg. 1 steps 3-10 for 3 views incl. tgs_lm_solve (Delta written, not applied: the scene stays the config's), eager launches; context: the paper's 77 s / 5000 "
                             "iterations = 15 ms per iteration of 3-10 views at ~0.6 M Gaussians on an RTX 5090 (PAPER.md:201, 508)"}
        del it_, tgts, Em, Ag, par, mI, vI
    stats_flops = FWD_FLOPS_WALK * w.walked + 12 * w.blended
    return {"lm_solve": lm, "iteration_paper_regime": iteration, "loss_sparse_ms": loss_ms, "loss_sparse_gbs": n * 44 / (loss_ms * 1e-3) / 1e9,
            "loss_sparse_hbm_frac": n * 44 / (loss_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
            "paper_regime": paper,
            "raster_stats_ms": stats_ms,
            "raster_stats_tflops": stats_flops / (stats_ms * 1e-3) / 1e12,
            "raster_stats_alu_frac": stats_flops / (stats_ms * 1e-3) / 1e12 / fp32_peak_measured,
            "note": "tgs_raster_stats_sparse (f3): 15 flop per walked + 12 per blended pair (w, 3 sums, recomputed "
                    "distance). tgs_loss_sparse (SURVEY.md 8f f1), timed alone, 44 algorithmic bytes per sampled pixel; "
                    "not inside the five-call step"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=HEADLINE_CONFIG, help="1..5, 1-based index into BASELINE.json configs "
                    "(default 4 = configs[3], the largest single-GPU configuration)")
    ap.add_argument("--pct", type=int, default=20, help="tile percentage for config 5")
    ap.add_argument("--impl", default="tgs", choices=["tgs", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block (the other configs and the sweep)")
    ap.add_argument("--step-only", action="store_true", help="skip the SURVEY 8f extras (loss, statistics forward, paper regime): "
                    "used for the profiler launch list of the five-call step")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_tgs(args)


if __name__ == "__main__":
    main()
