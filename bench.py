#!/usr/bin/env python
"""bench.py -- one TurboGS sparse-raster step (all five C-ABI calls) on seeded synthetic scenes.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--pct P] [--impl tgs|reference]

A "step" is one pass of the whole hot path over one view: tgs_preprocess -> tgs_bin_sort ->
tgs_sample -> tgs_raster_fwd_sparse -> tgs_raster_bwd_sparse (raster + projection halves).
Default workload = BASELINE.json configs[1] (100k Gaussians, 980x545, top 30% tiles).
Prints ONE JSON line (rank 0).  Multi-GPU = independent replicas, one view per rank, no data-path
collective (replicas only); the barrier / max-over-ranks timing uses NCCL.
"""
from __future__ import annotations

import argparse
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

# Algorithmic FP32 flops per Gaussian-pixel evaluation, counted from the oracle's arithmetic
# (DESIGN.md "Roofline accounting"): every visited (pixel, Gaussian) costs the power / exp / alpha
# test; a composited one additionally the blend (forward) or the nine partial derivatives (backward).
FWD_FLOPS_WALK, FWD_FLOPS_BLEND = 15, 10
BWD_FLOPS_WALK, BWD_FLOPS_BLEND = 15, 64
SM_COUNT, FP32_LANES, SM_MAX_GHZ = 148, 128, 1.965
FP32_PEAK_TFLOPS = SM_COUNT * FP32_LANES * 2 * SM_MAX_GHZ / 1e3  # 74.4: FMA = 2 flop, nominal max clock


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
def time_oracle(scene, steps, warmup):
    """The CPU oracle as it stands, single thread: one full step per iteration."""
    import oracle
    import workloads
    o = oracle.Oracle("f32")
    times, n = [], None
    g = None
    for i in range(warmup + steps):
        t0 = time.perf_counter()
        r = o.pipeline(scene, dL_dcolor=g, backward=g is not None, restrict=True)
        if g is None:  # first pass only sizes the upstream gradient (outside the timing)
            g = workloads.dl_dcolor(0, r.samp.n)
            t0 = time.perf_counter()
            r = o.pipeline(scene, dL_dcolor=g, backward=True, restrict=True)
        dt = time.perf_counter() - t0
        n = r.samp.n
        if i >= warmup:
            times.append(dt)
    return n, times, r


def run_reference(args):
    """--impl reference: the oracle timed on the host cores (this tier's reference arm)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    scene = load_scene(args.config, args.pct)
    n, times, r = time_oracle(scene, args.steps, args.warmup)
    total = sum(times)
    val = n * len(times) / total
    cfg = workload_config(scene, args, r.binned.P, r.samp.k, n)
    cfg["l2"] = "n/a (CPU)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": cfg,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle",
                             "sample": f"{len(times)} full steps of the workload, single thread"},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_config(scene, args, P, k, n):
    return {"workload": f"BASELINE.json configs[{args.config - 1}] ({scene.name})", "gaussians": scene.N,
            "sh_degree": scene.sh_degree, "image": [scene.cam.width, scene.cam.height],
            "tiles": scene.cam.num_tiles, "tile_pct": list(scene.tile_pct), "binning": "sampled tiles only (tile_select)",
            "pixel_mode": "all" if scene.pixel_mode == 0 else "bernoulli_err", "pairs_P": int(P),
            "sampled_tiles_k": int(k), "sampled_pixels_n": int(n), "parallelism": f"replicas x{args.gpus}"}


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

    scene = load_scene(args.config, args.pct)
    cam = scene.cam
    tg = pk.TGS(local)
    H = {k: torch.from_numpy(np.ascontiguousarray(getattr(scene, k))).pin_memory()
         for k in ("means3D", "scales", "quats", "opacities", "sh")}
    if scene.err is None:  # config 1: mask from the residual of a dense render; use a fixed seeded error map instead
        err_np = workloads.blob_error_map(np.random.default_rng(0), cam.width, cam.height, 8)
    else:
        err_np = scene.err
    H["err"] = torch.from_numpy(np.ascontiguousarray(err_np)).pin_memory()
    D = {k: v.to(dev) for k, v in H.items()}

    # size the pair buffers: one preprocess, then P = sum of tiles touched (plumbing, untimed)
    pre = tg.preprocess(cam, scene.sh_degree, D["means3D"], D["scales"], D["quats"], D["opacities"], D["sh"])
    rw = pre.splats[:, 10:12].contiguous().view(torch.int32)
    P_est = int((((rw[:, 0] >> 16) - (rw[:, 0] & 0xffff)).long() * ((rw[:, 1] >> 16) - (rw[:, 1] & 0xffff)).long()).sum())
    del pre, rw
    step = pk.SparseRasterStep(tg, cam, scene.N, scene.sh_degree, P_est + 1024, want_walked=True)

    def fwd():
        step.forward(D["means3D"], D["scales"], D["quats"], D["opacities"], D["sh"], scene.tile_pct, scene.pixel_mode,
                     scene.pix_rate, scene.sample_seed, err=D["err"])

    fwd()
    P, k, n = step.counts()
    walked = int(step.fwd.n_walked[:n].long().sum())
    blended = int(step.fwd.n_blended[:n].long().sum())
    replayed = int(step.fwd.n_contrib[:n].long().sum())
    g_host = torch.from_numpy(workloads.dl_dcolor(0, n) / np.float32(n)).pin_memory()
    g_dev = torch.zeros((cam.width * cam.height, 3), device=dev)
    g_dev[:n] = g_host.to(dev)
    step.fwd.n_walked = None   # work counters are not part of the timed step
    step.fwd.n_blended = None

    def full_step():
        fwd()
        step.backward(g_dev)

    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)  # 256 MiB > 126 MB L2

    barrier = rep.barrier

    # measured FFMA-only peak (tgs_fp32_peak): the roofline denominator of the raster kernels
    fp32_peak_measured = tg.fp32_peak(5)
    for _ in range(max(args.warmup, 3)):
        full_step()
    barrier()

    # ---- timed region: K steps, each bracketed by CUDA events, L2 flushed between steps ----
    sampler = ClockSampler(local)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    l0 = tg.launch_count()
    barrier()
    for s, e in ev:
        flush.fill_(1.0)
        s.record()
        full_step()
        e.record()
    barrier()
    launches = tg.launch_count() - l0
    sampler.stop_flag.set()
    sampler.join()
    step_ms = [s.elapsed_time(e) for s, e in ev]
    total_ms = sum(step_ms)
    total_ms = rep.max_over_ranks(total_ms)
    n_total = rep.sum_over_ranks(n)
    value = n_total * args.steps / (total_ms * 1e-3)

    # ---- the same step replayed from a CUDA graph (every call only enqueues; sizes are read on the device) ----
    graph_ms = None
    try:
        gs = torch.cuda.Stream()
        gs.wait_stream(torch.cuda.current_stream())
        cg = torch.cuda.CUDAGraph()
        with torch.cuda.stream(gs):
            with torch.cuda.graph(cg, stream=gs):
                full_step()
        torch.cuda.current_stream().wait_stream(gs)
        for _ in range(3):
            cg.replay()
        barrier()
        gev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for s_, e_ in gev:
            flush.fill_(1.0)
            s_.record()
            cg.replay()
            e_.record()
        barrier()
        graph_ms = rep.max_over_ranks(sum(s_.elapsed_time(e_) for s_, e_ in gev)) / args.steps
    except Exception as ex:  # without a capture the eagerly launched step above is the headline
        graph_ms = f"capture failed: {ex}"
    eager_ms = total_ms / args.steps
    launch_mode = "eager launches"
    if isinstance(graph_ms, float):
        # the step a user runs in a training loop: the same kernels, launched by one graph replay
        launch_mode = "cuda graph replay of the five calls (eager launches timed beside it)"
        total_ms = graph_ms * args.steps
        value = n_total * args.steps / (total_ms * 1e-3)

    # ---- per-call breakdown (separate pass; events between the calls) ----
    names = ["preprocess", "sample", "bin_sort", "raster_fwd", "raster_bwd", "project_bwd"]
    acc = {k_: 0.0 for k_ in names}
    tgs_, st = tg, step
    for _ in range(args.steps):
        flush.fill_(1.0)
        e_ = [torch.cuda.Event(enable_timing=True) for _ in range(7)]
        e_[0].record()
        tgs_.preprocess(cam, scene.sh_degree, D["means3D"], D["scales"], D["quats"], D["opacities"], D["sh"], out=st.pre)
        e_[1].record()
        tgs_.sample(cam, scene.tile_pct, scene.pixel_mode, scene.pix_rate, scene.sample_seed, err=D["err"], out=st.samp,
                    workspace=st.ws_sample, sync=False)
        e_[2].record()
        tgs_.bin_sort(cam, st.pre.splats, st.P_capacity, out=st.binned, workspace=st.ws_sort, sync=False,
                      tile_select=st.samp.tile_select)
        e_[3].record()
        tgs_.raster_fwd_sparse(cam, st.pre.splats, st.binned, st.samp, out=st.fwd)
        e_[4].record()
        tgs_.raster_bwd_sparse(cam, scene.sh_degree, st.pre.splats, st.binned, st.samp, st.fwd, g_dev, project=False,
                               out=st.bwd)
        e_[5].record()
        tgs_.raster_bwd_sparse(cam, scene.sh_degree, st.pre.splats, st.binned, st.samp, st.fwd, g_dev, D["means3D"],
                               D["scales"], D["quats"], D["sh"], st.pre.radii, st.pre.clamped, project=True, out=st.bwd)
        e_[6].record()
        torch.cuda.synchronize()
        d = [e_[i].elapsed_time(e_[i + 1]) for i in range(6)]
        for nm, v in zip(names[:5], d[:5]):
            acc[nm] += v
        acc["project_bwd"] += max(d[5] - d[4], 0.0)  # second call = raster + projection
    per_call_ms = {k_: v / args.steps for k_, v in acc.items()}

    peaks, peak_src = measured_peaks()
    next_rows = None
    if not args.step_only:
        # ---- SURVEY.md 8f f1 (not part of the five-call step): the fused sparse loss between forward and backward ----
        target_dev = torch.rand((cam.height, cam.width, 3), device=dev, generator=torch.Generator(device=dev).manual_seed(0))
        lo = tg.loss_sparse(cam, SimpleNamespace(k=k, n=n, tile_pix_offsets=st.samp.tile_pix_offsets, pix=st.samp.pix),
                            st.fwd.color, target_dev, n_capacity=cam.width * cam.height)
        la, lb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        loss_ms = 0.0
        for _ in range(args.steps):
            flush.fill_(1.0)
            la.record()
            tg.loss_sparse(cam, SimpleNamespace(k=k, n=n, tile_pix_offsets=st.samp.tile_pix_offsets, pix=st.samp.pix),
                           st.fwd.color, target_dev, out=lo)
            lb.record()
            torch.cuda.synchronize()
            loss_ms += la.elapsed_time(lb)
        loss_ms /= args.steps
        # the statistics forward (E_i, D_i, W_i, expected depth), fed with the loss kernel's per-pixel error
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

        # the paper's own regime -- N_pix = 25 pixels (r = 10 %) in EVERY tile with the
        # settings of its Tab. 6: r_hard = 0.4, r_stable = 0.3, 0.3 "mixed" remainder, beta = 0.4 --
        # sampler, binning of all tiles, sparse forward / backward / statistics on those lists, map updates
        paper = None
        if world == 1:
            gE = torch.Generator(device=dev).manual_seed(1)
            E_half = (torch.rand((cam.height, cam.width), device=dev, generator=gE) ** 3).to(torch.float16).view(torch.int16)
            age = torch.randint(0, 50, (cam.height, cam.width), device=dev, generator=gE, dtype=torch.int32).to(torch.int16)
            sp = tg.sample_paper(cam, E_half, age, 25, 10, 8, seed=1)
            bp = tg.bin_sort(cam, st.pre.splats, P_est + 1024, workspace=st.ws_sort, sync=True)
            fp = tg.raster_fwd_sparse(cam, st.pre.splats, bp, sp)
            gp = torch.randn((sp.n, 3), device=dev, generator=gE) / sp.n
            ob = SimpleNamespace(dL_dsplats=st.bwd.dL_dsplats)
            sop = tg.raster_stats_sparse(cam, st.pre.splats, bp, sp, lo.pix_err)
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(7)]
            accp = [0.0] * 6
            for _ in range(args.steps):
                flush.fill_(1.0)
                ev[0].record()
                tg.sample_paper(cam, E_half, age, 25, 10, 8, seed=1, out=sp, workspace=st.ws_sample, sync=False)
                ev[1].record()
                tg.bin_sort(cam, st.pre.splats, P_est + 1024, out=bp, workspace=st.ws_sort, sync=False)
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


        next_rows = {"loss_sparse_ms": loss_ms, "loss_sparse_gbs": n * 44 / (loss_ms * 1e-3) / 1e9,
                     "loss_sparse_hbm_frac": n * 44 / (loss_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                     "paper_regime": paper,
                     "raster_stats_ms": stats_ms,
                     "raster_stats_tflops": (FWD_FLOPS_WALK * walked + 12 * blended) / (stats_ms * 1e-3) / 1e12,
                     "raster_stats_alu_frac": (FWD_FLOPS_WALK * walked + 12 * blended) / (stats_ms * 1e-3) / 1e12 / fp32_peak_measured,
                     "note": "tgs_raster_stats_sparse (f3): 15 flop per walked + 12 per blended pair (w, 3 sums, recomputed "
                             "distance). tgs_loss_sparse (SURVEY.md 8f f1), timed alone, 44 algorithmic bytes per sampled pixel; "
                             "not inside the five-call step"}

    # ---- roofline of the dominant kernel ----
    peaks, peak_src = measured_peaks()
    fwd_flops = FWD_FLOPS_WALK * walked + FWD_FLOPS_BLEND * blended
    bwd_flops = BWD_FLOPS_WALK * replayed + BWD_FLOPS_BLEND * blended
    K = (scene.sh_degree + 1) ** 2
    hbm_bytes = {"preprocess": scene.N * (4 * (11 + 3 * K) + 48 + 5), "project_bwd": scene.N * (4 * (10 + 3 * K) + 48 + 5 + 4 * (11 + 3 * K)),
                 # rect/depth words of every record, then per emitted pair: segment write + read, gid_sorted write
                 "bin_sort": scene.N * 16 + P * (8 + 8 + 4) + cam.num_tiles * 12}
    kernels = {
        "raster_fwd": {"bound": "alu", "achieved": fwd_flops / (per_call_ms["raster_fwd"] * 1e-3) / 1e12,
                       "peak": fp32_peak_measured, "unit": "TFLOP/s"},
        "raster_bwd": {"bound": "alu", "achieved": bwd_flops / (per_call_ms["raster_bwd"] * 1e-3) / 1e12,
                       "peak": fp32_peak_measured, "unit": "TFLOP/s"},
    }
    for nm in ("preprocess", "project_bwd", "bin_sort"):
        kernels[nm] = {"bound": "hbm", "achieved": hbm_bytes[nm] / (per_call_ms[nm] * 1e-3) / 1e9,
                       "peak": peaks["hbm_gbs"], "unit": "GB/s"}
    kernels["bin_sort"]["note"] = "call of ~10 dependent kernels (launch list in profiles/), not one kernel"
    for v in kernels.values():
        v["frac"] = v["achieved"] / v["peak"]
    # dominant KERNEL of the step (bin_sort and sample are calls of several short kernels, each shorter
    # than these; profiles/ has the launch list that shows it)
    dominant = max(("raster_fwd", "raster_bwd", "preprocess", "project_bwd"), key=lambda k_: per_call_ms[k_])
    roof = dict(kernels[dominant])
    traffic = None
    tp = os.path.join(ROOT, "profiles", "r1d_traffic.csv")  # dram bytes per launch from the committed ncu --set full capture
    if os.path.exists(tp):
        with open(tp) as f:
            for ln in f.read().splitlines()[1:]:
                c_, k_, b_ = ln.split(",")
                if int(c_) == args.config and k_ == dominant:
                    traffic = float(b_)
    roof.update({"kernel": dominant + "_kernel", "traffic": traffic, "ms": per_call_ms[dominant],
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
    g_pin[:n] = g_host
    h2d = sum(v.numel() * v.element_size() for v in H.values()) + n * 12
    d2h = sum(v.numel() * v.element_size() for v in Hout.values())

    def e2e_step():
        for k_, v in H.items():
            D[k_].copy_(v, non_blocking=True)
        g_dev[:n].copy_(g_pin[:n], non_blocking=True)
        full_step()
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
            Dj = Dsets[j]
            step.forward(Dj["means3D"], Dj["scales"], Dj["quats"], Dj["opacities"], Dj["sh"], scene.tile_pct, scene.pixel_mode,
                         scene.pix_rate, scene.sample_seed, err=Dj["err"])
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

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / args.steps, "higher_is_better": True,
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
            "work": {"fwd_evals": walked, "bwd_evals": replayed, "blended": blended,
                     "fwd_evals_per_s": walked / (per_call_ms["raster_fwd"] * 1e-3),
                     "bwd_evals_per_s": replayed / (per_call_ms["raster_bwd"] * 1e-3),
                     "raster_px_per_s": n / ((per_call_ms["raster_fwd"] + per_call_ms["raster_bwd"]) * 1e-3)}}

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        reps = 10 if scene.N <= 200_000 else 1  # ~10 s of CPU work on configs[1]
        n_o, times, _ = time_oracle(scene, reps, 0)
        line["cpu_baseline"] = {"value": n_o * len(times) / sum(times), "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"{len(times)} full step(s) of the same workload, single thread, "
                                          f"{sum(times):.1f} s", "host_cores_available": os.cpu_count()}
    if rank == 0:
        print(json.dumps(line))
    rep.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=2, help="1..5, 1-based index into BASELINE.json configs")
    ap.add_argument("--pct", type=int, default=20, help="tile percentage for config 5")
    ap.add_argument("--impl", default="tgs", choices=["tgs", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--step-only", action="store_true", help="skip the SURVEY 8f extras (loss, statistics forward, paper regime): "
                    "used for the profiler launch list of the five-call step")
    args = ap.parse_args()
    if args.impl == "reference":
        if args.config > 2:  # bigger configs: keep the whole run within a few minutes
            args.steps, args.warmup = min(args.steps, 2), min(args.warmup, 1)
        run_reference(args)
    else:
        run_tgs(args)


if __name__ == "__main__":
    main()
