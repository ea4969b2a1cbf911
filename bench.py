#!/usr/bin/env python
"""bench.py -- throughput of the matched-filter trajectory search on B200.

Metric (BASELINE.json): trajectory x frame x pixel evaluations per second of one full search
(`tno_mf_search`: planner, table kernels, the search kernel, candidate merge), on the paper's
headline workload: 100 trajectories x 1000 frames x 2048 x 2048 (config 3).  A "step" is one
search over one resident synthetic stack.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

N > 1 (launched by torchrun, one rank per GPU): every rank searches its own stack (one CCD per
GPU, no data-path collective); value = all ranks' evaluations / max-over-ranks time ("weak").
`--impl reference` times the CPU oracle (oracle/, float64, as it stands) on a bounded sample of
the same workload on the host cores (rank 0 only).
Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import tno_synth  # noqa: E402

METRIC = "traj_frame_pixel_evals_per_sec"
UNIT = "evals/s"
FP32_LANES_PER_SM = 128          # FFMA lanes per SM per clock (4 sub-partitions x 32)


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def _oracle_sample_rate(frames_win, sigma_t, trajs, cfg, region, window, full_shape):
    """Time the CPU oracle (as it stands) on a bounded sample; returns (evals/s, seconds, cores)."""
    import oracle
    t = time.perf_counter()
    oracle.snr_map(frames_win, sigma_t, trajs, cfg.prf_sigma, cfg.t0, region=region, window=window,
                   full_shape=full_shape)
    dt = time.perf_counter() - t
    x_lo, x_hi, y_lo, y_hi = region
    evals = trajs.shape[0] * cfg.T * (x_hi - x_lo) * (y_hi - y_lo)
    return evals / dt, dt, oracle.threads()


def _sample_trajs(p, n):
    """n trajectories spread over the bank, slowest and fastest included."""
    speed = np.hypot(p.traj[:, 0], p.traj[:, 1])
    order = np.argsort(speed, kind="stable")
    pick = order[np.linspace(0, len(order) - 1, n).round().astype(int)]
    return np.ascontiguousarray(p.traj[np.unique(pick)])


def run_reference(args, cfg):
    """The oracle on host cores, on a sub-frame of the same recipe (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    block = min(512, cfg.H, cfg.W)
    reach = 0
    p_full = tno_synth.make_params(cfg)
    dtm = max(abs(0.0 - cfg.t0), abs(cfg.T - 1 - cfg.t0))
    for tr in p_full.traj:
        reach = max(reach, int(np.ceil(max(abs(tr[0]) * dtm + abs(tr[2]) * dtm * dtm,
                                           abs(tr[1]) * dtm + abs(tr[3]) * dtm * dtm))) + 3)
    side = min(cfg.H, block + 2 * reach)
    sub = tno_synth.scaled(cfg, H=side, W=side)
    p = tno_synth.make_params(sub)
    frames = tno_synth.stack_numpy(p)
    oracle.inject(frames, p.traj[p.src_k], p.src_x, p.src_y, p.src_amp, sub.prf_sigma, sub.t0)
    trajs = _sample_trajs(p, 2 if cfg.T >= 500 else min(8, cfg.n_traj))
    lo = (side - block) // 2
    region = (lo, lo + block, lo, lo + block)
    times = []
    for i in range(args.warmup + args.steps):
        rate, dt, cores = _oracle_sample_rate(frames, p.sigma_t, trajs, sub, region, None, None)
        if i >= args.warmup:
            times.append(dt)
    evals = trajs.shape[0] * sub.T * block * block
    ms = 1e3 * float(np.mean(times))
    value = evals / (ms * 1e-3)
    sample = "%d trajectories x all %d frames x %dx%d start pixels of a %dx%d sub-frame, same recipe" % (
        trajs.shape[0], sub.T, block, block, side, side)
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
           "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": _workload(cfg), "sample": sample},
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def _workload(cfg):
    return "cfg%d %s: T=%d frames of %dx%d fp32, %d trajectories, prf_sigma=%.1f, top-%d @ %.1f sigma%s" % (
        cfg.idx, cfg.name, cfg.T, cfg.H, cfg.W, cfg.n_traj, cfg.prf_sigma, cfg.topk, cfg.threshold,
        "" if cfg.want_maps else ", no maps")


def run_ours(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_2209_09848_b200 import MatchedFilter, multi

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    # ---- inputs: one stack per rank (a different CCD each), generated on the device
    p = tno_synth.make_params(multi.rank_config(cfg, rank))       # rank-specific seed, same recipe
    frames = tno_synth.stack_torch(p, dev)
    mf = MatchedFilter(local, cfg.topk, cfg.threshold, record_events=True)
    mf.inject(frames, p.traj[p.src_k], p.src_x, p.src_y, p.src_amp, cfg.prf_sigma, cfg.t0)
    out_snr = torch.empty((cfg.n_traj, cfg.H, cfg.W), dtype=torch.float32, device=dev) if cfg.want_maps else None
    out_topk = torch.empty((cfg.n_traj, cfg.topk, 4), dtype=torch.int32, device=dev)
    torch.cuda.synchronize()

    def step():
        mf.search(frames, p.sigma_t, p.traj, cfg.prf_sigma, cfg.t0, want_maps=cfg.want_maps,
                  out_snr=out_snr, out_topk=out_topk)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    launches_per_step, used_kernel = mf.stats()
    fma_x, fma_y, add_y = mf.work()

    # ---- timed region: K steps, device-timed, max over ranks
    sampler = ClockSampler(local)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    kernel_ms = []
    ev0.record()
    for _ in range(args.steps):
        step()
        kernel_ms.append(mf.kernel_ms())
    ev1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop()
    total_ms = multi.max_over_ranks(ev0.elapsed_time(ev1), dev)
    ms_per_step = total_ms / args.steps
    value = multi.aggregate_value(cfg.evals, world, ms_per_step)

    # ---- end to end through the C ABI with HOST buffers (H2D of the stack, D2H of the results)
    e2e = None
    try:
        e2e_steps = max(1, min(args.steps, 2))
        try:
            host_frames = torch.empty(frames.shape, dtype=torch.float32, pin_memory=True)
            pinned = True
        except RuntimeError:
            host_frames = torch.empty(frames.shape, dtype=torch.float32)
            pinned = False
        host_frames.copy_(frames)
        host_topk = torch.empty(out_topk.shape, dtype=torch.int32, pin_memory=pinned)
        host_snr = torch.empty(out_snr.shape, dtype=torch.float32, pin_memory=pinned) if cfg.want_maps else None
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        # the library's host-buffer entry point: banded upload of the stack overlapped with the search,
        # maps and lists copied back, all inside the call (it returns when the host buffers are filled)
        mf.search_host(host_frames, p.sigma_t, p.traj, cfg.prf_sigma, cfg.t0, host_snr, host_topk)   # warm-up
        torch.cuda.synchronize()
        e0.record()
        for _ in range(e2e_steps):
            mf.search_host(host_frames, p.sigma_t, p.traj, cfg.prf_sigma, cfg.t0, host_snr, host_topk)
        e1.record()
        torch.cuda.synchronize()
        e2e_ms = multi.max_over_ranks(e0.elapsed_time(e1) / e2e_steps, dev)
        # outside the timed region: the host-buffer call must return, bit for bit, what the timed device search
        # left in out_snr / out_topk (same stack, same bank)
        step()
        torch.cuda.synchronize()
        same = bool(torch.equal(host_topk, out_topk.cpu()))
        if cfg.want_maps:
            for k0 in range(0, cfg.n_traj, 16):           # by slices: no second 1.7 GB host copy
                same = same and bool(torch.equal(host_snr[k0:k0 + 16], out_snr[k0:k0 + 16].cpu()))
        h2d = frames.numel() * 4
        d2h = out_topk.numel() * 4 + (out_snr.numel() * 4 if cfg.want_maps else 0)
        e2e = {"value": multi.aggregate_value(cfg.evals, world, e2e_ms), "unit": UNIT, "ms_per_step": e2e_ms,
               "steps": e2e_steps, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
               "host_memory": "pinned" if pinned else "pageable", "equals_device_search": same,
               "api": "tno_mf_search_host (upload in bands of frame rows, overlapped with the search)"}
        del host_frames, host_snr
    except RuntimeError as ex:            # e.g. not enough host memory for the stack
        e2e = {"value": None, "unit": UNIT, "error": str(ex)[:200], "h2d_bytes_per_step": 0,
               "d2h_bytes_per_step": 0}

    # ---- roofline of the dominant kernel (plain FP32 ALUs)
    peaks, peaks_src = _peaks()
    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    clk_hz = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
    peak_tflops = n_sm * FP32_LANES_PER_SM * 2 * clk_hz / 1e12
    k_s = float(np.mean(kernel_ms)) * 1e-3
    flops = 2.0 * (fma_x + fma_y) + add_y        # an addition occupies a lane of the FP32 pipe like a multiply-add, counts 1
    achieved = flops / k_s / 1e12
    # dram__bytes_read + write of one launch, from the committed ncu --set full capture (a stored figure: the
    # source file names the commit and the profile it was measured at, printed beside it so a stale one shows)
    traffic, traffic_src = None, None
    tp = os.path.join(ROOT, "profiles", "dram_traffic.json")
    if os.path.exists(tp):
        with open(tp) as f:
            tj = json.load(f)
        traffic = tj.get("cfg%d" % cfg.idx)
        traffic_src = {"file": "profiles/dram_traffic.json", "measured_at_commit": tj.get("measured_at_commit"),
                       "profile": tj.get("profile")}
    roofline = {"bound": "alu", "kernel": "k_search_sep" if used_kernel == 1 else "k_search_generic",
                "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s", "frac": achieved / peak_tflops,
                "traffic": traffic, "traffic_source": traffic_src,
                "peak_source": "%d SMs x 128 FP32 lanes x 2 x %.0f MHz (sm_max_mhz, %s)" % (
                    n_sm, clk_hz / 1e6, peaks_src),
                "kernel_ms": k_s * 1e3, "kernel_share_of_step": k_s * 1e3 / ms_per_step,
                "fma_per_eval_executed": (fma_x + fma_y) / cfg.evals, "add_per_eval_executed": add_y / cfg.evals,
                "pipe_frac": (fma_x + fma_y + add_y) / k_s / (n_sm * FP32_LANES_PER_SM * clk_hz),
                "frac_vs_25fma_definition": (2.0 * 25.0 * cfg.evals / k_s / 1e12) / peak_tflops,
                "hbm_compulsory_gbs": (frames.numel() * 4 + (out_snr.numel() * 4 if cfg.want_maps else 0)) / k_s / 1e9,
                "hbm_peak_gbs": peaks.get("hbm_gbs")}

    # ---- CPU baseline: the oracle on a bounded sample of this very stack (rank 0, N = 1 only)
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        block = min(1024, cfg.H, cfg.W)
        trajs = _sample_trajs(p, 8 if cfg.T >= 500 else min(8, cfg.n_traj))
        dtm = max(abs(0.0 - cfg.t0), abs(cfg.T - 1 - cfg.t0))
        reach = int(np.ceil(max(max(abs(tr[0]) * dtm + abs(tr[2]) * dtm * dtm,
                                    abs(tr[1]) * dtm + abs(tr[3]) * dtm * dtm) for tr in trajs))) + 3
        x_lo = (cfg.W - block) // 2
        y_lo = (cfg.H - block) // 2
        wx0, wy0 = max(0, x_lo - reach), max(0, y_lo - reach)
        wx1, wy1 = min(cfg.W, x_lo + block + reach), min(cfg.H, y_lo + block + reach)
        win = frames[:, wy0:wy1, wx0:wx1].contiguous().cpu().numpy()
        rate, secs, cores = _oracle_sample_rate(win, p.sigma_t, trajs, cfg,
                                                (x_lo, x_lo + block, y_lo, y_lo + block), (wx0, wy0),
                                                (cfg.H, cfg.W))
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": secs,
               "sample": "%d trajectories x all %d frames x %dx%d start pixels (centre block) of the "
                         "benchmarked stack" % (trajs.shape[0], cfg.T, block, block),
               "full_search_extrapolated_s": cfg.evals / rate}

    # ---- optional: the calls around the search (DESIGN 8b, 8d, 8f) on the same stack, device-timed; run last
    # because the background fit overwrites the stack with its residuals
    extras = None
    if args.extras:
        def timed(fn, reps=3):
            fn()
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(reps):
                fn()
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b) / reps
        extras = {}
        hbm = peaks.get("hbm_gbs")
        if cfg.want_maps:
            step()                              # the context's D tables must be those of out_snr
            ms = timed(lambda: mf.best(out_snr))
            extras["best"] = {"ms": ms, "bytes": out_snr.numel() * 4, "what": "max over trajectories, local-sigma Z "
                              "(255 box), top-K of Z"}
            mx, ak, z, _ = mf.best(out_snr)
            ms = timed(lambda: mf.peaks(z, 5, ak))
            extras["peaks"] = {"ms": ms, "what": "non-maximum suppression of Z, radius 5, threshold %g, top-K" % cfg.threshold}
            mxf = torch.empty_like(mx)
            akf = torch.empty_like(ak)
            from paper_2209_09848_b200 import tno_mf_search_max
            ms = timed(lambda: tno_mf_search_max(mf.ctx, frames, None, p.sigma_t, None, None, p.traj, cfg.prf_sigma,
                                                 cfg.t0, mxf, akf, out_snr, out_topk), reps=2)
            extras["search_max"] = {"ms": ms, "what": "the timed search with the max over the bank fused in",
                                    "equals_best": bool(torch.equal(mxf, mx) and torch.equal(akf, ak))}
            ms = timed(lambda: mf.flux(out_snr))
            gb = 2.0 * out_snr.numel() * 4 / 1e9
            extras["flux"] = {"ms": ms, "achieved_gbs": gb / ms * 1e3, "peak_gbs": hbm}
        jit = (0.4 * np.random.default_rng(cfg.idx).standard_normal((cfg.T, 2))).astype(np.float32)
        if cfg.H % 4 == 0 and cfg.W == cfg.H and cfg.H >= 64:
            # the paper's low-resolution scattered-light solve (section 3.1) at this stack's size: N = H / 4, n = N / 8;
            # synthetic input of its own (DESIGN 8g): scattered light per frame + jittered background + noise
            import paper_2209_09848_b200 as P
            N, n = cfg.H // 4, cfg.H // 32
            gen = torch.Generator(device=dev)
            gen.manual_seed(cfg.idx)
            low = torch.empty((cfg.T, N, N), device=dev)
            ms = timed(lambda: P.tno_mf_downsample(mf.ctx, frames, 4, low))
            extras["downsample"] = {"ms": ms, "achieved_gbs": frames.numel() * 4 * (1 + 1 / 16) / 1e6 / ms, "peak_gbs": hbm}
            phi = torch.from_numpy(np.stack([np.ones(cfg.T), jit[:, 0], jit[:, 1], jit[:, 0] ** 2, jit[:, 1] ** 2,
                                             jit[:, 0] * jit[:, 1]], 1).astype(np.float32)).to(dev)
            beta = torch.randn((6, N, N), device=dev, generator=gen) * torch.tensor([20., 3, 3, 1, 1, 1], device=dev)[:, None, None]
            S = 10 + 5 * torch.randn((cfg.T, n, n), device=dev, generator=gen)
            low = torch.nn.functional.interpolate(S[None], size=(N, N), mode="bilinear", align_corners=False)[0]
            low = (low + torch.einsum("tk,kij->tij", phi, beta)
                   + 0.3 * torch.randn((cfg.T, N, N), device=dev, generator=gen)).contiguous()
            b = torch.zeros((6, N, N), device=dev)
            s = torch.zeros((cfg.T, n, n), device=dev)
            torch.cuda.synchronize()
            t_fit = time.perf_counter()
            loss, iters, evals = P.tno_mf_scatter_fit(mf.ctx, low, jit, 1.0, 1000, 0.0, b, s)      # blocking call
            t_fit = time.perf_counter() - t_fit
            extras["scatter_fit"] = {"seconds": t_fit, "iterations": iters, "loss_evaluations": evals,
                                     "launches": mf.stats()[0], "final_loss_per_sample": loss / low.numel(),
                                     "N": N, "n": n, "paper_a100_seconds": 40.0}
            ms = timed(lambda: P.tno_mf_scatter_subtract(mf.ctx, frames, s), reps=1)
            extras["scatter_subtract"] = {"ms": ms, "achieved_gbs": 2.0 * frames.numel() * 4 / 1e6 / ms, "peak_gbs": hbm}
            del low, beta, S, b, s
        for n_iter in (0, 10):
            ms = timed(lambda: mf.background(frames, jit, 1.0, n_iter, in_place=True), reps=2)
            gb = (n_iter + 3.0) * frames.numel() * 4 / 1e9
            extras["background_n_iter_%d" % n_iter] = {"ms": ms, "algorithmic_gb": gb, "achieved_gbs": gb / ms * 1e3,
                                                       "peak_gbs": hbm, "frac": gb / ms * 1e3 / hbm if hbm else None}

        if cfg.want_maps and cfg.H % 4 == 0 and cfg.W == cfg.H and cfg.H >= 64:
            # the paper's whole chain on this stack, back to back (README): downsample -> scattered-light fit ->
            # subtract -> per-pixel background -> search with the max over the bank -> local-sigma scores -> peaks.
            # Host-timed: the fit reads scalars back, the rest is asynchronous until the final synchronize.
            import paper_2209_09848_b200 as P
            N, n = cfg.H // 4, cfg.H // 32
            low = torch.empty((cfg.T, N, N), device=dev)
            b = torch.zeros((6, N, N), device=dev)
            s = torch.zeros((cfg.T, n, n), device=dev)
            mxf, akf = torch.empty((cfg.H, cfg.W), device=dev), torch.empty((cfg.H, cfg.W), dtype=torch.int32, device=dev)
            torch.cuda.synchronize()
            t_chain = time.perf_counter()
            P.tno_mf_downsample(mf.ctx, frames, 4, low)
            _, it_c, ev_c = P.tno_mf_scatter_fit(mf.ctx, low, jit, 1.0, 1000, 0.0, b, s)
            P.tno_mf_scatter_subtract(mf.ctx, frames, s)
            mf.background(frames, jit, 1.0, 4, in_place=True)
            P.tno_mf_search_max(mf.ctx, frames, None, p.sigma_t, None, None, p.traj, cfg.prf_sigma, cfg.t0, mxf, akf,
                                None, out_topk)
            _, _, zc, _ = mf.best(mxf[None])
            mf.peaks(zc, 5, akf)
            torch.cuda.synchronize()
            extras["chain"] = {"seconds": time.perf_counter() - t_chain, "scatter_fit_iterations": it_c,
                               "what": "downsample 4x -> L-BFGS scattered-light fit -> subtract -> Huber background "
                                       "(4 iterations, in place) -> search with fused max over the bank -> local-sigma "
                                       "Z -> non-maximum suppression, on the resident stack",
                               "paper": "3-5 min per CCD-sector on an A100 (PAPER.md:L25, L144), 1 min of it the "
                                        "two background steps"}
            del low, b, s

    mf.close()
    if rank == 0:
        out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
               "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
               "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
               "config": {"workload": _workload(cfg), "per_gpu": "one full stack and search per GPU",
                          "l2": "inputs (%.1f GB stack) larger than L2" % (frames.numel() * 4 / 1e9),
                          "search_wall_time_s": ms_per_step * 1e-3},
               "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_step * args.steps,
               "roofline": roofline, "cpu_baseline": cpu, "extras": extras,
               "context": {"paper_a100_evals_per_s": 1.4e9,
                           "paper_claim": "100 trajectories x 1000 frames x 2048^2 in ~5 min on one A100 (PAPER.md:L9)"}}
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index 1..5 (3 = headline)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--extras", action="store_true",
                    help="also time tno_mf_best / tno_mf_flux / tno_mf_background on the same stack (after the timed region)")
    ap.add_argument("--frames", type=int, default=0,
                    help="profiling only: shorten the stack to this many frames (same recipe)")
    args = ap.parse_args()
    cfg = tno_synth.CONFIGS[args.config]
    if args.frames:
        cfg = tno_synth.scaled(cfg, T=args.frames, name=cfg.name + "-short(profiling only)")
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
