#!/usr/bin/env python
"""bench.py — one JSON line for the driver.

A step = one pass of the whole hot path over the workload: one OS-SART iteration
(all ordered subsets: Ax on every view, residual with row weights, A^T b on every view,
column-weighted update) through libtigre_b200's plan API.  Default workload: BASELINE.json
configs[2] "C3" (512^3, 720 views of 1024x768, half-fan, Poisson noise, 20 ordered subsets,
Siddon Ax / matched A^T b) — the configuration north_star's target is quoted on.

  python bench.py --gpus N --steps K --warmup W [--config C3] [--impl reference]
  python bench.py --mode tv [--tv-op prox] | --mode chunked | --mode drivers     (the other measured rows)

N > 1 (torchrun): the path does not shard in this build (north_star: one GPU, no collectives),
so every rank runs an independent replica of the same workload; value = N * units / max time.
--impl reference times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import make_config, phantom_for  # noqa: E402

METRIC = "Ax ray-samples/s + A^T b voxel-updates/s (one OS-SART iteration)"
UNIT = "G(samples+updates)/s"

# Roofline of the projector kernels.  They are gather kernels with hundreds of updates per HBM byte:
# the binding resource is plain-ALU issue slots or the on-chip gather path (L1 for Ax, shared memory for A^T b), not HBM.
# Every machine rate below is MEASURED at the start of the run by the library's own microbenchmark kernels
# (tigre_microbench): thread-instructions/s (FFMA issue), shared-memory bytes/s, L1 lines
# (wavefronts)/s.  The per-unit demands are algorithmic, except the L1 wavefronts a warp needs per
# 32 Siddon samples, which depend on how the rays of a warp spread over cache lines and are taken from the committed ncu
# captures (l1tex__data_pipe_lsu_wavefronts / samples):
#   A^T b            22 thread-instr and 16 B of shared-memory taps per voxel-update
#   Ax Siddon        18 thread-instr per segment; L1: W wavefronts per warp-sample (measured, table below)
#   Ax interpolated  40 thread-instr per sample; L1: 8 tap requests per sample, each at least TWO wavefronts on C2 / C4, where the 32
#                    rays of a warp are 1.04 / cos(theta) voxels apart and one request spans 132-188 bytes of a row: 16 per warp-
#                    sample.  (SURVEY.md section 8(d) guessed 24, "~halved by reusing a cell's 8 corners": reuse saves no REQUEST in a
#                    SIMT gather, the lanes change cells at different samples; shared-memory staging measured 17.6:
#                    profiles/r2_ax_interp_tma.md.  The L1 kernel itself needs 22: ncu.)
SM_COUNT = 148
ALGO_INSTR = {"atb": 22.0, "ax_siddon": 18.0, "ax_interp": 40.0}
# L1 data-pipe wavefronts per 32 samples of the Siddon march, from ncu (profiles/r1_late_ax_siddon.md: data pipe 42.7 % busy at
# 1397.6 G samples/s, 148 SMs x 1965 MHz => 2.84 wavefronts per warp-sample on C3)
SIDDON_WAVEFRONTS_PER_WARP_SAMPLE = 2.84
INTERP_WAVEFRONTS_PER_WARP_SAMPLE = 16.0
NOMINAL_PEAKS = {"ffma": 148 * 128 * 1.965e9, "smem": 148 * 128 * 1.965e9, "l1_lines": 148 * 1.965e9}

PEAK_UNITS = {"ffma": "thread-instr/s", "smem": "B/s", "l1_lines": "128-B lines/s", "l2": "B/s", "h2d": "B/s", "d2h": "B/s",
              "hbm_copy": "B/s (read+write)", "sm_hz": "Hz"}


def measure_peaks(tg, kinds=("ffma", "smem", "l1_lines", "l2", "hbm_copy", "sm_hz")):
    """The machine rates the projector rooflines rest on, measured now on this device by the library's own microbenchmark
    kernels (tigre_microbench): a few hundred milliseconds in all."""
    return {k: tg.microbench(k) for k in kinds}


def model_bounds(kname, rates):
    """{resource: G units/s} the machine rates allow for one kernel."""
    out = {"issue": rates["ffma"] / ALGO_INSTR[kname] / 1e9}
    if kname == "atb":
        out["smem"] = rates["smem"] / 16.0 / 1e9
    elif kname == "ax_siddon":
        out["l1"] = rates["l1_lines"] * 32.0 / SIDDON_WAVEFRONTS_PER_WARP_SAMPLE / 1e9
    else:
        out["l1"] = rates["l1_lines"] * 32.0 / INTERP_WAVEFRONTS_PER_WARP_SAMPLE / 1e9
    return out


def model_peak(kname, rates):
    """G units/s of the binding bound."""
    return min(model_bounds(kname, rates).values())


def peak_source(kname, rates, measured):
    bd = model_bounds(kname, rates)
    bind = min(bd, key=bd.get)
    how = "measured now by tigre_microbench" if measured else "NOMINAL (no microbenchmark in this mode)"
    return (f"min over {', '.join(f'{k} {v:.0f}' for k, v in bd.items())} G/s: binding = {bind}; machine rates {how}: "
            f"FFMA issue {rates['ffma'] / 1e12:.2f} T thread-instr/s, shared memory {rates['smem'] / 1e12:.2f} TB/s, L1 "
            f"{rates['l1_lines'] / 1e9:.1f} G lines/s; per-unit demand algorithmic (DESIGN.md section 6), Siddon L1 wavefronts from "
            f"ncu (profiles/); HBM is not the bound (see hbm)")


def run_peaks(tg, rank):
    import torch
    m = measure_peaks(tg, tuple(PEAK_UNITS))
    if rank != 0:
        return
    sm_hz = m["sm_hz"]
    per_clk = {"ffma_per_clk_per_sm": m["ffma"] / sm_hz / SM_COUNT, "smem_bytes_per_clk_per_sm": m["smem"] / sm_hz / SM_COUNT,
               "l1_lines_per_clk_per_sm": m["l1_lines"] / sm_hz / SM_COUNT, "l2_bytes_per_clk": m["l2"] / sm_hz}
    print(json.dumps({"metric": "step-0 machine rates (tigre_microbench)", "n_gpus": 1, "device": torch.cuda.get_device_name(0),
                      "values": m, "units": PEAK_UNITS, "per_clock": per_clk,
                      "nominal": {"ffma_per_clk_per_sm": 128, "smem_bytes_per_clk_per_sm": 128, "l1_lines_per_clk_per_sm": 1}}))


def ncu_traffic(config_name, kernel_regex, skip=5, timeout_s=240):
    """dram__bytes_read + dram__bytes_write of ONE launch of the dominant kernel, from a separate `ncu` run of this file's
    probe mode (a number printed under a profiler is never a bench value: only the byte counters are taken).  None if ncu
    is missing or the run fails (e.g. when this process is itself being profiled)."""
    import shutil
    ncu = shutil.which("ncu") or "/usr/local/cuda/bin/ncu"
    if not os.path.exists(ncu):
        return None, "ncu not found"
    cmd = [ncu, "--metrics", "dram__bytes_read.sum,dram__bytes_write.sum", "--clock-control", "none", "--print-units", "base",
           "--kernel-name", "regex:" + kernel_regex, "--launch-skip", str(skip), "--launch-count", "1", "--csv",
           sys.executable, os.path.abspath(__file__), "--mode", "probe", "--config", config_name]
    try:
        out = subprocess.run(cmd, capture_output=True, text=True, timeout=timeout_s, cwd=ROOT).stdout
    except Exception as e:
        return None, f"ncu run failed: {e}"
    import csv
    tot, seen = 0.0, 0
    rows = [r for r in csv.reader(out.splitlines()) if len(r) > 5]
    hdr = next((r for r in rows if "Metric Name" in r and "Metric Value" in r), None)
    if hdr is None:
        return None, "no ncu csv in the output"
    iname, ival = hdr.index("Metric Name"), hdr.index("Metric Value")
    for r in rows:
        if len(r) > max(iname, ival) and r[iname] in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            try:
                tot += float(r[ival].replace(",", ""))
                seen += 1
            except ValueError:
                pass
    if seen < 2:
        return None, "dram counters not found in the ncu output"
    return tot, "ncu --metrics dram__bytes_read.sum,dram__bytes_write.sum --clock-control none, launch %d of %s in `bench.py --mode probe`" % (skip + 1, kernel_regex)


def max_over_ranks(ms, device="cpu"):
    """Device time of the slowest rank (the contract's max over ranks); identity without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms)
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank, ms_step, world):
    """Replicas only: every rank processes the same units; G units/s over all ranks."""
    return world * units_per_rank / (ms_step * 1e-3) / 1e9


def subsets_for(rec, nA):
    n = 20 if rec["name"] == "C3" else 1
    n = min(n, nA)
    return [np.arange(s, nA, n) for s in range(n)]        # interleaved, visited in order (P15)


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], False

    def run(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        while not self.stop_flag:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([c.strip() for c in out.strip().split(",")])
            except Exception:
                pass
            time.sleep(0.2)

    def summary(self):
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for r in self.rows if len(r) >= 7 for n, v in zip(names, r[3:7]) if v.lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def cpu_baseline(geo, ang, rec, vol_h, b_h, samples_per_step, updates_per_step, budget_s=20.0):
    """The oracle as it stands, timed on this box's host cores on a bounded sample of the same workload:
    seeded random rays for Ax and seeded random voxels (all views) for A^T b."""
    from oracle import oracle as orc
    ax_mode = orc.SIDDON if rec["ax"] == "siddon" else orc.INTERP
    atb_mode = orc.MATCHED if rec["atb"] == "matched" else orc.FDK
    nA = len(ang)
    rng = np.random.default_rng(12345)
    n_rays_total = nA * geo.nDetector[0] * geo.nDetector[1]
    n_vox_total = int(np.prod(geo.nVoxel))
    # calibrate on a small sample, then size the real one to ~budget/2 each
    def run_ax(n):
        ids = rng.integers(0, n_rays_total, n)
        t = time.perf_counter()
        _, info = orc.ax(vol_h, geo, ang, ax_mode, ray_ids=ids, info=True)
        return time.perf_counter() - t, int(info["nseg"].sum())

    def run_atb(n):
        ids = rng.integers(0, n_vox_total, n)
        t = time.perf_counter()
        orc.atb(b_h, geo, ang, atb_mode, vox_ids=ids)
        return time.perf_counter() - t, n * nA

    t0, s0 = run_ax(2000)
    n_ax = int(max(2000, min(5e6, 2000 * (budget_s / 2) / max(t0, 1e-3))))
    t_ax, s_ax = run_ax(n_ax)
    t0, u0 = run_atb(200)
    n_atb = int(max(200, min(5e6, 200 * (budget_s / 2) / max(t0, 1e-3))))
    t_atb, u_atb = run_atb(n_atb)
    rate_ax, rate_atb = s_ax / t_ax, u_atb / t_atb
    t_step = samples_per_step / rate_ax + updates_per_step / rate_atb
    # the same two rates on ONE thread ("all hardware threads ... and single-thread"), on a tenth of the sample
    threads = orc.num_threads()
    orc.set_num_threads(1)
    try:
        t1a, s1a = run_ax(max(200, n_ax // (10 * max(threads, 1))))
        t1b, u1b = run_atb(max(20, n_atb // (10 * max(threads, 1))))
    finally:
        orc.set_num_threads(threads)
    t_step1 = samples_per_step / (s1a / t1a) + updates_per_step / (u1b / t1b)
    return {"value": (samples_per_step + updates_per_step) / t_step / 1e9, "unit": UNIT, "cores": threads, "nproc": os.cpu_count(),
            "kind": "oracle", "single_thread_value": (samples_per_step + updates_per_step) / t_step1 / 1e9,
            "single_thread": {"ax_gsamples_per_s": s1a / t1a / 1e9, "atb_gups": u1b / t1b / 1e9, "seconds": t1a + t1b},
            "sample": f"{n_ax} seeded random rays ({s_ax} ray-samples, {t_ax:.1f} s) + {n_atb} seeded random voxels x "
                      f"{nA} views ({u_atb} updates, {t_atb:.1f} s) of the same workload; full-step time extrapolated "
                      f"linearly from the two rates",
            "ax_gsamples_per_s": rate_ax / 1e9, "atb_gups": rate_atb / 1e9}, t_ax + t_atb


def run_chunked(args, tg, geo, ang, rec, config, K, W, rank, world, local_rank):
    """Host-chunking path: a step = one tigre_Ax + one tigre_sirt_chunked iteration (configs[4]'s
    "Siddon Ax + matched A^T b for one SIRT iteration") with the volume and the projections in PINNED HOST memory, streamed
    through the device budget.  Everything is end to end by construction (H2D / D2H copies inside the timed region,
    overlapped with the kernels by the library).  --chunk-n / --chunk-views select a C5-shaped problem of another size."""
    import torch
    from workloads import c5_like
    if args.chunk_n:
        geo, ang, rec = c5_like(args.chunk_n, args.chunk_views or max(64, int(2400 * args.chunk_n / 3072)))
        config = dict(config, workload=f"C5-shaped: {args.chunk_n}^3 fp32 volume, {len(ang)} views of {args.chunk_n}x{args.chunk_n}, "
                                       f"siddon Ax / matched A^T b")
    nA = len(ang)
    if args.budget_gb > 0:
        tg.set_chunk_budget(int(args.budget_gb * 2 ** 30))
    free_hbm = torch.cuda.mem_get_info()[0]
    rates = measure_peaks(tg, ("ffma", "smem", "l1_lines", "h2d", "d2h"))
    # seeded uniform-random volume generated slab by slab on the device (a voxelised phantom of this size takes
    # minutes on the host; timing does not depend on the values), exact-size page-locked host arrays for everything
    gen = torch.Generator(device="cuda").manual_seed(rec["seed"])
    vol_h = tg.pinned_empty(geo.vol_shape)
    for z0 in range(0, geo.vol_shape[0], 64):
        z1 = min(z0 + 64, geo.vol_shape[0])
        vol_h[z0:z1].copy_(torch.rand((z1 - z0,) + tuple(geo.vol_shape[1:]), generator=gen, device="cuda") * 0.02)
    proj_h = tg.pinned_empty((nA,) + tuple(geo.proj_shape))
    samples = tg.Ax_count(geo, ang, rec["ax"])
    updates = int(np.prod(geo.nVoxel)) * nA
    # a step: Ax (1 pass of samples) + SIRT iteration (1 pass of samples, 3 passes of voxel updates in the first iteration of a
    # call: max(A^T 1), A^T r, A^T 1)
    units = 2 * samples + 3 * updates
    torch.cuda.synchronize()

    def step():
        t0 = time.perf_counter()
        tg.Ax(vol_h, geo, ang, rec["ax"], out=proj_h)          # synchronises before returning
        st_ax = tg.chunk_stats()
        t1 = time.perf_counter()
        vol_h.mul_(0.5)                                        # start of the SIRT step: not the solution (host arithmetic, untimed below)
        t2 = time.perf_counter()
        tg.sirt_chunked(proj_h, geo, ang, vol_h, 1, ax_mode=rec["ax"], atb_mode=rec["atb"])   # b doubles as the residual scratch
        st_sirt = tg.chunk_stats()
        t3 = time.perf_counter()
        return (t1 - t0) * 1e3, (t3 - t2) * 1e3, st_ax, st_sirt

    for _ in range(W):
        step()
    sampler = ClockSampler(local_rank)
    sampler.start()
    tg.profile(True)
    torch.cuda.synchronize()
    runs = [step() for _ in range(K)]
    torch.cuda.synchronize()
    ms = max_over_ranks(sum(r[0] + r[1] for r in runs), "cuda")     # the two library calls (both synchronise); host scaling excluded
    prof = tg.profile_read()
    tg.profile(False)
    sampler.stop_flag = True
    sampler.join(timeout=2)
    if rank != 0:
        return
    ms_step = ms / K
    call_ms = float(np.mean([r[0] for r in runs])), float(np.mean([r[1] for r in runs]))
    st_ax, st_sirt = runs[-1][2], runs[-1][3]
    kind = "ax" if prof["ms"]["ax"] >= prof["ms"]["atb"] else "atb"
    kname = ("ax_" + rec["ax"]) if kind == "ax" else "atb"
    k_units, k_ms = (2 * samples if kind == "ax" else 3 * updates), prof["ms"][kind] / K
    achieved, peak = k_units / (k_ms * 1e-3) / 1e9, model_peak(kname, rates)
    value = whole_job_value(units, ms_step, world)
    h2d, d2h = int(st_ax[0] + st_sirt[0]), int(st_ax[1] + st_sirt[1])
    host_bytes = (int(np.prod(geo.nVoxel)) + nA * geo.nDetector[0] * geo.nDetector[1]) * 4
    config = dict(config, workload=config["workload"].split(", OS-SART")[0] + ", host-chunked (pinned host arrays): tigre_Ax + one tigre_sirt_chunked iteration",
                  budget_gb=args.budget_gb or f"default: 3/4 of free HBM = {free_hbm * 0.75 / 2 ** 30:.1f} GiB",
                  host_array_gb=host_bytes / 2 ** 30, exceeds_budget=bool(host_bytes > (args.budget_gb * 2 ** 30 if args.budget_gb else free_hbm * 0.75)),
                  phantom="uniform random (device-generated)",
                  chunks={"ax": {"z_slabs": st_ax[2], "view_batches": st_ax[3]}, "sirt_last_pass": {"z_slabs": st_sirt[2], "view_batches": st_sirt[3]}})
    link_s = h2d / rates["h2d"] + d2h / rates["d2h"]
    line = {"metric": METRIC.replace("one OS-SART iteration", "one chunked Ax + one chunked SIRT iteration"), "value": value, "unit": UNIT,
            "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": config, "clocks": sampler.summary(),
            "call_ms": {"tigre_Ax": call_ms[0], "tigre_sirt_chunked": call_ms[1]},
            "kernel_ms_per_step": {k: v / K for k, v in prof["ms"].items()},
            "overlap": {"kernel_share_of_call_time": (prof["ms"]["ax"] + prof["ms"]["atb"] + prof["ms"]["ew"]) / ms,
                        "note": "kernels and copies run on different streams: a share near 1 means the copies are hidden"},
            "host_link": {"h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "measured_peak_h2d_gbs": rates["h2d"] / 1e9,
                          "measured_peak_d2h_gbs": rates["d2h"] / 1e9, "seconds_at_peak_if_serial": link_s,
                          "share_of_step_if_serial": link_s / (ms_step * 1e-3),
                          "achieved_gbs_over_whole_step": (h2d + d2h) / (ms_step * 1e-3) / 1e9},
            "ax_gsamples_per_s": samples / (call_ms[0] * 1e-3) / 1e9,
            "sirt_g_units_per_s": (samples + 3 * updates) / (call_ms[1] * 1e-3) / 1e9,
            "units_per_step": {"ray_samples": 2 * samples, "voxel_updates": 3 * updates},
            "gpu_launches": int(sum(prof["launches"].values())),
            "roofline": {"kernel": kname, "bound": "alu", "achieved": achieved, "peak": peak, "frac": achieved / peak,
                         "unit": "Gsamples/s" if kind == "ax" else "Gupdates/s", "traffic": None,
                         "peak_source": peak_source(kname, rates, True), "ms_per_pass": k_ms},
            "e2e": {"value": value, "unit": UNIT, "ms_per_step": ms_step, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h}}
    print(json.dumps(line))


def run_tv(args, tg, geo, rec, K, W, rank, world, local_rank):
    """TV / AwTV minimiser: a step = --tv-steps normalised steepest-
    descent steps on a volume of the config's size.  This path IS HBM-bound: per voxel and descent step the
    gradient kernel reads x and writes g (8 B), the step kernel reads x and g and writes x (12 B)."""
    import torch
    n_tv, delta = args.tv_steps, (args.tv_delta if args.tv_delta > 0 else None)
    prox = args.tv_op == "prox"
    bpv = 48 if prox else 20                  # algorithmic bytes per voxel and inner step
    shape = tuple(geo.vol_shape)
    nvox = int(np.prod(shape))
    gen = torch.Generator(device="cuda").manual_seed(rec["seed"])
    x0 = torch.from_numpy(phantom_for(rec, geo)).cuda() if nvox <= 512 ** 3 else torch.zeros(shape, device="cuda")
    x0 += 1e-3 * torch.rand(shape, generator=gen, device="cuda")          # noisy phantom: what the minimiser is for
    x = x0.clone()
    if prox:
        class _P:                              # same call shape as the minimiser: in place on x
            @staticmethod
            def minimize_awtv(x, n, alpha, delta):
                return tg.tv_prox(x, 0.05, n, out=x)
            awtv_gradient = staticmethod(lambda x, delta: tg.tv_prox(x, 0.05, 1))
        run = _P
    else:
        run = tg
    for _ in range(W):
        run.minimize_awtv(x, n_tv, 1e-3, delta)
    sampler = ClockSampler(local_rank)
    sampler.start()
    tg.profile(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(K):
        run.minimize_awtv(x, n_tv, 1e-3, delta)
    e1.record()
    torch.cuda.synchronize()
    ms = max_over_ranks(e0.elapsed_time(e1), "cuda")
    prof = tg.profile_read()
    tg.profile(False)
    # the gradient kernel alone (value and ||g||^2 from the same pass), K * n_tv launches
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    run.awtv_gradient(x, delta)
    torch.cuda.synchronize()
    g0.record()
    for _ in range(K * n_tv):
        run.awtv_gradient(x, delta)
    g1.record()
    torch.cuda.synchronize()
    gms = g0.elapsed_time(g1) / (K * n_tv)
    # end to end: the volume in pinned host memory, copied in and out around every step
    x_h = torch.empty(shape, dtype=torch.float32, pin_memory=True)
    x_h.copy_(x0)
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    t0.record()
    for _ in range(K):
        x.copy_(x_h, non_blocking=True)
        run.minimize_awtv(x, n_tv, 1e-3, delta)
        x_h.copy_(x, non_blocking=True)
    t1.record()
    torch.cuda.synchronize()
    ems = max_over_ranks(t0.elapsed_time(t1), "cuda") / K
    sampler.stop_flag = True
    sampler.join(timeout=2)
    if rank != 0:
        return
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm = float(peaks.get("hbm_gbs", 6539.5))
    ms_step = ms / K
    unit = "Gvoxel-steps/s"
    value = whole_job_value(nvox * n_tv, ms_step, world)
    ach = nvox * n_tv * bpv / (ms_step * 1e-3) / 1e9
    line = {"metric": "TV proximal operator voxel-iterations/s" if prox else "TV minimiser voxel-steps/s", "value": value, "unit": unit, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": f"{rec['name']}-sized volume {shape[2]}x{shape[1]}x{shape[0]} fp32, {n_tv} descent steps of "
                                   f"{'the TV prox (dual projection iterations)' if prox else 'TV' if delta is None else 'AwTV delta=%g' % delta} per step", "seed": rec["seed"],
                       "l2": "volume + gradient larger than L2" if nvox * 8 > 126e6 else "fits L2", "parallelism": "single GPU"},
            "clocks": sampler.summary(), "gpu_launches": int(sum(prof["launches"].values())),
            "roofline": {"kernel": "prox_div_kernel + prox_update_kernel" if prox else "tv_gradient_kernel + tv_step_kernel",
                         "bound": "hbm", "achieved": ach, "peak": hbm, "unit": "GB/s",
                         "frac": ach / hbm, "traffic": None, "bytes_per_voxel_step": bpv,
                         "peak_source": "MEASURED_PEAKS.json hbm_gbs (copy bandwidth)",
                         **({} if prox else {"gradient_kernel": {"ms_per_launch": gms, "achieved": nvox * 8 / (gms * 1e-3) / 1e9,
                                                                  "bytes_per_voxel": 8, "frac": nvox * 8 / (gms * 1e-3) / 1e9 / hbm}})},
            "e2e": {"value": whole_job_value(nvox * n_tv, ems, world), "unit": unit, "ms_per_step": ems,
                    "h2d_bytes_per_step": nvox * 4, "d2h_bytes_per_step": nvox * 4}}
    if world == 1 and not args.no_cpu_baseline:
        from oracle import tv as otv
        m = 160
        xs = x0[:m, :m, :m].double().cpu().numpy()
        t = time.perf_counter()
        if prox:
            from oracle import prox as oprox
            oprox.tv_prox(xs, 0.05, 2)
        else:
            otv.minimize_awtv(xs, 2, 1e-3, np.inf if delta is None else delta)
        dt = time.perf_counter() - t
        line["cpu_baseline"] = {"value": m ** 3 * 2 / dt / 1e9, "unit": unit, "cores": 1, "kind": "oracle",
                                "sample": f"2 descent steps on the {m}^3 corner of the same volume ({dt:.1f} s, numpy fp64)"}
    print(json.dumps(line))


def run_drivers(args, tg, geo, ang, rec, subsets, rank):
    """One iteration of every reconstruction driver on the config's workload, device-resident:
    the extra rows' measurement.  One JSON line: ms per iteration (CUDA events, second of two runs)."""
    import torch
    vol = torch.from_numpy(phantom_for(rec, geo)).cuda()
    b = tg.Ax(vol, geo, ang, rec["ax"])
    del vol

    def timed(f):
        f()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        f()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    want = set(filter(None, args.drivers.split(",")))
    plan_rows = {
        "os_sart": (0.0, lambda x: plan.iterate(b, x, 1, want_resid=False)),
        "os_asd_pocs_ng20": (0.0, lambda x: plan.asd_pocs(b, x, 1, ng=20)),
        "sart_tv_tviter50": (0.0, lambda x: plan.sart_tv(b, x, 1, tv_lambda=1e-3, tv_iter=50)),
        "osem": (1.0, lambda x: plan.osem(b, x, 1)),
    }
    free_rows = {
        "fista_tviter50": lambda: tg.fista(b, geo, ang, 1, 2e5, 1e-3, 50, rec["ax"], rec["atb"]),
        "cgls": lambda: tg.cgls(b, geo, ang, 1, rec["ax"], rec["atb"]),
        "gradient_descent": lambda: tg.gradient_descent(b, geo, ang, 1, 1e-6, rec["ax"], rec["atb"]),
        "fdk_ram_lak": lambda: tg.fdk(b, geo, ang),
        "fdk_hann": lambda: tg.fdk_ex(b, geo, ang, "hann"),
    }
    out = {}
    if not want or want & set(plan_rows):
        plan = tg.OssartPlan(geo, ang, subsets, rec["ax"], rec["atb"])
        x = torch.empty(geo.vol_shape, dtype=torch.float32, device="cuda")
        for name, (x0, f) in plan_rows.items():
            if not want or name in want:
                x.fill_(x0)
                out[name] = timed(lambda: f(x))
        plan.close()
        del x
    for name, f in free_rows.items():
        if not want or name in want:
            out[name] = timed(f)
    if rank == 0:
        print(json.dumps({"metric": "ms per iteration of each driver", "unit": "ms", "n_gpus": 1, "data": "synthetic", "dtype": "f32",
                          "config": {"workload": f"{rec['name']}: {geo.nVoxel[0]}^3, {len(ang)} views of {geo.nDetector[0]}x"
                                                 f"{geo.nDetector[1]}, {rec['ax']} Ax / {rec['atb']} A^T b, {len(subsets)} subsets"},
                          "ms_per_iteration": {k: round(v, 2) for k, v in out.items()}}))


def run_probe(tg, geo, ang, rec, subsets):
    """What `ncu` watches for the traffic leg: one OS-SART iteration of the config through the plan on a seeded random
    volume (DRAM traffic does not depend on the values).  Prints nothing the driver reads."""
    import torch
    gen = torch.Generator(device="cuda").manual_seed(rec["seed"])
    vol = torch.rand(geo.vol_shape, generator=gen, device="cuda") * 0.02
    b = tg.Ax(vol, geo, ang, rec["ax"])
    plan = tg.OssartPlan(geo, ang, subsets, rec["ax"], rec["atb"])
    x = torch.zeros(geo.vol_shape, dtype=torch.float32, device="cuda")
    plan.iterate(b, x, 1, want_resid=False)
    torch.cuda.synchronize()
    plan.close()


def run_kernel(args, tg, geo, ang, rec, rank):
    """One kernel of the library on one config, timed alone with CUDA events (best of 3 after a warm-up) on seeded random data:
    the command the per-kernel ncu captures under profiles/ profile, and the A/B switch of the kernel-path hooks.
      --kernel ax:siddon | ax:interp | atb:matched | atb:fdk | atb:exact_siddon | atb:exact_interp | fdk_filter[:hann]
      --views N (a subset of N views, evenly spaced)   --ax-path / --siddon-path / --atb-path / --fdk-path / --index-path (the library's test hooks)"""
    import torch
    if args.views:
        sel = np.arange(0, len(ang), max(1, len(ang) // args.views))[:args.views]
        ang = ang[sel]
        if geo.rotDetector_a is not None:
            geo.rotDetector_a = geo.rotDetector_a[sel]
    tg.set_ax_path(args.ax_path)
    tg.set_siddon_path(args.siddon_path)
    tg.set_atb_path(args.atb_path)
    tg.set_fdk_path(args.fdk_path)
    tg.set_index_path(args.index_path)
    kind, _, mode = args.kernel.partition(":")
    gen = torch.Generator(device="cuda").manual_seed(rec["seed"])

    def timed(f, reps=3):
        f()
        best = 1e30
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            f()
            e1.record()
            torch.cuda.synchronize()
            best = min(best, e0.elapsed_time(e1))
        return best

    nA = len(ang)
    if kind == "ax":
        vol = torch.rand(geo.vol_shape, generator=gen, device="cuda") * 0.02
        units, unit = tg.Ax_count(geo, ang, mode), "Gsamples/s"
        ms = timed(lambda: tg.Ax(vol, geo, ang, mode))
    elif kind == "atb":
        b = torch.rand((nA,) + tuple(geo.proj_shape), generator=gen, device="cuda")
        if mode.startswith("exact_"):
            units, unit = tg.Ax_count(geo, ang, mode[6:]), "Gsamples/s"
        else:
            units, unit = int(np.prod(geo.nVoxel)) * nA, "Gupdates/s"
        ms = timed(lambda: tg.Atb(b, geo, ang, mode))
    elif kind == "fdk_filter":
        b = torch.rand((nA,) + tuple(geo.proj_shape), generator=gen, device="cuda")
        units, unit = 3.0 * 2.0 * nA * geo.nDetector[1] * float(geo.nDetector[0]) ** 2 / 1e3, "TFLOP/s (tf32-equivalent: 6 per multiply-add of the row convolution)"
        ms = timed((lambda: tg.fdk_filter_ex(b, geo, ang, mode)) if mode else (lambda: tg.fdk_filter(b, geo, ang)))
    else:
        raise SystemExit("unknown --kernel " + args.kernel)
    if rank == 0:
        print(json.dumps({"metric": "one kernel, timed alone", "kernel": args.kernel, "ms": ms, "value": units / (ms * 1e-3) / 1e9, "unit": unit,
                          "n_gpus": 1, "dtype": "f32", "data": "synthetic (seeded uniform random)",
                          "config": {"workload": f"{rec['name']}: {geo.nVoxel[0]}^3, {nA} views of {geo.nDetector[0]}x{geo.nDetector[1]}",
                                     "ax_path": args.ax_path, "siddon_path": args.siddon_path, "atb_path": args.atb_path, "fdk_path": args.fdk_path, "index_path": args.index_path}}))


def kernel_rates_other_configs(tg, rates):
    """SURVEY.md section 8(d) "per kernel, per config C2-C5": the two projector kernels of C2 (full size) and C4 (full-size volume and
    detector, 64 of its 1600 views: a launch of the size its CGLS makes per subset-free pass would take 9 s) timed with CUDA events
    on seeded random data, against the same measured-rate bounds.  C5's rates are `--mode chunked`'s (profiles/)."""
    import torch
    out = {}
    try:
        mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        mp = {}
    for name, n_views in (("C2", None), ("C4", 64)):
        geo, ang, rec = make_config(name)
        if n_views:
            sel = np.arange(0, len(ang), len(ang) // n_views)[:n_views]
            ang = ang[sel]
            if geo.rotDetector_a is not None:
                geo.rotDetector_a = geo.rotDetector_a[sel]
        if torch.cuda.mem_get_info()[0] < 4 * (int(np.prod(geo.nVoxel)) * 3 + len(ang) * geo.nDetector[0] * geo.nDetector[1] * 2) + (4 << 30):
            continue
        gen = torch.Generator(device="cuda").manual_seed(rec["seed"])
        vol = torch.rand(geo.vol_shape, generator=gen, device="cuda") * 0.02
        samples = tg.Ax_count(geo, ang, rec["ax"])
        updates = int(np.prod(geo.nVoxel)) * len(ang)

        def timed(f, reps=3):
            f()
            best = 1e30
            for _ in range(reps):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                e0.record()
                r = f()
                e1.record()
                torch.cuda.synchronize()
                best = min(best, e0.elapsed_time(e1))
            return best, r

        # (tigre_Ax includes the transposed copy of the volume it makes per call: < 1 % of these times)
        ms_ax, b = timed(lambda: tg.Ax(vol, geo, ang, rec["ax"]))
        ms_atb, _ = timed(lambda: tg.Atb(b, geo, ang, rec["atb"]))
        kax = "ax_" + rec["ax"]
        ax_rate, atb_rate = samples / (ms_ax * 1e-3) / 1e9, updates / (ms_atb * 1e-3) / 1e9
        extra = {}
        if rec["atb"] == "fdk":
            # the FDK pre-filter (fdk_tc.cu): the path's dense contraction, on the tensor cores: 3 split tf32 products per multiply-add
            ms_f, _ = timed(lambda: tg.fdk_filter(b, geo, ang))
            flop = 3.0 * 2.0 * len(ang) * geo.nDetector[1] * float(geo.nDetector[0]) ** 2
            tf32_peak = float(mp.get("bf16_tflops", 1591.4)) * 0.5
            extra["fdk_filter"] = {"ms": ms_f, "achieved": flop / (ms_f * 1e-3) / 1e12, "unit": "TFLOP/s (tf32, 3 split products per fp32 multiply-add)",
                                   "bound": "tensor", "peak": tf32_peak, "frac": flop / (ms_f * 1e-3) / 1e12 / tf32_peak,
                                   "peak_source": "MEASURED_PEAKS.json bf16_tflops x the guide's nominal tf32 : bf16 ratio 1/2"}
        out[name] = {"workload": f"{geo.nVoxel[0]}^3, {len(ang)} views of {geo.nDetector[0]}x{geo.nDetector[1]}" + (f" (of {rec['nA']})" if n_views else ""), **extra,
                     kax: {"achieved": ax_rate, "unit": "Gsamples/s", "peak": model_peak(kax, rates), "frac": ax_rate / model_peak(kax, rates),
                           "ms": ms_ax},
                     "atb_" + rec["atb"]: {"achieved": atb_rate, "unit": "Gupdates/s", "peak": model_peak("atb", rates),
                                           "frac": atb_rate / model_peak("atb", rates), "ms": ms_atb}}
        del vol, b
        torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C3")
    ap.add_argument("--scale", type=int, default=1, help="geometric down-scaling of the config (debug only)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--atb-kernel", default="tma", choices=["tma", "gather"], help="A/B switch of the A^T b kernel")
    ap.add_argument("--tv-steps", type=int, default=20, help="tv mode: descent steps per timed step")
    ap.add_argument("--tv-delta", type=float, default=0.0, help="tv mode: AwTV delta (0 = plain TV)")
    ap.add_argument("--tv-op", default="minimise", choices=["minimise", "prox"],
                    help="tv mode: the gradient-descent minimiser (tigre_minimize_awtv) or the TV proximal operator of FISTA (tigre_tv_prox)")
    ap.add_argument("--mode", default="plan", choices=["plan", "chunked", "tv", "drivers", "peaks", "probe", "kernel"],
                    help="plan: OS-SART iteration in HBM (default); chunked: Ax + A^T b with all arrays in pinned host memory (S8)")
    ap.add_argument("--kernel", default="ax:siddon", help="kernel mode: ax:siddon | ax:interp | atb:matched | atb:fdk | atb:exact_siddon | atb:exact_interp | fdk_filter[:window]")
    ap.add_argument("--views", type=int, default=0, help="kernel mode: use N evenly spaced views of the config (0 = all)")
    ap.add_argument("--atb-path", type=int, default=0, help="kernel mode: tigre_set_atb_path (0 default, 1 gather kernel, 3 TMA kernel without the linearised z-runs of tilted views)")
    ap.add_argument("--siddon-path", type=int, default=0, help="kernel mode: tigre_set_siddon_path (0 L1 kernel, 1 TMA-staged kernel)")
    ap.add_argument("--ax-path", type=int, default=0, help="kernel mode: tigre_set_ax_path (0 default, 1 L1 kernel, 2 TMA kernel also for wide beams)")
    ap.add_argument("--fdk-path", type=int, default=0, help="kernel mode: tigre_set_fdk_path (0 tensor cores, 1 CUDA cores)")
    ap.add_argument("--index-path", type=int, default=0, help="kernel mode: tigre_set_index_path (1 = 64-bit element offsets)")
    ap.add_argument("--drivers", default="", help="drivers mode: comma-separated subset of the drivers to time (default: all)")
    ap.add_argument("--budget-gb", type=float, default=0.0, help="chunked mode: device bytes the chunked path may use (0 = 3/4 of free)")
    ap.add_argument("--chunk-n", type=int, default=0, help="chunked mode: C5-shaped problem with an n^3 volume and an n x n detector (0: --config as given)")
    ap.add_argument("--chunk-views", type=int, default=0, help="chunked mode with --chunk-n: number of views (0: 2400 n / 3072)")
    ap.add_argument("--no-traffic", action="store_true", help="skip the ncu leg that measures the dominant kernel's DRAM bytes")
    ap.add_argument("--no-extra", action="store_true", help="skip the per-config kernel rates of C2 and C4")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    K, W = max(1, args.steps), max(0, args.warmup)

    geo, ang, rec = make_config(args.config, scale=args.scale)
    nA = len(ang)
    subsets = subsets_for(rec, nA)
    workload = (f"{rec['name']}{'' if args.scale == 1 else '/' + str(args.scale)}: {geo.nVoxel[0]}^3 fp32 volume, {nA} views of "
                f"{geo.nDetector[0]}x{geo.nDetector[1]}, {rec['ax']} Ax / {rec['atb']} A^T b, OS-SART with {len(subsets)} ordered subsets")
    config = {"workload": workload, "phantom": rec["phantom"], "seed": rec["seed"],
              "l2": "inputs larger than L2 (no flush needed)", "parallelism": "replicas only" if world > 1 else "single GPU"}

    if args.impl == "reference":
        if rank != 0:
            return
        vol_h = phantom_for(rec, geo)
        from oracle import oracle as orc
        # projections for the A^T b sample: the oracle's own Ax is too slow at full size, so the sample uses
        # seeded uniform-random projections of the right shape (timing does not depend on the values)
        b_h = np.random.default_rng(rec["seed"]).random((nA, geo.nDetector[1], geo.nDetector[0]), dtype=np.float32)
        n_rays = nA * geo.nDetector[0] * geo.nDetector[1]
        ids = np.random.default_rng(1).integers(0, n_rays, 20000)
        _, info = orc.ax(vol_h, geo, ang, orc.SIDDON if rec["ax"] == "siddon" else orc.INTERP, ray_ids=ids, info=True)
        samples = float(info["nseg"].mean()) * n_rays
        updates = float(np.prod(geo.nVoxel)) * nA
        vals, t_all = [], 0.0
        for i in range(W + K):
            cb, t = cpu_baseline(geo, ang, rec, vol_h, b_h, samples, updates, budget_s=8.0)
            if i >= W:
                vals.append(cb)
                t_all += t
        v = float(np.mean([c["value"] for c in vals]))
        cb = dict(vals[-1], value=v)
        line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
                "warmup": W, "ms_per_step": (samples + updates) / (v * 1e9) * 1e3, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": config,
                "cpu_baseline": cb, "gpu_launches": 0,
                "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
        print(json.dumps(line))
        return

    import torch
    import paper_2412_10129_b200 as tg
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (libtigre_b200 has no CPU fallback)"
    torch.cuda.set_device(local_rank)
    tg.set_atb_path(0 if args.atb_kernel == "tma" else 1)
    config["atb_kernel"] = args.atb_kernel
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    if args.mode == "probe":
        run_probe(tg, geo, ang, rec, subsets)
        return
    if args.mode == "kernel":
        run_kernel(args, tg, geo, ang, rec, rank)
        return
    if args.mode == "peaks":
        run_peaks(tg, rank)
        if world > 1:
            dist.destroy_process_group()
        return
    if args.mode == "drivers":
        run_drivers(args, tg, geo, ang, rec, subsets, rank)
        if world > 1:
            dist.destroy_process_group()
        return
    if args.mode == "tv":
        run_tv(args, tg, geo, rec, K, W, rank, world, local_rank)
        if world > 1:
            dist.destroy_process_group()
        return
    if args.mode == "chunked":
        run_chunked(args, tg, geo, ang, rec, config, K, W, rank, world, local_rank)
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- synthetic inputs (seeded)
    vol_h = phantom_for(rec, geo)
    vol = torch.from_numpy(vol_h).cuda()
    b = tg.Ax(vol, geo, ang, rec["ax"])
    if rec["name"] == "C3":           # Poisson noise on I0 = 1e5 then -log (configs[2]); timing input only
        g = torch.Generator(device="cuda").manual_seed(rec["seed"])
        counts = torch.poisson(1e5 * torch.exp(-b), generator=g)
        b = -torch.log(torch.clamp(counts, min=1.0) / 1e5)
        del counts
    samples = tg.Ax_count(geo, ang, rec["ax"])
    updates = int(np.prod(geo.nVoxel)) * nA
    units = samples + updates
    rates = measure_peaks(tg)          # the machine rates the roofline rests on, measured now (a few hundred ms, untimed)

    plan = tg.OssartPlan(geo, ang, subsets, rec["ax"], rec["atb"])
    x = torch.zeros(geo.vol_shape, dtype=torch.float32, device="cuda")
    for _ in range(W):
        plan.iterate(b, x, 1, want_resid=False)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    tg.profile(True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(K):
        plan.iterate(b, x, 1, want_resid=False)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    prof = tg.profile_read()
    tg.profile(False)
    sampler.stop_flag = True
    sampler.join(timeout=2)
    ms = max_over_ranks(ms, "cuda")
    ms_step = ms / K
    value = whole_job_value(units, ms_step, world)

    # ---- end to end through the C ABI with HOST buffers: b and x in pinned host memory, copied in / out per step
    e2e = None
    if not args.no_e2e:
        b_h = torch.empty(b.shape, dtype=torch.float32, pin_memory=True)
        b_h.copy_(b)
        x_h = torch.zeros(geo.vol_shape, dtype=torch.float32, pin_memory=True)
        plan.iterate(b_h, x_h, 1, want_resid=False)
        barrier()
        t0 = torch.cuda.Event(enable_timing=True)
        t1 = torch.cuda.Event(enable_timing=True)
        t0.record()
        for _ in range(K):
            plan.iterate(b_h, x_h, 1, want_resid=False)
        t1.record()
        barrier()
        ems = t0.elapsed_time(t1)
        ems = max_over_ranks(ems, "cuda")
        e2e = {"value": whole_job_value(units, ems / K, world), "unit": UNIT, "ms_per_step": ems / K,
               "h2d_bytes_per_step": int(b_h.numel() * 4 + x_h.numel() * 4), "d2h_bytes_per_step": int(x_h.numel() * 4)}
        del b_h, x_h

    if rank != 0:
        return
    clocks = sampler.summary()
    # ---- roofline of the dominant kernel (in-library CUDA events around every launch of the timed region)
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    kind = "ax" if prof["ms"]["ax"] >= prof["ms"]["atb"] else "atb"
    kname = ("ax_" + rec["ax"]) if kind == "ax" else "atb"
    other = "atb" if kind == "ax" else "ax_" + rec["ax"]
    k_units = samples if kind == "ax" else updates
    k_ms = prof["ms"][kind] / K                       # per full pass over all views
    achieved = k_units / (k_ms * 1e-3) / 1e9
    peak = model_peak(kname, rates)
    n_launch = len(subsets)                           # launches of the dominant kernel per step (one per subset)
    hbm_bytes = (vol.numel() + b.numel()) * 4         # compulsory: volume once + projections once
    traffic, traffic_src = (None, "skipped")
    if world == 1 and not args.no_traffic and args.scale == 1:
        del plan, x
        torch.cuda.empty_cache()
        traffic, traffic_src = ncu_traffic(rec["name"], "ax_siddon_kernel|ax_interp_kernel" if kind == "ax" else "atb_tma_kernel|atb_gather_kernel")
    other_ach = (updates if kind == "ax" else samples) / (prof["ms"]["atb" if kind == "ax" else "ax"] / K * 1e-3) / 1e9
    roofline = {"kernel": kname, "bound": "alu", "achieved": achieved, "peak": peak,
                "unit": "Gsamples/s" if kind == "ax" else "Gupdates/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": traffic_src,
                "algorithmic_hbm_bytes_per_launch": hbm_bytes / n_launch if kind == "atb" else (vol.numel() * 4 + b.numel() * 4 / n_launch),
                "bounds": model_bounds(kname, rates), "peak_source": peak_source(kname, rates, True),
                "machine_rates": dict(rates, nominal=NOMINAL_PEAKS),
                "launches_per_step": n_launch, "ms_per_launch": k_ms / n_launch,
                "units_per_launch": k_units / n_launch,
                "share_of_step": prof["ms"][kind] / ms, "ms_per_pass": k_ms,
                "other_kernel": {"kernel": other, "achieved": other_ach, "peak": model_peak(other, rates),
                                 "frac": other_ach / model_peak(other, rates), "bounds": model_bounds(other, rates),
                                 "note": "in the plan's OS-SART step this kernel also forms the update x <- max(0, x + lambda V .* A^T r) in its epilogue "
                                         "(fusion F2: no separate update kernel, no gradient volume); the kernel with a plain store: per_config / --mode kernel"},
                "hbm": {"algorithmic_bytes_per_pass": hbm_bytes, "achieved_gbs": hbm_bytes / (k_ms * 1e-3) / 1e9,
                        "peak_gbs": peaks.get("hbm_gbs"), "peak_source": "MEASURED_PEAKS.json hbm_gbs",
                        "note": "compulsory HBM traffic is ~1% of the time: not the bound"}}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": config, "clocks": clocks,
            "ax_gsamples_per_s": samples / (prof["ms"]["ax"] / K * 1e-3) / 1e9,
            "atb_gups": updates / (prof["ms"]["atb"] / K * 1e-3) / 1e9,
            "kernel_ms_per_step": {k: v / K for k, v in prof["ms"].items()},
            "units_per_step": {"ray_samples": samples, "voxel_updates": updates},
            "gpu_launches": int(sum(prof["launches"].values())), "roofline": roofline}
    if e2e:
        line["e2e"] = e2e
    if world == 1 and not args.no_cpu_baseline:
        b_host = b.cpu().numpy()
        line["cpu_baseline"], _ = cpu_baseline(geo, ang, rec, vol_h, b_host, samples, updates)
    if world == 1 and not args.no_extra and args.scale == 1:
        del vol, b
        torch.cuda.empty_cache()
        line["per_config"] = kernel_rates_other_configs(tg, rates)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
