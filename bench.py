#!/usr/bin/env python
"""bench.py -- throughput of the pCMD hot path (stages 1-7) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--batch 1] [--impl ours|reference]

A "step" is one pass of the whole hot path -- pcmd_simulate (stages 1-5), pcmd_hess (6),
pcmd_loglike (7) -- over one batch of `--batch` parameter vectors of the BASELINE.json
configuration `--config` (default c3: 512x512 px, 3 bands, 10 500 isochrone points, the
configuration the metric "model evals/s and Poisson draws/s at 512^2 px" is quoted on).

`value`      model evaluations/s, device-timed (CUDA events around every step on the launching
             stream, inputs resident in HBM, L2 flushed between steps), whole job over all ranks.
`e2e`        the same metric through pcmd_evaluate_host (HOST buffers: parameters and data Hess
             copied host->device, model Hess and lnL copied device->host inside the timed region).
`roofline`   the dominant kernel (stage 2, Poisson draws -> pixel flux): bound "alu";
             achieved = draws x I_alg thread-instructions / stage-2 time (events recorded by the
             library on the same stream), peak = 148 SM x 4 schedulers x 32 lanes x max SM clock
             (DESIGN.md "Rooflines").
`cpu_baseline` the fp64 CPU oracle as it stands, timed on this box's host cores on a bounded
             sample (the same tables on a smaller image), scaled to the metric's unit.

N > 1 (torchrun, one rank per GPU): the path shards over independent model evaluations; every
rank runs its own batch with its own model indices (weak scaling), no data-path collective.
`--impl reference` times the CPU oracle (rank 0 only) on the same metric and configuration.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from workloads import synthetic as W  # noqa: E402

METRIC = "pcmd_model_evals_per_s"
UNIT = "evals/s"
SM_COUNT, SCHED_PER_SM, LANES = 148, 4, 32
# The Philox-only ceiling (a kernel that does nothing but Philox4x32-10 calls) is measured live by
# pcmd_pipe_bench in every run (outside the timed region): roofline.frac_of_philox_ceiling.
PHILOX_TEST = "Philox4x32-10 call"
# dram__bytes_read.sum + dram__bytes_write.sum of one k_stage2 launch from the committed captures: c3 and c5 from
# `ncu --set full` (profiles/r2_stage2.md), c4 x 64 models from the `--metrics` launch list (profiles/r2_launches.md);
# None for configurations / batches that were not captured
NCU_TRAFFIC_BYTES = {("c3", 1): 1.273e6 + 0.144e6, ("c5", 1): 8.408e6 + 0.102e6, ("c4", 64): 41.04e6 + 3.06e6}


def i_alg(n_bands: int) -> int:
    """Thread-instructions one Poisson draw needs: a quarter Philox4x32-10
    call = 5 wide multiplies + 5 three-input XORs, 1 threshold compare, 1 count/convert,
    n_bands FMAs, 1 for table search and loop control."""
    return 13 + n_bands


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            return json.load(fh), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, reasons, n_in = [], None, set(), 0
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                clk, mx = float(f[0]), float(f[1])
            except ValueError:
                continue
            smax = mx
            if t0 <= ts <= t1 + 0.1:
                n_in += 1
                sm.append(clk)
                for nm, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
        if not sm:   # the timed region was shorter than one sample: use everything seen
            sm = [float(l.split(",")[0]) for _, l in self.lines if l and l.split(",")[0].strip().replace(".", "").isdigit()]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax,
                "reasons": sorted(reasons), "samples": n_in}


# ------------------------------------------------------------------------------ oracle legs
def oracle_sample(c: int, sample_n_im: int):
    """One full pass (stages 1-7) of the oracle on config c's tables at a smaller image.
    Returns (seconds, pixel fraction of the full workload, threads)."""
    from oracle import pcmd_oracle as O
    full = W.config(c)
    wl = W.scaled(full, sample_n_im) if sample_n_im < full["n_im"] else full
    orc = O.Oracle(wl)
    t0 = time.perf_counter()
    sim = orc.simulate(wl["params"][0], seed=int(wl["seed"]))
    lnl = 0.0
    for h, d in zip(wl["hess"], wl["data_hess"]):
        H, _ = orc.hess(h, sim["mag"])
        lnl += O.loglike_poisson(H, d, wl["like_floor"])
    dt = time.perf_counter() - t0
    frac = (wl["n_im"] / full["n_im"]) ** 2
    return dt, frac, O.num_threads(), int((sim["lam"] > 0).sum()) * wl["n_im"] ** 2


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import pcmd_oracle as O
    O.build()
    full = W.config(args.config)
    S = min(args.ref_sample, full["n_im"])
    for _ in range(args.warmup):
        oracle_sample(args.config, min(S, 64))
    times, draws = [], 0
    for _ in range(args.steps):
        dt, frac, cores, draws = oracle_sample(args.config, S)
        times.append(dt)
    per_eval = float(np.mean(times)) / frac          # seconds one full-size evaluation would take
    val = 1.0 / per_eval
    sample = "config c%d tables at %dx%d px (%.4g of the pixels), all 7 stages, scaled by pixel count" % (
        args.config, S, S, frac)
    line = {"impl": "reference", "extrapolated": bool(frac < 1.0), "sample_n_im": int(S), "scale_factor": 1.0 / frac,
            "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": per_eval * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "gpu_launches": 0,
            "config": {"workload": "c%d" % args.config, "n_im": full["n_im"], "n_bands": full["n_bands"],
                       "n_points": full["n_points"], "batch": 1, "sample": sample},
            "draws_per_s": draws / float(np.mean(times)),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------ CUDA leg
def shard_models(batch: int, rank: int) -> int:
    """Weak scaling over independent evaluations: rank r owns model indices [r*batch, (r+1)*batch)."""
    return rank * batch


def max_over_ranks(x: float, device=None) -> float:
    """Timing of a multi-rank job = the slowest rank (all_reduce MAX); identity for one rank."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: float, world: int, seconds: float) -> float:
    """Whole-job throughput: units of ALL ranks over the slowest rank's time."""
    return units_per_rank * world / seconds


def batch_params(wl: dict, batch: int):
    prm = wl["params"]
    return [prm[i % len(prm)] for i in range(batch)]


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_1904_00011_b200 as G

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus and world > 1:
        raise SystemExit("--gpus %d but WORLD_SIZE=%d" % (args.gpus, world))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    wl = W.config(args.config)
    if args.sampler_mode == 1:      # aggregated sampler (PAPER.md:75 fn. 3; DESIGN.md R-A1): a different random stream
        wl = dict(wl, sampler_mode=1)
    g = G.Pcmd(wl, separable=True)
    prm = batch_params(wl, args.batch)
    if args.sfh_scale != 1.0:       # diagnostic: the same tables with every expected star count scaled (1e-6: every group of
        prm = [dict(p, sfh=np.asarray(p["sfh"]) * args.sfh_scale) for p in prm]   # points in the rare-star class = Philox + one vote)
    n = len(prm)
    seed, m0 = int(wl["seed"]), shard_models(n, rank)
    data = np.concatenate([d.ravel() for d in wl["data_hess"]]).astype(np.uint32)
    d_data = torch.from_numpy(data.view(np.int32)).cuda()
    mag = torch.empty((n, g.B, g.N, g.N), dtype=torch.float32, device="cuda")
    H = torch.empty((n, g.bins_total), dtype=torch.int32, device="cuda")
    l2_bytes = torch.cuda.get_device_properties(local).L2_cache_size
    flush = torch.empty(int(2 * l2_bytes) // 4, dtype=torch.int32, device="cuda")

    def step():
        g.simulate(prm, seed=seed, model_index0=m0, mag=mag)
        Hh, st = g.hess(mag, out=H)
        return g.loglike(Hh, st, d_data)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
        flush.zero_()
    torch.cuda.synchronize()
    if g.status() != 0:
        raise SystemExit("device status %d" % g.status())
    # draws of one step on this rank: P x #{j: lambda_j > 0}, summed over the batch's models
    # (models with a narrow MDF have whole isochrones cut to lambda = 0: those are not drawn)
    if args.sampler_mode == 1:      # random numbers that decide a star: one per star (expected N_pix per pixel) + the total
        draws_step = int(sum(float(np.sum(p["sfh"])) + 1.0 for p in prm) * g.P)
    else:
        draws_step = sum(int((g.debug_weights(i)["lam"] > 0).sum()) for i in range(n)) * g.P
    g.profile(True)

    # ---- device-timed leg
    clocks = ClockSampler(local)
    clocks.start()
    time.sleep(0.25)
    barrier()
    l0 = g.launch_count()
    t_wall0 = time.time()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    stage = np.zeros(5)
    for a, b in ev:
        a.record()
        step()
        b.record()
        b.synchronize()
        stage += np.maximum(g.stage_ms(), 0.0)
        flush.zero_()           # L2 flush between timed iterations (outside the events)
    barrier()
    t_wall1 = time.time()
    launches = g.launch_count() - l0
    clk = clocks.stop(t_wall0, t_wall1)
    ms = np.array([a.elapsed_time(b) for a, b in ev])
    total_ms = max_over_ranks(float(ms.sum()), "cuda")
    g.profile(False)
    philox_draws = None
    if rank == 0:       # the Philox-only kernel of the library, same device, same clocks (5 ms)
        philox_draws = 4.0 * G.pipe_bench(only=PHILOX_TEST)[0]["steps_per_s"]

    # ---- end to end through the host-buffer entry point
    for _ in range(2):
        g.evaluate_host(prm, data, seed=seed, model_index0=m0)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        lnl_h, H_h, st_h = g.evaluate_host(prm, data, seed=seed, model_index0=m0)
    torch.cuda.synchronize()
    e2e_s = max_over_ranks(time.perf_counter() - t0, "cuda")
    h2d = data.nbytes + n * (g.A * 8 + 5 * 8)
    d2h = n * (8 + g.bins_total * 4 + len(g.hess_specs) * 32)

    if rank == 0:
        peaks, which = measured_peaks()
        ms_step = total_ms / args.steps
        evals = whole_job_rate(n * args.steps, world, total_ms * 1e-3)
        s2_ms = float(stage[1]) / args.steps
        draws = draws_step
        # aggregated sampler: half a Philox call per star (10 wide multiplies + 10 xors), the 64 x 64 -> high 64
        # product (4 wide multiplies), guide look-up + ~2 search steps (8), B flux adds
        ia = i_alg(g.B) if args.sampler_mode == 0 else 32 + g.B
        peak_inst = SM_COUNT * SCHED_PER_SM * LANES * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12
        ach = draws * ia / (s2_ms * 1e-3) / 1e12 if s2_ms > 0 else 0.0
        line = {"metric": METRIC, "value": evals, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "u32+f32", "data": "synthetic",
                "config": {"workload": "c%d" % args.config, "n_im": g.N, "n_bands": g.B, "n_points": g.J,
                           "batch": n, "psf_k": int(wl["psf_k"]), **({"sfh_scale": args.sfh_scale} if args.sfh_scale != 1.0 else {}),
                           "sampler": "aggregated (sampler_mode 1)" if args.sampler_mode == 1 else "per-point Poisson (sampler_mode 0)", "l2": "flushed between steps (2x L2 written)",
                           "parallelism": "replicas over model index x%d" % world},
                "draws_per_s": draws * world * args.steps / (total_ms * 1e-3),
                "draws_per_s_stage2": draws / (s2_ms * 1e-3) if s2_ms > 0 else None,
                "stage_ms": {k: float(v) / args.steps for k, v in
                             zip(("stage1", "stage2", "stage4_5", "stage6", "stage7"), stage)},
                "gpu_launches": int(launches),
                "clocks": clk,
                "e2e": {"value": n * world * args.steps / e2e_s, "unit": UNIT,
                        "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h)},
                "roofline": {"kernel": "k_stage2_agg (stars placed by table inversion)" if args.sampler_mode == 1 else "k_stage2 (Poisson draws -> pixel flux)", "bound": "alu",
                             "achieved": ach, "peak": peak_inst, "unit": "Tinst/s",
                             "frac": ach / peak_inst, "traffic": NCU_TRAFFIC_BYTES.get(("c%d" % args.config, n)),
                             "frac_of_philox_ceiling": (draws / (s2_ms * 1e-3)) / philox_draws if s2_ms > 0 else None,
                             "philox_only_draws_per_s": philox_draws,
                             "i_alg_thread_inst_per_draw": ia, "draws_per_launch": draws,
                             "ms_per_launch": s2_ms, "peak_source": which + " sm_max_mhz"}}
        if world == 1 and not args.no_cpu:
            from oracle import pcmd_oracle as O
            O.build()
            dt, frac, cores, _ = oracle_sample(args.config, min(args.cpu_sample, wl["n_im"]))
            line["cpu_baseline"] = {
                "value": 1.0 / (dt / frac), "unit": UNIT, "cores": cores, "kind": "oracle",
                "sample": "config c%d tables at %dx%d px (%.4g of the pixels), all 7 stages, %.1f s, scaled "
                          "by pixel count" % (args.config, min(args.cpu_sample, wl["n_im"]),
                                              min(args.cpu_sample, wl["n_im"]), frac, dt)}
        print(json.dumps(line), flush=True)
    g.close()
    if world > 1:
        dist.destroy_process_group()


def run_hbm_stages(args):
    """HBM fraction of stage 4 alone (noise off), the fused stages 4-5 and stage 6 on an L2-exceeding batch
    (DESIGN.md "Rooflines"): the images of `--hbm-batch` models of config `--config` geometry (default c4:
    256x256 px, 2 bands) exceed the L2 several times, so every stage streams from / to HBM.  Also: the general
    2-D K x K convolution against the FP32 FMA peak, and stage 6 on a collapsed pCMD
    (every pixel in a handful of bins: the shared-memory atomic contention case).
    Prints one JSON line."""
    import torch
    import paper_1904_00011_b200 as G
    torch.cuda.set_device(0)
    n = args.hbm_batch
    reps = max(args.steps, 3)
    peaks, which = measured_peaks()

    def timed(wl, separable, n_models, collapsed=False):
        g = G.Pcmd(wl, separable=separable)
        prm = batch_params(wl, n_models)
        mag = torch.empty((n_models, g.B, g.N, g.N), dtype=torch.float32, device="cuda")
        H = torch.empty((n_models, g.bins_total), dtype=torch.int32, device="cuda")
        g.profile(True)
        acc = np.zeros(5)
        for it in range(2 + reps):
            g.simulate(prm, seed=1, mag=mag)
            if collapsed and it == 0:      # every pixel of every image within +-0.01 mag of one point inside the window
                h0 = g.hess_specs[0]
                yc = 0.5 * (h0["y_lo"] + h0["y_hi"]); xc = 0.5 * (h0["x_lo"] + h0["x_hi"])
                base = torch.rand((n_models, 1, g.N, g.N), device="cuda") * 0.02 - 0.01
                cmag = torch.empty_like(mag)
                for b in range(g.B):
                    cmag[:, b:b + 1] = yc + base + (xc if b == h0["band_plus"] and b != h0["band_minus"] else 0.0)
            g.hess(cmag if collapsed else mag, out=H)
            ms = g.stage_ms()
            if it >= 2:
                acc += np.maximum(ms, 0.0)
        acc /= reps
        img_bytes = n_models * g.B * g.P * 4
        used = len({b for h in g.hess_specs for b in (h["band_plus"], h["band_minus"], h["band_y"])})
        hess_bytes = n_models * used * g.P * 4 + n_models * g.bins_total * 4
        out = dict(ms45=float(acc[2]), ms6=float(acc[3]), img_bytes=img_bytes, hess_bytes=hess_bytes, K=int(wl["psf_k"]),
                   pixel_bands=n_models * g.B * g.P, stage2_ms=float(acc[1]))
        g.close()
        return out

    def gbs(nbytes, ms):
        return nbytes / (ms * 1e-3) / 1e9

    wl_on = W.config(args.config)
    wl_off = dict(wl_on, shot_noise=0, poisson_sky=0, read_sigma=np.zeros(int(wl_on["n_bands"])),
                  sky=np.zeros(int(wl_on["n_bands"])))
    if args.hbm_variant != "all":      # one variant only (profiling): stage times on stderr
        r = timed(wl_on if args.hbm_variant == "on" else wl_off, args.hbm_variant != "general", n,
                  collapsed=args.hbm_variant == "collapsed")
        print(json.dumps({"hbm_variant": args.hbm_variant, **r}), flush=True)
        return
    on = timed(wl_on, True, n)
    off = timed(wl_off, True, n)
    col = timed(wl_off, True, n, collapsed=True)
    n2 = max(1, n // 8)                    # the K x K kernel is FMA-bound: a smaller batch keeps the run short
    gen = timed(wl_off, False, n2)
    fma_peak = SM_COUNT * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12          # TFLOP/s: 128 FP32 FMA lanes per SM
    gen_tflops = 2.0 * gen["K"] ** 2 * gen["pixel_bands"] / (gen["ms45"] * 1e-3) / 1e12
    res = {"hbm_stages": {
        "workload": "c%d geometry x %d models (%.0f MB of images, L2 126 MB)" % (args.config, n, on["img_bytes"] / 1e6),
        "stage4_noise_off": {"kernel": "k_conv2<%d> (separable)" % off["K"], "ms": off["ms45"], "algorithmic_bytes": 2 * off["img_bytes"],
                             "GBps": gbs(2 * off["img_bytes"], off["ms45"]), "frac": gbs(2 * off["img_bytes"], off["ms45"]) / peaks["hbm_gbs"]},
        "stage4_5": {"kernel": "k_conv2<%d> (separable) + noise + magnitudes" % on["K"], "ms": on["ms45"], "algorithmic_bytes": 2 * on["img_bytes"],
                     "GBps": gbs(2 * on["img_bytes"], on["ms45"]), "frac": gbs(2 * on["img_bytes"], on["ms45"]) / peaks["hbm_gbs"],
                     "bound": "alu (one Philox4x32-10 call + Box-Muller + log2 per pixel-band; DESIGN.md)"},
        "stage4_general_2d": {"kernel": "k_conv_noise (direct K x K)", "models": n2, "ms": gen["ms45"], "flops": 2.0 * gen["K"] ** 2 * gen["pixel_bands"],
                              "TFLOPs": gen_tflops, "peak_TFLOPs": fma_peak, "frac_of_fp32_fma_peak": gen_tflops / fma_peak},
        "stage6": {"ms": on["ms6"], "algorithmic_bytes": on["hess_bytes"], "GBps": gbs(on["hess_bytes"], on["ms6"]),
                   "frac": gbs(on["hess_bytes"], on["ms6"]) / peaks["hbm_gbs"]},
        "stage6_collapsed": {"ms": col["ms6"], "algorithmic_bytes": col["hess_bytes"], "GBps": gbs(col["hess_bytes"], col["ms6"]),
                             "frac": gbs(col["hess_bytes"], col["ms6"]) / peaks["hbm_gbs"],
                             "what": "every pixel within 0.01 mag of one point of the window (PAPER.md:198)"},
        "peak_GBps": peaks["hbm_gbs"], "peak_source": which}}
    print(json.dumps(res), flush=True)


def run_pipes(args):
    """The pipe table DESIGN.md "Rooflines" quotes: sustained warp-instructions per clock per scheduler of
    each instruction stream, and the draws/s of a kernel that does nothing but Philox4x32-10."""
    import torch
    import paper_1904_00011_b200 as G
    torch.cuda.set_device(0)
    rows = G.pipe_bench()
    philox = [r for r in rows if r["name"].startswith("Philox4x32-10")][0]
    print(json.dumps({"pipes": [{"stream": r["name"], "warp_instr_per_clk_per_scheduler": round(r["rate"], 4),
                                 "ms": round(r["ms"], 4)} for r in rows],
                      "philox_calls_per_s": philox["steps_per_s"], "philox_draws_per_s": 4.0 * philox["steps_per_s"],
                      "launch": "148 SMs x 2 CTAs x 512 threads, 8 independent chains per thread"}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--batch", type=int, default=1)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cpu-sample", type=int, default=256, help="image side of the cpu_baseline sample")
    ap.add_argument("--ref-sample", type=int, default=512,
                    help="image side of the --impl reference sample (default: the full image up to 512 px, i.e. c1-c4 are "
                         "timed at full size and only c5 is a sample scaled by pixel count; the line says which)")
    ap.add_argument("--all-configs", action="store_true", help="one line per BASELINE configuration c1 ... c5 (c4 with --batch 64)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--hbm-batch", type=int, default=0,
                    help="instead of the benchmark: HBM fraction of stages 4-6 on this many models (L2-exceeding)")
    ap.add_argument("--sfh-scale", type=float, default=1.0,
                    help="diagnostic: multiply every model's SFH (N_pix) by this factor; not a BASELINE workload")
    ap.add_argument("--sampler-mode", type=int, default=0, choices=[0, 1],
                    help="0: one Poisson draw per (pixel, point), the headline path; 1: aggregated sampler (PAPER.md:75 fn. 3)")
    ap.add_argument("--hbm-variant", default="all", choices=["all", "on", "off", "collapsed", "general"],
                    help="with --hbm-batch: run one variant only (noise on / off, collapsed Hess, general 2-D PSF)")
    ap.add_argument("--pipes", action="store_true",
                    help="instead of the benchmark: instruction-pipe micro-benchmarks (pcmd_pipe_bench), one JSON line")
    args = ap.parse_args()
    if args.pipes:
        run_pipes(args)
    elif args.hbm_batch > 0:
        run_hbm_stages(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.all_configs:
        for c in (1, 2, 3, 4, 5):
            a = argparse.Namespace(**vars(args))
            a.config, a.batch = c, (64 if c == 4 else 1)
            run_ours(a)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
