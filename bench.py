#!/usr/bin/env python
"""bench.py -- headline measurement of libgbk on B200 (contract: see the task prompt / DESIGN.md
"Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config C]

One "step" = one pass of the whole hot path over one batch:
`gbk_eval_batch` on K_rows parameter rows of BASELINE.json config 3 (64x64 spaxels x 64 channels,
K_rows = 4096 = one nested-grid level, chi^2 only), the configuration BASELINE.json's metric is
quoted on.  Prints ONE JSON line on rank 0.

  value      model evaluations / s, inputs resident in HBM, CUDA events around each launch on the
             launching stream, L2 flushed between timed launches, max over ranks
  e2e        the same through gbk_eval_batch_host: HOST (pinned) params in, HOST chi^2 out, copies
             inside the timed region (wall clock around a blocking call)
  roofline   the fused kernel against the SM arithmetic pipe that bounds it (FP32 FMA pipe, "alu"):
             `frac` by the algorithmic count of SURVEY.md section 8(d), `frac_executed` by the work the
             kernel reports through gbk_eval_batch_counted in this very run
  cpu_baseline   the CPU oracle (oracle/, untouched) on a bounded sample of the same rows
  configs    all five BASELINE.json configs at their own K: device ms per launch (median of >= 20,
             L2 flushed), evals/s, tiling, op counts and fractions, the oracle beside each

The oracle is executed only by the cpu_baseline leg and by --impl reference.  Nothing here reads
/root/reference.  All inputs are seeded and synthetic (paper_1510_01815_b200/workloads.py).
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1510_01815_b200 import workloads as wl  # noqa: E402

METRIC = "model evals/sec (cube+PSF+moments+\u03c7\u00b2) at 64\u00d764\u00d764, K=4096; % FP32/SFU peak"
UNIT = "evals/s"
SM_COUNT_B200 = 148
MUFU_LANES_PER_SM_CLK = 16      # 4 SMSPs x 4 MUFU lanes
FP32_LANES_PER_SM_CLK = 128


# ------------------------------------------------------------------------------ inputs ----

def true_row_for(cfg: int, w: wl.Workload, rng) -> np.ndarray:
    true = wl.draw_rows(w, rng, 1)[0]
    if cfg == 3:   # centre and V_sys fixed at truth; DESIGN.md "Input recipe"
        true[[wl.IX_XO, wl.IX_YO, wl.IX_VSYS]] = (31.7, 32.4, 0.0)
    return true


def batch_rows(cfg: int, w: wl.Workload, true: np.ndarray, rng, n_batches: int) -> list:
    """The parameter batches the timed steps cycle through (float32 [K, P] each)."""
    if cfg == 3:   # the four nested-grid levels, each 8^4 nodes, re-centred on the truth
        centre = true[[wl.IX_PA, wl.IX_INC, wl.IX_VT, wl.IX_RT]].astype(np.float64)
        return [wl.nested_grid_rows(w, true, level=l, centre=None if l == 0 else centre)
                for l in range(min(4, max(1, n_batches)))]
    return [wl.draw_rows(w, rng, w.K) for _ in range(min(4, max(1, n_batches)))]


def desc_for(w: wl.Workload, obs: wl.Observed) -> dict:
    d = dict(nx=w.nx, ny=w.ny, nv=w.nv, u=w.u, v_center=w.v_center, dv=w.dv, rc_model=w.rc_model,
             n_gal=1, vobs=obs.vobs, verr=obs.verr, sobs=obs.sobs, serr=obs.serr, mask=obs.mask,
             psf_kind=w.psf_kind, lsf_sigma=w.lsf_sigma)
    if w.psf_kind == wl.PSF_GAUSSIAN:
        d["psf_fwhm"] = np.asarray([w.psf_fwhm], dtype=np.float32)
    else:
        d["psf_image"] = wl.moffat_image(w.psf_fwhm, w.moffat_beta, w.psf_n)
    return d


def observation_from_gpu(gbk, torch, w: wl.Workload, true: np.ndarray, rng) -> wl.Observed:
    """Clean maps of the true row from the CUDA path itself (the GPU leg never calls the oracle),
    then seeded noise / errors / mask."""
    blank = wl.Observed(*(np.zeros((1, w.ny, w.nx), np.float32) for _ in range(2)),
                        *(np.zeros((1, w.ny, w.nx), np.float32) for _ in range(2)),
                        np.zeros((1, w.ny, w.nx), np.uint8))
    blank.verr[:] = 1.0
    blank.serr[:] = 1.0
    with gbk.Problem(**desc_for(w, blank)) as prob:
        out = prob.eval(torch.from_numpy(true[None].copy()).cuda(), want_maps=True)
        torch.cuda.synchronize()
        m0, m1, m2 = (out[k].cpu().numpy().astype(np.float64) for k in ("m0", "m1", "m2"))
    return wl.observe(w, m0, m1, m2, rng)


# ------------------------------------------------------------------------------ clocks ----

class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (profiling recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.thread.join(timeout=2)
        rows = [l for (t, l) in self.lines if t0 <= t <= t1 + 0.11] or [l for (_, l) in self.lines]
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for l in rows:
            f = [x.strip() for x in l.split(",")]
            try:
                sm.append(float(f[0])), mx.append(float(f[1])), pw.append(float(f[2]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------- the CPU oracle legs ----

def oracle_grid(oracle, w: wl.Workload):
    """Oracle Grid of workload w (its own tap builders; nothing shared with the CUDA path)."""
    f32 = lambda x: float(np.float32(x))
    if w.psf_kind == wl.PSF_GAUSSIAN:
        psf = oracle.psf_gaussian_image(f32(w.psf_fwhm), w.u)
    else:
        img = wl.moffat_image(w.psf_fwhm, w.moffat_beta, w.psf_n).astype(np.float64)
        psf = img / img.sum()
    lsf = oracle.gaussian_taps(f32(w.lsf_sigma) / f32(w.dv) if w.lsf_sigma > 0 else 0.0)
    return oracle.Grid(nx=w.nx, ny=w.ny, nv=w.nv, u=w.u, v_center=f32(w.v_center), dv=f32(w.dv),
                       rc_model=w.rc_model, psf=psf, lsf=lsf)


def host_cores() -> int:
    return len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)


def oracle_case(cfg: int):
    """Workload, oracle grid, observation (clean maps from the ORACLE here) and batches."""
    from oracle import gbk_oracle as oracle
    w = wl.config(cfg)
    if cfg == 5:      # one galaxy of the survey at the mean PSF FWHM (the GPU leg mixes 1000 of them)
        w = w.scaled(psf_fwhm=2.75)
    rng = wl.rng_for(cfg, 100)
    true = true_row_for(cfg, w, rng)
    g = oracle_grid(oracle, w)
    m0, m1, m2 = oracle.model_maps(g, true.astype(np.float64))
    obs = wl.observe(w, m0[None], m1[None], m2[None], rng)
    return oracle, w, g, obs, batch_rows(cfg, w, true, rng, 4)


def time_oracle(cfg: int, rows_per_step: int, steps: int, warmup: int, threads: int) -> dict:
    """The oracle as it stands on `threads` host threads: `steps` timed calls of `rows_per_step`
    rows each (the first rows of the batches the GPU leg cycles through)."""
    oracle, w, g, obs, batches = oracle_case(cfg)
    o = obs
    call = lambda rows: oracle.eval_rows(g, o.vobs[0], o.verr[0], o.sobs[0], o.serr[0], o.mask[0],
                                         rows, nthreads=threads)
    take = lambda b, n: b[:n] if len(b) >= n else np.resize(b, (n, b.shape[1]))   # K < sample: rows repeated
    for i in range(warmup):
        call(take(batches[i % len(batches)], max(1, min(rows_per_step, threads))))
    t0 = time.perf_counter()
    for i in range(steps):
        call(take(batches[i % len(batches)], rows_per_step))
    dt = time.perf_counter() - t0
    return {"value": rows_per_step * steps / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
            "seconds": dt,
            "sample": f"first {rows_per_step} rows of each of {steps} config-{cfg} batches "
                      f"(K={w.K} per batch on the GPU), double precision, OpenMP over rows"}


def time_fast_cpu(cfg: int, rows_per_step: int, threads: int) -> dict | None:
    """A second, clearly labelled CPU baseline: oracle/gbk_cpu_fast.c, the straightforward optimised CPU
    restatement (float32, moment-first, separable PSF, OpenMP + SIMD) -- Gaussian-PSF configs only."""
    from oracle import gbk_cpu_fast as fast
    oracle, w, g, obs, batches = oracle_case(cfg)
    if w.psf_kind != wl.PSF_GAUSSIAN:
        return None
    f32 = lambda x: float(np.float32(x))
    psf1d = oracle.gaussian_taps(w.u * oracle.fwhm_to_sigma(f32(w.psf_fwhm)))
    lsf = oracle.gaussian_taps(f32(w.lsf_sigma) / f32(w.dv) if w.lsf_sigma > 0 else 0.0)
    b = batches[0]
    rows = b[:rows_per_step] if len(b) >= rows_per_step else np.resize(b, (rows_per_step, b.shape[1]))
    call = lambda r: fast.eval_rows(nx=w.nx, ny=w.ny, nv=w.nv, u=w.u, v_center=w.v_center, dv=w.dv,
                                    rc_model=w.rc_model, psf_taps=psf1d, lsf_taps=lsf, vobs=obs.vobs[0],
                                    verr=obs.verr[0], sobs=obs.sobs[0], serr=obs.serr[0], mask=obs.mask[0],
                                    params=r, nthreads=threads)
    call(rows[:max(1, threads)])
    t0 = time.perf_counter()
    call(rows)
    dt = time.perf_counter() - t0
    return {"value": rows_per_step / dt, "unit": UNIT, "cores": threads, "kind": "optimised-cpu",
            "seconds": dt,
            "sample": f"first {rows_per_step} rows of a config-{cfg} batch; float32, moment-first identity, separable "
                      f"PSF, LSF folded into channel weights, OpenMP over rows + SIMD channel loop "
                      f"(gcc -O3 -ffast-math -march=native)",
            "note": "NOT the parity oracle: a tuned CPU restatement, checked against the oracle by tests/test_cpu_fast.py"}


def run_reference(args, ranks) -> None:
    """--impl reference: the oracle is this tier's reference arm.  Rank 0 only."""
    if not ranks.is_main:
        return
    cores = host_cores()
    rows_per_step = args.ref_rows or max(cores, 4 * cores)
    r = time_oracle(args.config, rows_per_step, args.steps, min(args.warmup, 1), cores)
    w = wl.config(args.config)
    line = {
        "impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT,
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * r["seconds"] / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"config {args.config}: {w.nx}x{w.ny} spaxels x {w.nv} channels, "
                               f"u={w.u}; each step = {rows_per_step} rows sampled from a K={w.K} batch",
                   "rows_per_step": rows_per_step},
        "cpu_baseline": {k: r[k] for k in ("value", "unit", "cores", "kind", "sample")},
        "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# --------------------------------------------------------------------------- the GPU leg ----

def measure_pipe_peaks(gbk, torch, sm_count: int) -> dict:
    """Register-only MUFU.EX2 and FFMA loops on every SM (gbk_probe_pipe): the measured
    denominators quoted beside the derived ones."""
    sink = torch.zeros(4, dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    out = {}
    for which, name, iters in ((0, "mufu", 4096), (1, "ffma", 32768)):
        best = 0.0
        for rep in range(4):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ops = gbk.gbk_probe_pipe(which, iters, sm_count * 8, 256, sink, st)
            e1.record()
            e1.synchronize()
            if rep:
                best = max(best, ops / (e0.elapsed_time(e1) * 1e-3))
        out[name + "_gops_measured"] = best / 1e9
    return out


def psf_radius(w: wl.Workload, fwhm: float) -> int:
    """Tap radius the library derives for a Gaussian PSF (include/gbk.h: R = ceil(4 sigma_fine))."""
    if w.psf_kind == wl.PSF_IMAGE:
        return w.psf_n // 2
    if fwhm <= 0:
        return 0
    return int(np.ceil(4.0 * w.u * float(np.float32(fwhm)) / (2.0 * np.sqrt(2.0 * np.log(2.0)))))


def ext_samples_per_eval(info, w: wl.Workload, R: int) -> int:
    """Extended fine samples a row of PSF radius R EVALUATES in the kernel's tiling: sum over its tiles of
    (tw+2R)(th+2R) -- every tile carries its own PSF halo."""
    tw, th, fw, fh = info.tile_w * w.u, info.tile_h * w.u, w.nx * w.u, w.ny * w.u
    tot = 0
    for ty in range(info.tiles_y):
        for tx in range(info.tiles_x):
            tot += (min(tw, fw - tx * tw) + 2 * R) * (min(th, fh - ty * th) + 2 * R)
    return tot


def op_counts(info, w: wl.Workload, radii: np.ndarray) -> dict:
    """Algorithmic FP32 lane-ops per evaluation: 5 per extended voxel, 45 per
    extended sample, 3 maps x (2 x taps separable | taps^2 image) per fine pixel, 12 per spaxel --
    averaged over the PSF radii of the batch's rows.  "Extended" is the WHOLE FIELD plus one PSF halo
    (SURVEY's table: 270 x 270 x 56 for config 4), whatever tiling the kernel uses: the halos that tiles
    re-evaluate are the kernel's overhead, not the method's work.  `*_tiled` are the figures of the tiling
    (equal for one tile per row: configs 3 and 5)."""
    nvx = info.nv + 2 * info.r_v
    fw, fh = w.u * w.nx, w.u * w.ny
    tot = tot_tiled = samples = samples_tiled = 0.0
    for R in np.unique(radii):
        share = float(np.mean(radii == R))
        ns = (fw + 2 * int(R)) * (fh + 2 * int(R))
        ns_tiled = ext_samples_per_eval(info, w, int(R))
        taps = 2 * int(R) + 1
        psf = taps * taps if w.psf_kind == wl.PSF_IMAGE else 2 * taps
        rest = 3.0 * psf * fw * fh + 12.0 * w.nx * w.ny
        tot += share * (5.0 * ns * nvx + 45.0 * ns + rest)
        tot_tiled += share * (5.0 * ns_tiled * nvx + 45.0 * ns_tiled + rest)
        samples += share * ns
        samples_tiled += share * ns_tiled
    return {"ops_per_eval": tot, "ext_samples_per_eval": samples, "ext_voxels_per_eval": samples * nvx,
            "ops_per_eval_tiled": tot_tiled, "ext_samples_per_eval_tiled": samples_tiled,
            "ext_voxels_per_eval_tiled": samples_tiled * nvx}


def executed_ops(counters: np.ndarray, K: int, nominal: dict, info, w: wl.Workload) -> float:
    """FP32 lane-ops per evaluation the kernel executed, from its own work counters: a polynomial
    block costs 27 per pixel and 8 channels (three degree-7 Horner chains, the g0 P products and the
    restart), a directly summed channel 5 per voxel, the geometry 45 per sample of every warp item
    (128 samples, padding lanes included); PSF passes and moments as in the algorithmic count."""
    items, poly, direct = (float(counters[i]) for i in range(3))
    nvx = info.nv + 2 * info.r_v
    rest = nominal["ops_per_eval"] - 5.0 * nominal["ext_voxels_per_eval"] - 45.0 * nominal["ext_samples_per_eval"]
    return (poly * 128 * 27 + direct * 128 * 5 + items * 128 * 45) / K + rest


def build_case(gbk, torch, cfg: int, rank: int = 0) -> dict:
    """Problem, batches and PSF radii of BASELINE.json config `cfg` at its own K (seeded, synthetic;
    clean maps from the CUDA path itself)."""
    w = wl.config(cfg)
    rng = wl.rng_for(cfg, 100 + rank)
    if cfg == 5:   # the 1000-galaxy survey: own PSF per galaxy, per-spaxel errors, LM-shaped slots
        n = w.n_gal
        fwhms = wl.galaxy_fwhms(w, rng)
        trues = wl.draw_rows(w, rng, n)
        shp = (n, w.ny, w.nx)
        blank = wl.Observed(np.zeros(shp, np.float32), np.ones(shp, np.float32), np.zeros(shp, np.float32),
                            np.ones(shp, np.float32), np.zeros(shp, np.uint8))
        d = desc_for(w, blank)
        d.update(n_gal=n, psf_fwhm=fwhms, psf_per_gal=True)
        gi = torch.arange(n, dtype=torch.int32, device="cuda")
        with gbk.Problem(**d) as prob:
            o = prob.eval(torch.from_numpy(trues).cuda(), gi, want_maps=True)
            torch.cuda.synchronize()
            m0, m1, m2 = (o[k].cpu().numpy().astype(np.float64) for k in ("m0", "m1", "m2"))
        obs = wl.observe(w, m0, m1, m2, rng)
        d = desc_for(w, obs)
        d.update(n_gal=n, psf_fwhm=fwhms, psf_per_gal=True)
        slots = w.K // 8                                  # 2048 LM slots of base + 7 differences
        gal = (np.arange(slots) % n).astype(np.int32)
        batches = []
        for _ in range(2):
            starts = trues[gal].astype(np.float64)
            b = wl.box(w)
            free7 = [wl.IX_XO, wl.IX_YO, wl.IX_PA, wl.IX_INC, wl.IX_VSYS, wl.IX_VT, wl.IX_RT]
            starts[:, free7] += 0.05 * (b[free7, 1] - b[free7, 0]) * rng.uniform(-1, 1, (slots, 7))
            starts[:, wl.IX_INC] = np.clip(starts[:, wl.IX_INC], 20.0, 80.0)
            starts[:, wl.IX_RT] = np.clip(starts[:, wl.IX_RT], 1.0, 8.0)
            batches.append(np.concatenate([wl.lm_rows(w, r) for r in starts]).astype(np.float32))
        gal_rows = np.repeat(gal, 8)
        radii = np.asarray([psf_radius(w, f) for f in fwhms])[gal_rows]
        return dict(cfg=cfg, w=w, desc=d, batches=batches, gal=gal_rows, radii=radii, true=trues[0],
                    what=f"{n} galaxies with their own PSF (R 3..7), {slots} LM slots x 8 rows, gal_index mixed")
    true = true_row_for(cfg, w, rng)
    obs = observation_from_gpu(gbk, torch, w, true, rng)
    if cfg == 1:
        batches = [wl.cfg1_trial_row()]
        what = "the trial row (K = 1), chi2 only"
    elif cfg == 2:
        batches = [wl.lm_rows(w, r) for r in wl.draw_rows(w, rng, 4)]
        what = "one LM iteration: base row + 7 forward differences (K = 8)"
    elif cfg == 3:
        batches = batch_rows(cfg, w, true, rng, 4)
        what = "nested-grid levels 0-3 cycled (K = 8^4), chi2 only"
    else:
        batches = batch_rows(cfg, w, true, rng, 4)
        what = "K = 256 rows uniform in the prior box (nested-sampling batch), chi2 only"
    K = batches[0].shape[0]
    radii = np.full(K, psf_radius(w, w.psf_fwhm))
    return dict(cfg=cfg, w=w, desc=desc_for(w, obs), batches=batches, gal=None, radii=radii, true=true,
                what=what)


def time_case(gbk, torch, case: dict, launches: int, flush, sm_max_mhz: float, tile=(0, 0)) -> dict:
    """Device time per launch of one config: CUDA events on the launching stream around every launch,
    L2 flushed in between; then one counted launch for the executed-work fraction."""
    w = case["w"]
    with gbk.Problem(**case["desc"], tile_w=tile[0], tile_h=tile[1]) as prob:
        info = prob.info
        dev = [torch.from_numpy(b).cuda() for b in case["batches"]]
        gal = None if case["gal"] is None else torch.from_numpy(case["gal"]).cuda()
        K = dev[0].shape[0]
        chi2 = torch.empty(K, dtype=torch.float32, device="cuda")
        stream = torch.cuda.current_stream()
        st = stream.cuda_stream
        for i in range(3):
            flush.zero_()
            gbk.gbk_eval_batch(prob.handle, dev[i % len(dev)], gal, K, chi2, stream=st)
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
              for _ in range(launches)]
        for i in range(launches):
            flush.zero_()
            ev[i][0].record(stream)
            gbk.gbk_eval_batch(prob.handle, dev[i % len(dev)], gal, K, chi2, stream=st)
            ev[i][1].record(stream)
        torch.cuda.synchronize()
        ms = [a.elapsed_time(b) for a, b in ev]
        counters = torch.zeros(gbk.GBK_N_COUNTERS, dtype=torch.int64, device="cuda")
        gbk.gbk_eval_batch_counted(prob.handle, dev[0], gal, K, chi2, counters, stream=st)
        torch.cuda.synchronize()
        cnt = counters.cpu().numpy()
        # which tiling the library picked for this K (levels are chosen per call)
        nominal = op_counts(info, w, case["radii"])
    med = statistics.median(ms)
    peak = info.sm_count * FP32_LANES_PER_SM_CLK * sm_max_mhz * 1e6 / 1e9
    ex = executed_ops(cnt, K, nominal, info, w)
    out = {"workload": f"config {case['cfg']}: {w.nx}x{w.ny} spaxels x {w.nv} channels, u={w.u}; {case['what']}",
           "K": K, "launches": launches, "ms_per_launch_median": med, "ms_per_launch_min": min(ms),
           "evals_per_s": K / (med * 1e-3), "ext_voxels_per_s": nominal["ext_voxels_per_eval"] * K / (med * 1e-3),
           "tile_of_large_batches": [info.tile_w, info.tile_h], "block_threads": info.block_threads,
           "ops_per_eval": int(nominal["ops_per_eval"]),
           "frac": nominal["ops_per_eval"] * K / (med * 1e-3) / 1e9 / peak,
           "ops_per_eval_tiled": int(nominal["ops_per_eval_tiled"]),
           "frac_tiled": nominal["ops_per_eval_tiled"] * K / (med * 1e-3) / 1e9 / peak,
           "ops_executed_per_eval": int(ex), "frac_executed": ex * K / (med * 1e-3) / 1e9 / peak,
           "voxel_loop": {"warp_items": int(cnt[0]), "poly_blocks": int(cnt[1]), "direct_channels": int(cnt[2]),
                          "precise_items": int(cnt[3])},
           "checksum": float(chi2[torch.isfinite(chi2)].double().sum().item())}
    if K * max(info.tiles_x * info.tiles_y, 1) < info.sm_count:
        out["note"] = "launch-latency-bound: fewer thread blocks than SMs at the tile of large batches; " \
                      "the library picks smaller tiles for such K"
    return out


def oracle_for_config(cfg: int, cores: int) -> dict:
    """The oracle's evals/s on a bounded sample of config `cfg` (a few CPU-seconds)."""
    rows = {1: 4 * cores, 2: cores, 3: 8 * cores, 4: cores, 5: 4 * cores}[cfg]
    r = time_oracle(cfg, rows, 1, 0, cores)
    return {"oracle_evals_per_s": r["value"], "oracle_cores": cores, "oracle_sample": r["sample"]}


def run_ours(args, ranks) -> None:
    import torch
    from paper_1510_01815_b200 import dist, gbk
    gbk.lib()                                   # raises if libgbk.so is missing: no fallback
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(ranks.local_rank)
    cfg = args.config
    case = build_case(gbk, torch, cfg, ranks.rank)     # every rank its own galaxy: weak scaling
    w, batches = case["w"], case["batches"]
    K = batches[0].shape[0]
    prob = gbk.Problem(**case["desc"], tile_w=args.tile[0], tile_h=args.tile[1])
    info = prob.info
    dev_batches = [torch.from_numpy(b).cuda() for b in batches]
    gal = None if case["gal"] is None else torch.from_numpy(case["gal"]).cuda()
    chi2 = torch.empty(K, dtype=torch.float32, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB of L2
    stream = torch.cuda.current_stream()
    st = stream.cuda_stream
    launches_per_step = 1          # one fused kernel per batch, tiled or not

    def step(i):
        gbk.gbk_eval_batch(prob.handle, dev_batches[i % len(dev_batches)], gal, K, chi2, stream=st)

    sampler = ClockSampler(ranks.local_rank)
    sampler.start()
    t_warm = time.perf_counter()
    for i in range(max(args.warmup, 3)):
        flush.zero_()
        step(i)
    torch.cuda.synchronize()

    # ---- device-resident timing: CUDA events on the launching stream, L2 flushed between ----
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True))
          for _ in range(args.steps)]
    dist.barrier(ranks)
    torch.cuda.synchronize()
    for i in range(args.steps):
        flush.zero_()
        ev[i][0].record(stream)
        step(i)
        ev[i][1].record(stream)
    torch.cuda.synchronize()
    dist.barrier(ranks)
    ms = [a.elapsed_time(b) for a, b in ev]
    sec_rank = sum(ms) * 1e-3
    checksum = float(chi2[torch.isfinite(chi2)].sum().item())
    value, sec_max = dist.aggregate_throughput(ranks, K * args.steps, sec_rank)

    # ---- end to end through the host entry: pinned host params in, host chi^2 out ----------
    host_batches = [torch.from_numpy(b).pin_memory() for b in batches]
    host_gal = None if case["gal"] is None else torch.from_numpy(case["gal"]).pin_memory()
    host_chi2 = torch.empty(K, dtype=torch.float32).pin_memory()
    for i in range(3):
        gbk.gbk_eval_batch_host(prob.handle, host_batches[i % len(host_batches)], host_gal, K, host_chi2, st)
    dist.barrier(ranks)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(args.steps):
        gbk.gbk_eval_batch_host(prob.handle, host_batches[i % len(host_batches)], host_gal, K, host_chi2, st)
    torch.cuda.synchronize()
    e2e_rank = time.perf_counter() - t0
    t_end = time.perf_counter()
    e2e_value, _ = dist.aggregate_throughput(ranks, K * args.steps, e2e_rank)
    clocks = sampler.stop(t_warm, t_end)
    same = bool(np.array_equal(host_chi2.numpy(),
                               _chi2_of(gbk, prob, dev_batches[(args.steps - 1) % len(dev_batches)], gal, K, torch)))

    # ---- roofline of the dominant kernel (the fused kernel: the only one of the step) -------
    nominal = op_counts(info, w, case["radii"])
    counters = torch.zeros(gbk.GBK_N_COUNTERS, dtype=torch.int64, device="cuda")
    for b in dev_batches:                                         # the same batches the timed steps cycle
        gbk.gbk_eval_batch_counted(prob.handle, b, gal, K, chi2, counters, stream=st)
    torch.cuda.synchronize()
    cnt = counters.cpu().numpy()
    executed = executed_ops(cnt, K * len(dev_batches), nominal, info, w)
    nvx = info.nv + 2 * info.r_v
    mufu_per_eval = nominal["ext_voxels_per_eval"] + 3 * nominal["ext_samples_per_eval"]
    sm_max = (clocks.get("sm_max_mhz") or 1965.0)
    # The voxel loop sums the Gaussian line over blocks of 8 channels as a polynomial in the line ratio
    # (two MUFU.EX2 per pixel and block, no ex2 per voxel), so the binding pipe is the FP32 FMA pipe
    # (quote the fraction against that pipe); the MUFU figures of a direct
    # evaluation are kept beside it.
    peak_fp32 = info.sm_count * FP32_LANES_PER_SM_CLK * sm_max * 1e6 / 1e9           # G lane-op/s
    peak_mufu = info.sm_count * MUFU_LANES_PER_SM_CLK * sm_max * 1e6 / 1e9
    evals_per_s_rank = K * args.steps / sec_rank
    achieved = nominal["ops_per_eval"] * evals_per_s_rank / 1e9
    roofline = {"bound": "alu", "pipe": "FP32 FMA pipe, 128 lanes/clk/SM (FFMA2 = 2 lanes x 2 clk)",
                "achieved": achieved, "peak": peak_fp32, "unit": "Gop/s", "frac": achieved / peak_fp32,
                # dram__bytes_read.sum + dram__bytes_write.sum of ONE launch, copied from the committed ncu --set full
                # capture of this command (config 3 only) -- NOT measured in this run
                "traffic": 319744 if (cfg == 3 and tuple(args.tile) == (0, 0)) else None,
                "traffic_unit": "bytes per launch",
                "traffic_source": "profiles/r02_fused_kernel_ncu.md (319.7 KB read + 0 B written -- the 16 KB of chi^2 stay in L2 -- per launch of 4096 "
                                  "rows); a constant from that capture, not measured live; irrelevant to an ALU-bound kernel",
                "peak_how": f"derived: {info.sm_count} SMs x 128 FP32 lanes x {sm_max:.0f} MHz (max SM clock)",
                "ops_per_eval": int(nominal["ops_per_eval"]),
                "ops_how": "ALGORITHMIC FP32 lane-ops of SURVEY.md 8(d): 5/ext voxel + 45/ext sample + 3 maps x "
                           "(2 x taps separable | taps^2 image)/fine pixel + 12/spaxel; ext = the whole field plus ONE "
                           "PSF halo, whatever the tiling (halos re-evaluated per tile are overhead, not work)",
                "ops_per_eval_tiled": int(nominal["ops_per_eval_tiled"]),
                "ops_executed_per_eval": int(executed),
                "achieved_executed": executed * evals_per_s_rank / 1e9,
                "frac_executed": executed * evals_per_s_rank / 1e9 / peak_fp32,
                "executed_how": "counted by the kernel in this run (gbk_eval_batch_counted on the timed batches): "
                                "27 lane-ops per pixel and executed 8-channel polynomial block, 5 per directly summed "
                                "voxel, 45 per sample of every warp item; PSF passes and moments as in ops_per_eval",
                "voxel_loop": {"warp_items": int(cnt[0]), "poly_blocks": int(cnt[1]),
                               "direct_channels": int(cnt[2]), "precise_items": int(cnt[3]),
                               "channels_summed_per_sample": float((cnt[1] * 8 + cnt[2]) / max(cnt[0], 1)),
                               "extended_channels": int(nvx)},
                "note": "frac follows the contract (algorithmic work of SURVEY.md 8(d) / time / peak): it says how fast "
                        "the method's nominal work gets done and can exceed what the pipe executes, because the kernel "
                        "sums a line only where it is non-negligible (lines centred in the band: |d| < 6.5, i.e. beyond "
                        "7.7 sigma_0 left out, < 2^-42 of the sum) and as a block polynomial (27 lane-ops per 8 voxels "
                        "instead of 40).  frac_executed is the FP32 work actually executed / time / peak, the figure to "
                        "compare with ncu's FMA-pipe utilisation in profiles/",
                "mufu_ops_per_eval_direct": int(mufu_per_eval),
                "mufu_frac_if_direct": mufu_per_eval * evals_per_s_rank / 1e9 / peak_mufu,
                "kernel_ms_avg": statistics.mean(ms), "kernel_ms_median": statistics.median(ms),
                "kernel_ms_min": min(ms)}
    if ranks.is_main:
        pk = measure_pipe_peaks(gbk, torch, info.sm_count)
        roofline.update(pk)
        roofline["frac_of_measured"] = achieved / pk["ffma_gops_measured"]
        roofline["frac_executed_of_measured"] = roofline["achieved_executed"] / pk["ffma_gops_measured"]
        if clocks.get("sm_mhz"):
            roofline["frac_at_sampled_clock"] = achieved / (peak_fp32 * clocks["sm_mhz"] / sm_max)

    cpu = None
    cores = host_cores()
    if ranks.is_main and ranks.world == 1 and not args.no_cpu_baseline:
        cpu = time_oracle(cfg, args.cpu_rows or 32 * cores, 1, 1, cores)
        one = time_oracle(cfg, 24, 1, 1, 1)          # the paper's single-thread column
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample")}
        cpu["value_1_thread"] = one["value"]
        cpu["sample_1_thread"] = one["sample"]
        try:
            cpu["optimised_cpu"] = time_fast_cpu(cfg, 128 * cores, cores)
        except Exception as e:   # gcc flags unavailable on some host: the labelled extra is optional
            cpu["optimised_cpu"] = {"unavailable": str(e)[:200]}
        cpu["note"] = ("the parity oracle as it stands: the paper's definition written out literally in FP64 (materialised "
                       "cube, direct non-separable PSF sum per channel, gcc -O2, OpenMP over rows only) -- a correctness "
                       "reference, NOT a tuned CPU implementation; the GPU/oracle ratio says nothing about kernel quality")

    # ---- all five configs at their own K (rank 0; outside the timed region) -----------------
    configs = None
    if ranks.is_main and not args.no_configs:
        configs = {}
        for c in (1, 2, 3, 4, 5):
            cc = case if c == cfg else build_case(gbk, torch, c, ranks.rank)
            entry = time_case(gbk, torch, cc, max(20, args.config_launches), flush, sm_max,
                              tile=args.tile if c == cfg else (0, 0))
            if ranks.world == 1 and not args.no_cpu_baseline:
                entry.update(oracle_for_config(c, cores))
            configs[f"cfg{c}"] = entry

    unfused = time_unfused(gbk, torch, prob, dev_batches[0], gal, K, info) \
        if (ranks.is_main and not args.no_fits) else None
    vfield = time_vfield(gbk, torch, prob, dev_batches[0], gal, K, info, sm_max) \
        if (ranks.is_main and not args.no_fits) else None
    fits = time_fits(gbk, torch, prob, w, case["true"]) if (ranks.is_main and cfg == 3 and not args.no_fits) else None
    if ranks.is_main:
        core_vox = w.nx * w.ny * w.nv * w.u * w.u
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": ranks.world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": 1e3 * sec_max / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": f"config {cfg}: {w.nx}x{w.ny} spaxels x {w.nv} channels, u={w.u}, "
                                   f"K={K} rows per launch; {case['what']}",
                       "rows_per_launch": K, "l2": "flushed between timed launches (256 MiB memset)",
                       "tile": [info.tile_w, info.tile_h], "block_threads": info.block_threads,
                       "smem_bytes": info.smem_bytes, "blocks_per_sm": info.blocks_per_sm,
                       "ext_voxels_per_eval": int(nominal["ext_voxels_per_eval"]),
                       "parallelism": f"rows sharded, {ranks.world} rank(s), no collective"},
            "voxels_per_s": value * core_vox, "ext_voxels_per_s": value * nominal["ext_voxels_per_eval"],
            "e2e": {"value": e2e_value, "unit": UNIT,
                    "h2d_bytes_per_step": K * wl.P * 4 + (K * 4 if case["gal"] is not None else 0),
                    "d2h_bytes_per_step": K * 4, "matches_device_path": same},
            "gpu_launches": launches_per_step * args.steps,
            "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu, "checksum": checksum,
            "configs": configs, "fits": fits, "unfused": unfused, "vfield": vfield,
        }
        print(json.dumps(line), flush=True)
    prob.close()


def run_probe_umma() -> None:
    """--probe-umma: the tcgen05.mma sequence that one 64x64 tile of config 4's 15x15 PSF pass would need as a
    banded BF16 contraction (gbk_probe_umma), timed with CUDA events: how long the tensor pipe would be busy per
    tile, to set beside the FFMA2 pass (profiles/r02_tcgen05_probe.md)."""
    import torch
    from paper_1510_01815_b200 import gbk
    gbk.lib()
    torch.cuda.set_device(0)
    chk = torch.full((1,), -1.0, dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    out = {"probe": "tcgen05 banded contraction of the 15x15 pass", "sm_count": sms, "runs": []}
    for per_sm, iters in ((1, 400), (2, 400)):
        gbk.gbk_probe_umma(iters, per_sm * sms, chk, st)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        flops = gbk.gbk_probe_umma(iters, per_sm * sms, chk, st)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        out["runs"].append({"ctas_per_sm": per_sm, "tile_sequences_per_cta": iters, "ms": ms,
                            "tflops_bf16_issued": flops / ms / 1e9,
                            "us_of_tensor_pipe_per_tile_per_sm": ms * 1e3 / (iters * per_sm)})
    out["check_max_abs_error"] = float(chk[0].item())
    print(json.dumps(out), flush=True)


def time_fits(gbk, torch, prob3, w3, true3) -> dict:
    """Wall time to a converged fit through the host drivers (outside the timed region; rank 0):
    nested grids on the config-3 problem (4 levels x 8^4 rows) and LM on a config-2
    problem (64x64x128, u=2, 7 free parameters, K=8 per iteration)."""
    out = {}
    b = wl.box(w3)
    free4 = [wl.IX_PA, wl.IX_INC, wl.IX_VT, wl.IX_RT]
    dev_true = torch.from_numpy(np.ascontiguousarray(true3[None], dtype=np.float32)).cuda()
    chi_true = float(prob3.eval(dev_true)["chi2"].item())

    def ng_quality(best, chi):
        """Fit error beside the fit time.  V_t and i are degenerate along V_t sin i = const (PAPER.md:658-662,
        Fig. 12), so that product is reported too; chi2 <= chi2_of_truth means the grid found a node at least
        as good as the true row on this noisy data."""
        err = [float(abs(best[j] - true3[j])) for j in free4]
        err[0] = float(abs((err[0] + 180.0) % 360.0 - 180.0))
        vsini = lambda r: float(r[wl.IX_VT] * np.sin(np.radians(r[wl.IX_INC])))
        return {"abs_err": dict(zip(("pa_deg", "inc_deg", "vt_kms", "rt_px"), err)),
                "vt_sin_i_err_kms": abs(vsini(best) - vsini(true3)), "chi2": chi, "chi2_of_truth": chi_true,
                "table3_thresholds": {"pa_deg": 1.0, "inc_deg": 1.0, "vt_kms": 5.0, "rt_px": 1.0},
                "note": "data carry N(0, 5 km/s) noise; Table 3's thresholds (PAPER.md:408-414) are for noise-free mocks"}

    gbk.gbk_fit_ng(prob3.handle, true3, 0, free4, b[free4, 0], b[free4, 1], 8, 4)      # warm-up
    best, chi, st = gbk.gbk_fit_ng(prob3.handle, true3, 0, free4, b[free4, 0], b[free4, 1], 8, 4)
    out["ng_cfg3"] = {"ms": st["ms_total"], "evals": st["evals"], "levels": st["iterations"],
                      "what": "BASELINE.json config 3: 8^4 nodes over (PA, i, V_t, r_t), 4 levels", **ng_quality(best, chi)}
    # the paper's stopping rule: refine until the spacing is <= 0.1 (0.01 for r_t)
    acc = [0.1, 0.1, 0.1, 0.01]
    best, chi, st = gbk.gbk_fit_ng(prob3.handle, true3, 0, free4, b[free4, 0], b[free4, 1], 8, 30, accuracy=acc)
    out["ng_cfg3_to_accuracy"] = {"ms": st["ms_total"], "evals": st["evals"], "levels": st["iterations"],
                                  "converged": st["converged"], "accuracy": acc, **ng_quality(best, chi)}
    w2 = wl.config(2)
    rng = wl.rng_for(2, 200)
    true2 = wl.draw_rows(w2, rng, 1)[0]
    obs2 = observation_from_gpu(gbk, torch, w2, true2, rng)
    b2 = wl.box(w2)
    free7 = [wl.IX_XO, wl.IX_YO, wl.IX_PA, wl.IX_INC, wl.IX_VSYS, wl.IX_VT, wl.IX_RT]
    lo, hi = b2[free7, 0].copy(), b2[free7, 1].copy()
    lo[2], hi[2] = -360.0, 720.0                      # PA is periodic: no wall for LM
    start = true2.astype(np.float64)
    start[free7] += 0.1 * (b2[free7, 1] - b2[free7, 0]) * rng.uniform(-1, 1, 7)
    start[wl.IX_INC] = np.clip(start[wl.IX_INC], 20.0, 80.0)
    start[wl.IX_RT] = np.clip(start[wl.IX_RT], 1.0, 8.0)
    with gbk.Problem(**desc_for(w2, obs2)) as prob2:
        gbk.gbk_fit_lm(prob2.handle, start, None, free7, lo, hi, max_iter=2)             # warm-up
        rows, chi2, iters, st = gbk.gbk_fit_lm(prob2.handle, start, None, free7, lo, hi,
                                               rel_step=1e-3, max_iter=50, ftol=1e-6)
    out["lm_cfg2"] = {"ms": st["ms_total"], "evals": st["evals"], "iterations": int(iters[0]),
                      "converged": st["converged"], "failed": st["failed"], "chi2": float(chi2[0]),
                      "abs_err": [float(abs(rows[0, j] - true2[j])) for j in free7]}
    out["lm_cfg5_survey"] = time_survey(gbk, torch)
    # config 4: nested sampling with K = 256 live points and batches of 256 candidates
    # (256x256x48, Moffat 15x15 image PSF, ramp curve)
    w4 = wl.config(4)
    rng4 = wl.rng_for(4, 400)
    true4 = wl.draw_rows(w4, rng4, 1)[0]
    obs4 = observation_from_gpu(gbk, torch, w4, true4, rng4)
    b4 = wl.box(w4)
    free5 = [wl.IX_PA, wl.IX_INC, wl.IX_VSYS, wl.IX_VT, wl.IX_RT]
    with gbk.Problem(**desc_for(w4, obs4)) as prob4:
        r = gbk.gbk_fit_ns(prob4.handle, true4, 0, free5, b4[free5, 0], b4[free5, 1], n_live=256,
                           batch=256, max_batches=1000, enlarge=0.2, tol=0.05, seed=4)
    err = [float(abs(r["best_row"][j] - true4[j])) for j in free5]
    err[0] = float(abs((err[0] + 180.0) % 360.0 - 180.0))
    out["ns_cfg4"] = {"ms": r["stats"]["ms_total"], "evals": r["stats"]["evals"],
                      "batches": r["stats"]["iterations"], "converged": r["stats"]["converged"],
                      "chi2": r["best_chi2"], "log_evidence": r["log_evidence"], "abs_err": err}
    return out


def time_survey(gbk, torch) -> dict:
    """Config 5: 1000 synthetic galaxies (48x48x96, own PSF FWHM, per-spaxel errors, noise N(0, E)),
    LM with 7 free parameters from 2 starts per galaxy, all 2000 fits in ONE gbk_fit_lm call
    (mixed-galaxy batches of 16000 rows per Jacobian launch).  Reports galaxies fitted per hour."""
    w = wl.config(5)
    rng = wl.rng_for(5, 300)
    n = w.n_gal
    fwhms = wl.galaxy_fwhms(w, rng)
    trues = wl.draw_rows(w, rng, n)
    shp = (n, w.ny, w.nx)
    blank = wl.Observed(np.zeros(shp, np.float32), np.ones(shp, np.float32), np.zeros(shp, np.float32),
                        np.ones(shp, np.float32), np.zeros(shp, np.uint8))
    d = desc_for(w, blank)
    d.update(n_gal=n, psf_fwhm=fwhms, psf_per_gal=True)
    gi = torch.arange(n, dtype=torch.int32, device="cuda")
    with gbk.Problem(**d) as prob:
        o = prob.eval(torch.from_numpy(trues).cuda(), gi, want_maps=True)
        torch.cuda.synchronize()
        m0, m1, m2 = (o[k].cpu().numpy().astype(np.float64) for k in ("m0", "m1", "m2"))
    obs = wl.observe(w, m0, m1, m2, rng)
    d = desc_for(w, obs)
    d.update(n_gal=n, psf_fwhm=fwhms, psf_per_gal=True)
    b = wl.box(w)
    free7 = [wl.IX_XO, wl.IX_YO, wl.IX_PA, wl.IX_INC, wl.IX_VSYS, wl.IX_VT, wl.IX_RT]
    lo, hi = b[free7, 0].copy(), b[free7, 1].copy()
    lo[2], hi[2] = -360.0, 720.0
    starts = np.repeat(trues.astype(np.float64), 2, axis=0)
    starts[:, free7] += 0.1 * (b[free7, 1] - b[free7, 0]) * rng.uniform(-1, 1, (2 * n, 7))
    starts[:, wl.IX_INC] = np.clip(starts[:, wl.IX_INC], 20.0, 80.0)
    starts[:, wl.IX_RT] = np.clip(starts[:, wl.IX_RT], 1.0, 8.0)
    gal = np.repeat(np.arange(n, dtype=np.int32), 2)
    with gbk.Problem(**d) as prob:
        # warm-up at the full size, so that the library's cached workspace is sized before the timed call (on a
        # fresh box the first large cudaMalloc alone can take tens of ms of the wall-clock fit time)
        gbk.gbk_fit_lm(prob.handle, starts, gal, free7, lo, hi, max_iter=2)
        rows, chi2, iters, st = gbk.gbk_fit_lm(prob.handle, starts, gal, free7, lo, hi,
                                               rel_step=1e-3, max_iter=50, ftol=1e-6)
    best = np.where(chi2[0::2] <= chi2[1::2], 0, 1) + 2 * np.arange(n)
    err = np.abs(rows[best][:, free7].astype(np.float64) - trues[:, free7])
    err[:, 2] = np.abs((err[:, 2] + 180.0) % 360.0 - 180.0)
    thr = np.array([1.0, 1.0, 1.0, 1.0, 5.0, 5.0, 1.0])           # Table 3
    return {"ms": st["ms_total"], "galaxies": n, "fits": 2 * n, "evals": st["evals"],
            "launches": st["launches"], "max_iterations": st["iterations"],
            "converged": st["converged"], "failed": st["failed"],
            "galaxies_per_hour": n / (st["ms_total"] / 3.6e6),
            "within_table3_thresholds": [float(x) for x in (err <= thr).mean(axis=0)],
            "note": "noisy data (N(0,E), E~U[3,15] km/s): the thresholds are the paper's for noise-free mocks"}


def time_unfused(gbk, torch, prob, params, gal, K: int, info, reps: int = 5) -> dict:
    """The unfused comparison path (one kernel per pipeline step, FP32 cube in HBM) on the same
    batch: evals/s and achieved HBM GB/s = algorithmic bytes / device time, against the measured copy
    bandwidth of MEASURED_PEAKS.json (outside the timed region; rank 0)."""
    chi = torch.empty(K, dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    gbk.gbk_eval_batch_unfused(prob.handle, params, gal, K, chi, stream=st)      # warm-up + scratch
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        gbk.gbk_eval_batch_unfused(prob.handle, params, gal, K, chi, stream=st)
    e1.record()
    torch.cuda.synchronize()
    sec = e0.elapsed_time(e1) * 1e-3 / reps
    peak = None
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            peak = float(json.load(f)["hbm_gbs"])
    except (OSError, KeyError, ValueError):
        peak = 6500.0      # fallback of the profiling recipe's order; MEASURED_PEAKS.json absent
    gbs = info.unfused_bytes_per_eval * K / sec / 1e9
    out = {"value": K / sec, "unit": UNIT, "ms_per_batch": sec * 1e3, "bound": "hbm",
           "bytes_per_eval": int(info.unfused_bytes_per_eval), "achieved": gbs, "peak": peak,
           "unit_bw": "GB/s", "frac": gbs / peak,
           "bytes_how": "algorithmic: cube, LSF output and convolved cube each written once and read once"}
    # the Gaussian-profile extraction needs whole spectra, so it runs on this pipeline
    Kg = min(K, 1024)
    gbk.gbk_set_extraction(prob.handle, gbk.GBK_EXTRACT_GAUSSFIT)
    try:
        gbk.gbk_eval_batch(prob.handle, params[:Kg], None if gal is None else gal[:Kg], Kg, chi[:Kg], stream=st)
        torch.cuda.synchronize()
        e0.record()
        gbk.gbk_eval_batch(prob.handle, params[:Kg], None if gal is None else gal[:Kg], Kg, chi[:Kg], stream=st)
        e1.record()
        torch.cuda.synchronize()
        out["gaussfit_extraction"] = {"value": Kg / (e0.elapsed_time(e1) * 1e-3), "unit": UNIT, "rows": Kg,
                                      "ms_per_batch": e0.elapsed_time(e1),
                                      "note": "GBK_EXTRACT_GAUSSFIT: a Gaussian fitted to every spectrum instead of "
                                              "moments; cannot use the moment-first identity of the fused kernel"}
    finally:
        gbk.gbk_set_extraction(prob.handle, gbk.GBK_EXTRACT_MOMENTS)
    return out


def time_vfield(gbk, torch, prob, params, gal, K: int, info, sm_max_mhz: float, reps: int = 20) -> dict:
    """The paper's other strategy (velocity-field modelling) on the same batch:
    gbk_eval_vfield_batch, chi^2 only.  27 FP32 lane-ops per spaxel and row (eq. 1-4, 6, 8, residual,
    square-accumulate); bound by the FP32 pipe / issue, not by memory (the observation is read from
    L2 once per 4 rows).  Outside the timed region; rank 0."""
    chi = torch.empty(K, dtype=torch.float32, device="cuda")
    st = torch.cuda.current_stream().cuda_stream
    for _ in range(3):
        gbk.gbk_eval_vfield_batch(prob.handle, params, gal, K, chi, stream=st)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        gbk.gbk_eval_vfield_batch(prob.handle, params, gal, K, chi, stream=st)
    e1.record()
    torch.cuda.synchronize()
    sec = e0.elapsed_time(e1) * 1e-3 / reps
    ops = 27 * info.nx * info.ny
    peak = info.sm_count * FP32_LANES_PER_SM_CLK * sm_max_mhz * 1e6 / 1e9
    return {"value": K / sec, "unit": UNIT, "ms_per_batch": sec * 1e3, "bound": "alu",
            "ops_per_eval": ops, "achieved": ops * K / sec / 1e9, "peak": peak, "unit_ops": "Gop/s",
            "frac": ops * K / sec / 1e9 / peak,
            "note": "back-to-back launches on a warm L2 (64 KB observation, 160 KB parameters)"}


def _chi2_of(gbk, prob, params, gal, K, torch):
    out = torch.empty(K, dtype=torch.float32, device="cuda")
    gbk.gbk_eval_batch(prob.handle, params, gal, K, out, stream=torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    return out.cpu().numpy()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=400)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config number (metric: 3)")
    ap.add_argument("--cpu-rows", type=int, default=0, help="rows of the cpu_baseline sample")
    ap.add_argument("--ref-rows", type=int, default=0, help="rows per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-fits", action="store_true", help="skip the wall-time-to-fit legs")
    ap.add_argument("--no-configs", action="store_true", help="skip the per-config table (configs 1-5)")
    ap.add_argument("--config-launches", type=int, default=25, help="timed launches per config of the table")
    ap.add_argument("--probe-umma", action="store_true", help="run the tcgen05 probe of the 15x15 pass and exit")
    ap.add_argument("--tile", type=int, nargs=2, default=(0, 0), metavar=("W", "H"),
                    help="spatial tile in spaxels (default 0 0 = the library's automatic tiling)")
    args = ap.parse_args()
    from paper_1510_01815_b200 import dist
    if args.probe_umma:
        run_probe_umma()
        return
    if args.impl == "reference":
        rank = int(os.environ.get("RANK", "0"))
        if rank == 0:
            run_reference(args, dist.Ranks())
        return
    ranks = dist.init_from_env("nccl")
    try:
        run_ours(args, ranks)
    finally:
        dist.finalize(ranks)


if __name__ == "__main__":
    main()
