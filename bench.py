#!/usr/bin/env python
"""Benchmark of the TLS period-search hot path (libgtls, sm_100a) -- one JSON line on stdout.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c1..c4] [--impl reference]

A "step" is one pass of the whole hot path (fold, sort, pad + scans, per-window chi2, argmin,
SR/SDE) over one synthetic light curve.  Metric: (period x duration) trials per second
(BASELINE.json), plus seconds per light curve.  `value` is measured with all inputs resident in
HBM; `e2e` is the same metric through the C ABI with host buffers (H2D + D2H inside the timed
region).  `roofline` describes the dominant kernel (the in-transit chi2 kernel, fp64 ALU bound);
`cpu_baseline` is the CPU oracle timed on a bounded sample of the same workload.

For N > 1 (torchrun, one rank per GPU) every rank searches its own light curve of the same
shape (independent problems, weak scaling, no data-path collective); time is the max over ranks.
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

import gtls_inputs as gi  # noqa: E402

METRIC = "TLS (period x duration) trials/sec"
UNIT = "trials/s"
SM_COUNT = 148
DFMA_PER_CLK_PER_SM = 64            # fp64 FMA lanes per SM (B200_PROFILING.md / B300_MICROARCH.md unit counts)


def log(*a):
    print(*a, file=sys.stderr, flush=True)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons while the timed region runs."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.idx = gpu_index
        self.proc = None
        self.lines = []
        self.first = 0

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.idx}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "500"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def mark(self):
        """Start of the timed region: nvidia-smi is started before the warm-up (its start-up takes driver
        locks for most of a second, which a 10 ms step would see); samples before this call are dropped."""
        self.first = len(self.lines)

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines[self.first:] or self.lines[-1:]:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); mx.append(float(f[2])); pw.append(float(f[3]))
            except ValueError:
                continue
            for name, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        load = [s for s, p in zip(sm, pw) if p > 0.5 * max(pw)] or sm
        return {"sm_mhz": float(np.median(load)), "sm_max_mhz": float(max(mx)),
                "power_w_max": float(max(pw)), "samples": len(sm), "reasons": sorted(reasons)}


def build_workload(name: str, curve: int = 0, every: int = 1, dt0=None):
    cfg = int(name[1])
    w = gi.make_workload(cfg, curve=curve) if dt0 is None else gi.make_workload(cfg, curve=curve, dt0=float(dt0))
    return w.subset(every) if every > 1 else w


def oracle_sample(w, target_s: float):
    """Deterministic period subset sized so the oracle runs for about target_s seconds."""
    import oracle
    cores = oracle.num_threads()
    # ~1.2e-8 s per window-point per core measured for the plain oracle; refine with a probe
    probe = w.subset(max(1, w.n_per // 64))
    t0 = time.perf_counter()
    r = oracle.search(probe.lc.t, probe.lc.y, probe.lc.dy, probe.periods, probe.durations, probe.tmpl,
                      dt0=w.dt0)
    dt = time.perf_counter() - t0
    per_period = dt / probe.n_per
    want = int(max(8, min(w.n_per, target_s / max(per_period, 1e-9))))
    every = max(1, w.n_per // want)
    return w.subset(every), cores, every


def run_reference(args, w):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample per step."""
    import oracle
    sample, cores, every = oracle_sample(w, args.ref_seconds)
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        r = oracle.search(sample.lc.t, sample.lc.y, sample.lc.dy, sample.periods, sample.durations,
                          sample.tmpl, dt0=w.dt0)
        oracle.sde(r.chi2, 151)
        if i >= args.warmup:
            times.append(time.perf_counter() - t0)
    ms = 1e3 * float(np.mean(times))
    value = sample.trials / (ms / 1e3)
    desc = f"every {every}th period of {w.name} ({sample.n_per} of {w.n_per} periods, all {w.n_dur} durations)"
    return {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_desc(w), "sample": desc, "dt0": w.dt0},
        "s_per_light_curve_extrapolated": w.trials / value,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }


def run_survey(args, g, torch, devname):
    """c5: `--survey N` curves (each with its own Ofir grid and per-period durations) per step through
    gtls_search_batch, device-resident inputs; the same curves as a loop of gtls_search calls beside it."""
    ws_ = [gi.make_workload(5, curve=c) for c in range(args.survey)]
    cat = lambda xs, ax=0: np.ascontiguousarray(np.concatenate(xs, axis=ax))
    co = np.concatenate([[0], np.cumsum([w.lc.n for w in ws_])]).astype(np.int64)
    po = np.concatenate([[0], np.cumsum([w.n_per for w in ws_])]).astype(np.int64)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(devname)
    t, y, dy = (dev(cat([getattr(w.lc, k) for w in ws_])) for k in ("t", "y", "dy"))
    per, dur, tm = dev(cat([w.periods for w in ws_])), dev(cat([w.durations for w in ws_])), dev(ws_[0].tmpl)
    wsp = torch.empty(g.gtls_batch_workspace_bytes(co, po, ws_[0].n_dur), dtype=torch.uint8, device=devname)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=devname)
    trials = int(sum(w.trials for w in ws_))

    def timed(fn, sampler=None):
        for _ in range(max(args.warmup, 3)):
            fn()
        torch.cuda.synchronize()
        if sampler:
            sampler.mark()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for _ in range(args.steps):
            flush.zero_()
            r = fn()
        ev1.record()
        torch.cuda.synchronize()
        return ev0.elapsed_time(ev1) / args.steps, r

    dt0 = ws_[0].dt0 if args.dt0 is None else float(args.dt0)
    sampler = ClockSampler(int(devname.split(":")[1]))
    sampler.start()
    ms_batch, res = timed(lambda: g.gtls_search_batch(t, y, dy, co, per, po, dur, tm, dt0=dt0, sde_kernel=151,
                                                      workspace=wsp), sampler)
    one_ws = wsp[:max(g.gtls_workspace_bytes(w.lc.n, w.n_per, w.n_dur) for w in ws_)]

    def loop():
        for c in range(len(ws_)):
            r = g.gtls_search(t[co[c]:co[c + 1]], y[co[c]:co[c + 1]], dy[co[c]:co[c + 1]], per[po[c]:po[c + 1]],
                              dur[po[c]:po[c + 1]], tm, dt0=dt0, sde_kernel=151, workspace=one_ws)
        return r
    ms_loop, _ = timed(loop)
    clocks = sampler.stop()                      # both legs ran with the sampler polling
    found = sum(1 for c, w in enumerate(ws_) if c % 2 == 0 and res.summaries[c]["sde_max"] > 9.0)
    # per-curve agreement with the oracle (BASELINE.json config 5) on a seeded subset of the curves, in full:
    # same best period index and |SDE_max difference| <= 1e-6; chi2 and indices as in the parity tests
    agreement = None
    if args.survey_check > 0:
        import oracle
        rng = np.random.default_rng(20260700348)
        pick = sorted(rng.choice(len(ws_), size=min(args.survey_check, len(ws_)), replace=False).tolist())
        chi2_all, sde_all, best_all = res.chi2.cpu().numpy(), res.sde.cpu().numpy(), res.best()
        rows, t_or = [], 0.0
        for c in pick:
            w = ws_[c]
            t0 = time.perf_counter()
            ro = oracle.search(w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl, dt0=dt0)
            so = oracle.sde(ro.chi2, 151)
            t_or += time.perf_counter() - t0
            sl = slice(int(po[c]), int(po[c + 1]))
            strict = ro.gap > 1e-12 * np.abs(ro.chi2)
            mism = (best_all[sl]["dur_idx"] != ro.best["dur_idx"]) | (best_all[sl]["start"] != ro.best["start"])
            rows.append({"curve": c, "same_best_period_idx": bool(res.summaries[c]["best_period_idx"] == so.best_period_idx),
                         "sde_max_abs_diff": float(abs(res.summaries[c]["sde_max"] - so.sde.max())),
                         "sde_abs_diff_max": float(np.abs(sde_all[sl] - so.sde).max()),
                         "chi2_max_rel_err": float(np.max(np.abs(chi2_all[sl] - ro.chi2) / ro.chi2)),
                         "index_mismatches": int(np.sum(mism & strict))})
        ok = all(r["same_best_period_idx"] and r["sde_max_abs_diff"] <= 1e-6 and r["chi2_max_rel_err"] <= 1e-9 and
                 r["index_mismatches"] == 0 for r in rows)
        agreement = {"curves_checked": len(rows), "of": len(ws_), "all_agree": ok, "oracle_seconds": t_or,
                     "oracle_cores": oracle.num_threads(), "per_curve": rows}
    return {"metric": METRIC, "value": trials / (ms_batch / 1e3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_batch, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"c5 survey batch: {len(ws_)} independent 90-day curves (~{int(co[-1] / len(ws_))} points, "
                                   f"~{int(po[-1] / len(ws_))} periods x {ws_[0].n_dur} durations each), dt0={dt0}, one gtls_search_batch call",
                       "l2_flush": "256 MiB memset between timed steps"},
            "curves_per_s": len(ws_) / (ms_batch / 1e3), "ms_per_curve": ms_batch / len(ws_),
            "loop_of_single_calls": {"curves_per_s": len(ws_) / (ms_loop / 1e3), "ms_per_curve": ms_loop / len(ws_)},
            "curves_with_injected_transit_above_sde_9": f"{found} of {(len(ws_) + 1) // 2}",
            "per_curve_agreement": agreement,
            "clocks": clocks}


def chi2_stage_traffic(workload, period_tile):
    """DRAM bytes of the chi2 stage of one period tile, read from the committed ncu summary
    profiles/chi2_stage_traffic.csv (columns: workload, period_tile, dram_bytes, capture); None when
    no capture of this workload / tile size is on file."""
    path = os.path.join(ROOT, "profiles", "chi2_stage_traffic.csv")
    if workload is None or not os.path.exists(path):
        return None, "no ncu capture of this workload and tile size on file (profiles/chi2_stage_traffic.csv)"
    for ln in open(path).read().splitlines()[1:]:
        f = [x.strip() for x in ln.split(",")]
        if len(f) >= 4 and f[0] == workload and int(f[1]) == int(period_tile):
            return float(f[2]), f"profiles/chi2_stage_traffic.csv: {f[3]}"
    return None, "no ncu capture of this workload and tile size on file (profiles/chi2_stage_traffic.csv)"


def max_over_ranks(x: float, world: int, device="cpu") -> float:
    """Multi-rank runs (replicas only): the job time is the slowest rank's."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    tt = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def workload_desc(w) -> str:
    return (f"{w.name}: {w.lc.n} points, {w.n_per} periods (Ofir grid, OS=3), {w.n_dur} durations/period, "
            f"dt0={w.dt0}, template 512 nodes")


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=os.environ.get("GTLS_BENCH_WORKLOAD", "c4"))
    ap.add_argument("--impl", default="gtls", choices=["gtls", "reference"])
    ap.add_argument("--ref-seconds", type=float, default=20.0, help="CPU seconds per oracle sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--period-tile", type=int, default=0)
    ap.add_argument("--dt0", type=float, default=None,
                    help="T0 skip fraction of Eq. 18 (default: the workload's 0.05); the paper's sweep is 0.1 .. 0.01")
    ap.add_argument("--every", type=int, default=1,
                    help="profiling aid: search only every k-th period of the workload (default 1 = the "
                         "full workload; any other value is named in config.workload)")
    ap.add_argument("--peak-fp64", type=float, default=0.0, metavar="SECONDS",
                    help="measure the fp64 FMA rate of this GPU (gtls_peak_fp64: register-only DFMA kernel) as a "
                         "0.1 s burst and sustained over SECONDS, with the clocks seen; prints one JSON line")
    ap.add_argument("--survey-check", type=int, default=3,
                    help="survey mode: number of (seeded) curves searched in full by the CPU oracle for the "
                         "per-curve agreement report (0 = none)")
    ap.add_argument("--survey", type=int, default=0,
                    help="survey mode (BASELINE.json config 5): search this many c5 curves per step with one "
                         "gtls_search_batch call and report curves/s beside trials/s")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        if rank != 0:
            return 0
        w = build_workload(args.workload, every=args.every, dt0=args.dt0)
        print(json.dumps(run_reference(args, w)), flush=True)
        return 0

    import torch
    import torch.distributed as dist
    import paper_2607_00348_b200 as g

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    devname = f"cuda:{local_rank}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(devname))
    g.load_library()

    if args.peak_fp64 > 0:
        if rank == 0:
            peaks, peak_src = measured_peaks()
            sm_max = float(peaks.get("sm_max_mhz", 1965.0))
            burst = g.gtls_peak_fp64(0.1, device=local_rank)
            time.sleep(1.0)
            sampler = ClockSampler(local_rank)
            sampler.start()
            time.sleep(1.0)
            sampler.mark()
            sus = g.gtls_peak_fp64(args.peak_fp64, device=local_rank)
            clocks = sampler.stop()
            print(json.dumps({"metric": "fp64 FMA rate (register-only DFMA kernel, 16 warps/SM)", "unit": "TFLOP/s",
                              "burst_0.1s": burst["tflops"], "sustained": sus["tflops"], "sustained_seconds": sus["ms"] / 1e3,
                              "derived_peak": SM_COUNT * DFMA_PER_CLK_PER_SM * 2 * sm_max * 1e6 / 1e12,
                              "derived_from": f"{SM_COUNT} SMs x {DFMA_PER_CLK_PER_SM} DFMA/clk x 2 flop x {sm_max:.0f} MHz ({peak_src})",
                              "clocks_during_sustained": clocks}), flush=True)
        return 0

    if args.survey > 0:
        if rank == 0:
            print(json.dumps(run_survey(args, g, torch, devname)), flush=True)
        return 0

    # every rank searches its own curve of the same shape (independent problems)
    w = build_workload(args.workload, curve=rank, every=args.every, dt0=args.dt0)
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(devname)
    d_in = [dev(x) for x in (w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl)]
    ws = torch.empty(g.gtls_workspace_bytes(w.lc.n, w.n_per, w.n_dur, args.period_tile), dtype=torch.uint8,
                     device=devname)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=devname)     # > 126 MB L2

    def step(stats=False):
        return g.gtls_search(*d_in, dt0=w.dt0, sde_kernel=151, workspace=ws, stats=stats,
                             period_tile=args.period_tile)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local_rank)
    sampler.start()
    for _ in range(max(args.warmup, 3)):
        res = step()
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.mark()
    ev0.record()
    for _ in range(args.steps):
        flush.zero_()                                   # L2 flush between timed iterations
        res = step()                                    # no per-stage events, no per-tile host syncs
    ev1.record()
    barrier()
    clocks = sampler.stop()
    ms_total = ev0.elapsed_time(ev1)
    ms_total = max_over_ranks(ms_total, world, devname)
    ms_step = ms_total / args.steps
    value = world * w.trials / (ms_step / 1e3)
    # stage split, window counters and the roofline of the chi2 stage: ONE more step of the same workload
    # with the library's per-stage CUDA events on (one stream synchronisation per period tile), untimed
    flush.zero_()
    st_acc = dict(step(stats=True).stats)

    out = None
    if rank == 0:
        peaks, peak_src = measured_peaks()
        # ---- roofline of the dominant kernel (in-transit chi2, fp64 FMA pipe) -------------------
        chi2_ms_per_launch = st_acc["ms_chi2"] / max(1, st_acc["chi2_launches"])
        flop_per_wp = 2.0 if st_acc["uniform_dy"] else 4.0          # 1 or 2 DFMA per window point
        flops_per_launch = st_acc["window_points"] * flop_per_wp / max(1, st_acc["chi2_launches"])
        achieved = flops_per_launch / (chi2_ms_per_launch * 1e-3) / 1e12
        sm_max = float(peaks.get("sm_max_mhz", 1965.0))
        peak = SM_COUNT * DFMA_PER_CLK_PER_SM * 2 * sm_max * 1e6 / 1e12
        # DRAM traffic of one such launch from the ncu --set full capture of this workload's tile: sum of
        # dram__bytes_read.sum + dram__bytes_write.sum over the eleven ring-kernel launches of one
        # 4144-period tile of c4 (profiles/r1_F_final_c4e64.md: the first tile of the every-64th-period
        # subsample, periods spread over the longer 63 % of the grid; the full run's tiles are 4144
        # consecutive periods of the same kernels).  Other workloads / tile sizes have no capture: null
        traffic, traffic_src = chi2_stage_traffic(args.workload if args.dt0 is None and args.every == 1 else None,
                                                   st_acc["period_tile"])
        roofline = {"bound": "alu", "kernel": "k_chi2_ring (in-transit chi2, a5-a8; one 'launch' = the chi2 stage of one period tile: trial binning + the ring-kernel variants)", "achieved": achieved,
                    "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic,
                    "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum over the stage's kernels)",
                    "traffic_source": traffic_src,
                    "peak_source": f"derived: {SM_COUNT} SMs x {DFMA_PER_CLK_PER_SM} DFMA/clk x 2 flop x "
                                   f"{sm_max:.0f} MHz ({peak_src} sm_max_mhz); measured beside it: `bench.py --peak-fp64` "
                                   f"(register-only DFMA kernel), line kept in profiles/r2_peak_fp64.md",
                    "measured_from": "one untimed step of the same workload with per-stage CUDA events (gtls_stats)",
                    "algorithmic_flops_per_launch": flops_per_launch,
                    "ms_per_launch": chi2_ms_per_launch,
                    "share_of_step": st_acc["ms_chi2"] / max(1e-9, st_acc["ms_total"])}
        stages = {k: st_acc[k] for k in st_acc if k.startswith("ms_")}
        hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
        pp = float(st_acc["period_points"])
        # fold + sort + gather + scan are one fused stage (bucket_sort.cu); algorithmic HBM bytes per
        # period-point: 8 (bucketed key written) + 8 (read back) + 4 (permutation) + 1.15 x 16 (x1, S1 with
        # the wrap pad) = 38.4 B when dy is uniform, + 18.4 B for x0, S0 otherwise
        fss_bytes = 38.4 if st_acc["uniform_dy"] else 56.8
        fss_ms = stages["ms_fold"] + stages["ms_sort"] + stages["ms_scan"]
        stage_roof = {
            "fold_sort_scan_GBps": pp * fss_bytes / (fss_ms * 1e-3) / 1e9 if fss_ms else None,
            "fold_sort_scan_bytes_per_period_point": fss_bytes,
            "fold_sort_scan_frac_of_hbm_peak": (pp * fss_bytes / (fss_ms * 1e-3) / 1e9 / hbm_peak) if fss_ms else None,
            "hbm_peak_GBps": hbm_peak, "peak_source": peak_src,
        }
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_desc(w), "l2_flush": "256 MiB memset between timed steps",
                       "period_tile": st_acc["period_tile"], "path": st_acc["path"],
                       "uniform_dy": st_acc["uniform_dy"],
                       "multi_gpu": "one independent light curve per rank, no collective"},
            "s_per_light_curve": ms_step / 1e3,
            "clocks": clocks,
            "gpu_launches": int(st_acc["kernel_launches"]) * args.steps,
            "stage_ms_per_step": stages, "stage_bandwidth": stage_roof,
            "roofline": roofline,
            "summary": res.summary,
            "paper_context": {"gtls_rtx4090_s": 138.0, "tls_cpu_7950x_s": 3289.0,
                              "note": "PAPER.md:411, 3000-d curve, other hardware: context only"},
        }

    # ---- e2e: host buffers through the C ABI, H2D + D2H inside the timed region ------------------
    if not args.no_e2e:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
        h_in = [pin(x) for x in (w.lc.t, w.lc.y, w.lc.dy, w.periods, w.durations, w.tmpl)]
        del ws
        torch.cuda.empty_cache()
        barrier()
        n_e2e = max(1, min(2, args.steps))
        g.gtls_search(*h_in, dt0=w.dt0, sde_kernel=151)          # warm-up (allocations)
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            r2 = g.gtls_search(*h_in, dt0=w.dt0, sde_kernel=151)
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) / n_e2e
        dt = max_over_ranks(dt, world, devname)
        if rank == 0:
            h2d = int(sum(x.nbytes for x in h_in))
            d2h = int(w.n_per * (8 * 3 + 24))
            out["e2e"] = {"value": world * w.trials / dt, "unit": UNIT, "h2d_bytes_per_step": h2d,
                          "d2h_bytes_per_step": d2h, "ms_per_step": dt * 1e3, "steps": n_e2e,
                          "note": "gtls_search with host pointers: H2D + search + D2H per call; device blocks up to 8 GiB come from the library's pool after the warm-up call, larger ones are cudaMalloc'ed per call"}

    parity_ok = True
    if rank == 0:
        if not args.no_cpu_baseline:
            import oracle
            sample, cores, every = oracle_sample(w, args.ref_seconds)
            t0 = time.perf_counter()
            ro = oracle.search(sample.lc.t, sample.lc.y, sample.lc.dy, sample.periods, sample.durations,
                               sample.tmpl, dt0=w.dt0)
            dt = time.perf_counter() - t0
            out["cpu_baseline"] = {
                "value": sample.trials / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                "sample": f"every {every}th period of {w.name} ({sample.n_per} of {w.n_per} periods), {dt:.1f} s",
                "s_per_light_curve_extrapolated": w.trials / (sample.trials / dt)}
            # parity spot check on the sample while we are here (not timed): chi2 within 1e-9 relative and the
            # best (duration, start) indices identical wherever the oracle's runner-up gap is above 1e-12 chi2
            got = np.asarray(res.chi2.cpu())[::every][:sample.n_per]
            gb = res.best()[::every][:sample.n_per]
            rel = float(np.max(np.abs(got - ro.chi2) / ro.chi2))
            strict = ro.gap > 1e-12 * np.abs(ro.chi2)
            mism = (gb["dur_idx"] != ro.best["dur_idx"]) | (gb["start"] != ro.best["start"])
            t0_ok = bool(np.array_equal(gb["t0"][~mism], ro.best["t0"][~mism]))
            out["cpu_baseline"]["chi2_max_rel_err_vs_gpu"] = rel
            out["cpu_baseline"]["index_mismatches_vs_gpu"] = int(np.sum(mism & strict))
            out["cpu_baseline"]["near_tie_periods"] = int(np.sum(~strict))
            parity_ok = rel <= 1e-9 and not np.any(mism & strict) and t0_ok
            out["cpu_baseline"]["parity_spot_check"] = "ok" if parity_ok else "FAILED"
        print(json.dumps(out), flush=True)
        if not args.no_cpu_baseline and not parity_ok:
            log("bench.py: parity spot check against the oracle FAILED")
            return 1
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
