#!/usr/bin/env python
"""bench.py -- point-periods folded per second on B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path (period grid -> phase ->
bin map -> accumulate -> bin mean -> noise normalisation) over one batch of
synthetic light curves, through the C ABI of libgpfc.so:

    gpfc_make_period_grid(...)                       -> periods (device)
    gpfc_fold_batch(..., out_sum, out_count, out_norm)   (fold + fused normalise)

Default workload: BASELINE.json configs[2], the batched Kepler-shaped fold the
north_star target is quoted on (1,024 curves x 65,000 samples x 20,000 periods,
nbins = 256).  Inputs are resident in HBM for `value`; `e2e` runs the same step
through gpfc_fold_batch_host with pinned HOST buffers (copies inside the timed
region).  One JSON line on stdout (rank 0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]
    python -m torch.distributed.run --nproc-per-node N ... bench.py --gpus N ...

N > 1: the path shards by curve with no exchange step; every rank
folds its own batch of the same shape (weak scaling), no collective on the data
path; timing is max over ranks.
--impl reference: the CPU oracle (oracle/), as it stands, on the host cores, on a
bounded sample of the same workload (rank 0 only).
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

METRIC = "point-periods folded/sec (samples x trial periods)"
UNIT = "point-periods/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2,
                    help="BASELINE.json config index (0-4); 5 = the paper's own two-tier fold "
                         "(70,000 epochs x 100,000 periods, 4096 -> 256 bins, PAPER.md Table 1)")
    ap.add_argument("--impl", default="gpfc", choices=["gpfc", "reference"])
    ap.add_argument("--curves", type=int, default=0, help="debug: override the number of curves")
    ap.add_argument("--periods", type=int, default=0, help="debug: override the number of periods")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-peaks", action="store_true", help="skip gpfc_measure_peaks")
    ap.add_argument("--generated-inputs", action="store_true",
                    help="draw the light curves on the device with gpfc_make_light_curves (PAPER.md 2.6 "
                         "simulator, same shape and cadence as the config) instead of the numpy recipe; "
                         "the graded inputs are the numpy ones")
    ap.add_argument("--nb2", type=int, default=256,
                    help="config 5: final equal-count bins (256 = the paper's; a value the fused kernel "
                         "does not cover, e.g. 300, runs fold + merge_equal_count_kernel: profiling)")
    ap.add_argument("--standalone-normalize", action="store_true",
                    help="profiling: fold writes sums and counts, gpfc_normalize makes the normalised "
                         "profiles in a second kernel (the default step fuses it into the fold)")
    ap.add_argument("--no-others", action="store_true",
                    help="skip the other_configs block of the default run (configs 1, 3, 4, 5)")
    return ap.parse_args()


def make_workload(args, rank):
    from paper_2312_02063_b200 import workloads
    kw = {}
    if args.periods:
        kw["nperiods"] = args.periods
    if args.config in (2, 4):
        full = 1024 if args.config == 2 else 4096
        nc = args.curves or full
        kw["ncurves"] = nc
        kw["first_curve"] = rank * nc        # every rank its own curves (weak scaling)
    return workloads.make(args.config, **kw)


def max_over_ranks(value, world, device=None):
    """Max of a per-rank scalar over all ranks (no-op for world == 1).  The tensor lives on
    `device` (cuda under NCCL, cpu under gloo)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    tt = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def workload_desc(w, args):
    if w.config_id == 5:
        return {"workload": "PAPER.md Table 1 fold: %s" % w.name, "curves": 1,
                "samples_per_curve": int(w.n_total), "nperiods": int(w.nperiods),
                "nbins": "4096 intermediary -> 256 equal-count (gpfc_fold_two_tier)",
                "outputs": "mean+norm [Np][256]",
                "grid": "uniform in period, %.1f..%.1f d" % (w.pmin, w.pmax),
                "l2": "205 MB of outputs per step exceed the 126 MB L2; the 0.84 MB curve is L2-resident "
                      "by design (re-read by every work item)"}
    d = {"workload": "BASELINE.json configs[%d] %s" % (w.config_id, w.name),
         "curves": w.ncurves, "samples_per_curve": int(w.n_total // max(w.ncurves, 1)),
         "nperiods": int(w.nperiods), "nbins": int(w.nbins),
         "outputs": "norm" if w.fused_normalize else "sum+count+norm",
         "grid": "uniform in frequency, 1/%.1f..1/%.1f d^-1" % (w.pmax, w.pmin),
         "l2": "inputs + outputs per step exceed the 126 MB L2; no explicit flush"}
    if args.curves or args.periods:
        d["reduced"] = True
    return d


# --------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "200"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(mx)) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# --------------------------------------------------------------------------- oracle legs
def oracle_sample(w, periods_host, budget_pp):
    """Bounded sample of the workload for the CPU oracle: the first curves and the first
    periods, about `budget_pp` point-periods -> (ncurves, nperiods)."""
    n0 = int(w.offsets[1] - w.offsets[0]) if w.ncurves else 0
    npd = int(min(w.nperiods, max(1, budget_pp // max(n0, 1))))
    nc = int(min(w.ncurves, max(1, budget_pp // max(n0 * npd, 1))))
    return nc, npd


def run_oracle(w, periods_host, ncurves, npd, threads):
    """Oracle fold + normalise of the first `ncurves` curves x first `npd` periods.  Tasks
    (one curve x one slice of the period axis) go to a thread pool; each task is the plain
    single-threaded C routine (ctypes releases the GIL)."""
    from concurrent.futures import ThreadPoolExecutor
    from oracle import ref
    per = np.ascontiguousarray(periods_host[:npd])
    nsl = max(1, min(npd, -(-threads // max(ncurves, 1))))
    edges = np.linspace(0, npd, nsl + 1).astype(np.int64)
    tasks = [(c, int(edges[i]), int(edges[i + 1])) for c in range(ncurves) for i in range(nsl)]

    def work(task):
        c, lo, hi = task
        if hi > lo:
            a, b = int(w.offsets[c]), int(w.offsets[c + 1])
            ref.fold_batch(w.times[a:b], w.flux[a:b], np.array([0, b - a], np.int64), per[lo:hi],
                           w.nbins, want_norm=True, want64=False)

    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(work, tasks))
    dt = time.perf_counter() - t0
    pp = int(w.offsets[ncurves]) * npd
    return pp, dt


def cpu_baseline(w, periods_host):
    from oracle import ref
    ref.build()
    cores = os.cpu_count() or 1
    # calibrate on a small slice, then size the sample for ~15 s
    nc, npd0 = oracle_sample(w, periods_host, 65000 * cores * 2)
    pp0, dt0 = run_oracle(w, periods_host, nc, npd0, cores)
    rate0 = pp0 / max(dt0, 1e-9)
    nc, npd = oracle_sample(w, periods_host, int(rate0 * 15.0))
    pp, dt = run_oracle(w, periods_host, nc, npd, cores)
    return {"value": pp / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "first %d curve(s) x first %d periods (%.3g point-periods, %.1f s), fold + "
                      "normalise, %d threads" % (nc, npd, pp, dt, cores)}


def reference_arm(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import ref
    ref.build()
    w = make_workload(args, 0)
    periods = ref.make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode)
    cores = os.cpu_count() or 1
    nc, npd0 = oracle_sample(w, periods, 65000 * cores)
    pp0, dt0 = run_oracle(w, periods, nc, npd0, cores)
    total = max(args.steps + args.warmup, 1)
    per_step_s = min(20.0, 150.0 / total)
    nc, npd = oracle_sample(w, periods, int(pp0 / max(dt0, 1e-9) * per_step_s))
    for _ in range(args.warmup):
        run_oracle(w, periods, nc, npd, cores)
    pps, dts = 0, 0.0
    for _ in range(args.steps):
        pp, dt = run_oracle(w, periods, nc, npd, cores)
        pps += pp
        dts += dt
    value = pps / max(dts, 1e-12)
    sample = ("each step: first %d curve(s) x first %d periods (%.3g point-periods), fold + "
              "normalise, %d threads" % (nc, npd, float(pp), cores))
    out = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT,
           "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": 1e3 * dts / max(args.steps, 1), "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": workload_desc(w, args),
           "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                            "sample": sample},
           "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0,
                   "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


# --------------------------------------------------------------------------- GPU arm
def csrc_digest():
    """sha256 over the CUDA sources: stamps the ncu captures under profiles/ (no .git on the box)."""
    import glob
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2312_02063_b200", "csrc")
    for f in sorted(glob.glob(os.path.join(d, "*.cu")) + glob.glob(os.path.join(d, "*.cuh"))):
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def fold_kernel_name(w):
    if w.nbins <= 256:
        return "fold_lp_kernel"
    return "fold_pk_kernel<%d>" % {512: 10, 1024: 10, 2048: 11, 4096: 12}[w.nbins]


class DeviceRun:
    """One workload resident in HBM: buffers, the step, its timing (CUDA events, max over ranks)."""

    def __init__(self, gp, torch, w, generated=False, seed=0, nb2=256, standalone_normalize=False):
        self.gp, self.torch, self.w = gp, torch, w
        self.nb2, self.standalone_normalize = nb2, standalone_normalize
        dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        self.generator = None
        if generated:
            # rectangular batch of the config's shape: n samples at its median cadence
            n = w.n_total // max(w.ncurves, 1)
            cad = float(np.median(np.diff(w.times[:n])))
            prm = gp.gpfc_lc_params_default(cadence=cad, flags=gp.LC_CENTERED)
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
            gp.gpfc_make_light_curves(seed, w.ncurves, n, prm)          # warm-up
            ev[0].record()
            t_, f_, o_, _ = gp.gpfc_make_light_curves(seed, w.ncurves, n, prm)
            ev[1].record()
            torch.cuda.synchronize()
            ms = ev[0].elapsed_time(ev[1])
            self.times, self.flux, self.offsets = t_.reshape(-1), f_.reshape(-1), o_
            ns = float(w.ncurves) * n
            self.generator = {"api": "gpfc_make_light_curves", "samples": ns, "ms": ms,
                              "samples_per_s": ns / (ms * 1e-3), "bytes_written": ns * 12.0,
                              "hbm_gbs": ns * 12.0 / (ms * 1e-3) / 1e9, "cadence_d": cad, "seed": seed}
        else:
            self.times, self.flux, self.offsets = dev(w.times), dev(w.flux), dev(w.offsets)
        self.two_tier = (w.config_id == 5)
        self.shape = (w.ncurves, w.nperiods, self.nb2 if self.two_tier else w.nbins)
        self.periods = torch.empty(w.nperiods, dtype=torch.float64, device="cuda")
        f32 = lambda: torch.empty(self.shape, dtype=torch.float32, device="cuda")
        self.out_sum = self.out_count = self.out_norm = self.out_mean = None
        if self.two_tier:
            self.out_mean, self.out_norm = f32(), f32()
        else:
            self.out_norm = f32()
            if not w.fused_normalize:
                self.out_sum = f32()
                self.out_count = torch.empty(self.shape, dtype=torch.int32, device="cuda")
        self.ws = torch.empty(gp.gpfc_workspace_bytes(w.ncurves, w.n_total, w.nperiods, w.nbins),
                              dtype=torch.uint8, device="cuda")
        self.noutputs = 2 if self.two_tier else (1 if w.fused_normalize else 3)
        self.out_bytes = float(np.prod(self.shape)) * 4 * self.noutputs

    def step(self):
        gp, w = self.gp, self.w
        gp.gpfc_make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode, out=self.periods)
        if self.two_tier:
            gp.gpfc_fold_two_tier(self.times, self.flux, self.offsets, self.periods, w.nbins, self.nb2,
                                  out_mean=self.out_mean, out_norm=self.out_norm)
        elif self.standalone_normalize and self.out_sum is not None:
            gp.gpfc_fold_batch(self.times, self.flux, self.offsets, self.periods, w.nbins,
                               out_sum=self.out_sum, out_count=self.out_count, want=("sum", "count"))
            gp.gpfc_normalize(self.out_sum, self.out_count, out_norm=self.out_norm)
        else:
            gp.gpfc_fold_batch(self.times, self.flux, self.offsets, self.periods, w.nbins,
                               out_sum=self.out_sum, out_count=self.out_count, out_norm=self.out_norm)

    def timed(self, steps, warmup, barrier, world, sampler=None):
        gp, torch = self.gp, self.torch
        gp.gpfc_set_workspace(self.ws)
        for _ in range(warmup):
            self.step()
        barrier()
        if sampler:
            sampler.start()
        gp.gpfc_profile(True)
        e0 = torch.cuda.Event(enable_timing=True)
        e1 = torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            self.step()
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        prof = gp.gpfc_profile_read()
        paths = gp.gpfc_path_counters()
        gp.gpfc_profile(False)
        clocks = sampler.stop() if sampler else None
        gp.gpfc_set_workspace(None)
        ms = max_over_ranks(ms, world, "cuda")
        return ms, prof, paths, clocks

    def free(self):
        for k in ("times", "flux", "offsets", "periods", "out_sum", "out_count", "out_norm",
                  "out_mean", "ws"):
            setattr(self, k, None)
        self.torch.cuda.empty_cache()


def roofline_of(w, run, prof, sm_max, peaks, traffic_db, digest):
    """the fold kernel against the shared-memory atomic bound (2 lane-updates per
    point-period) and, beside it, the HBM bound on its algorithmic bytes."""
    fold_ms = prof["fold_kernel_ms"] / max(prof["fold_launches"], 1)
    updates = 2.0 * float(w.point_periods)
    peak_nominal = 148 * 32 * sm_max * 1e6              # 32 shared-memory atomic lanes / clk / SM
    achieved = updates / (fold_ms * 1e-3)
    alg_bytes = run.out_bytes + w.n_total * 12.0
    roof = {"bound": "alu", "achieved": achieved / 1e9, "peak": peak_nominal / 1e9,
            "unit": "G shared-atomic lane-updates/s", "frac": achieved / peak_nominal,
            "traffic": None, "kernel": fold_kernel_name(w), "kernel_ms": fold_ms,
            "peak_source": "derived: 148 SMs x 32 lanes/clk x %.0f MHz" % sm_max,
            "algorithmic_bytes": alg_bytes,
            "hbm_bound": {"algorithmic_bytes": alg_bytes,
                          "achieved_gbs": alg_bytes / (fold_ms * 1e-3) / 1e9}}
    try:
        mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        roof["hbm_bound"]["peak_gbs"] = mp["hbm_gbs"]
        roof["hbm_bound"]["peak_source"] = "MEASURED_PEAKS.json"
    except (OSError, KeyError, ValueError):
        roof["hbm_bound"]["peak_gbs"] = 6650.0
        roof["hbm_bound"]["peak_source"] = "fallback (B200_PROFILING.md)"
    roof["hbm_bound"]["frac"] = roof["hbm_bound"]["achieved_gbs"] / roof["hbm_bound"]["peak_gbs"]
    tj = (traffic_db or {}).get(w.name)
    if tj and (tj["curves"], tj["nperiods"], tj["nbins"]) == (w.ncurves, w.nperiods, w.nbins):
        # DRAM bytes per launch from the committed ncu --set full capture of this workload
        roof["traffic"] = tj["traffic_bytes"]
        roof["traffic_source"] = "profiles/r2_traffic.json (ncu --set full of this command, sources %s)" \
                                 % tj.get("csrc_digest", "?")
        roof["traffic_stale"] = tj.get("csrc_digest") != digest
    if peaks:
        roof["measured_peak"] = peaks["smem_atomic_lane_updates_per_s"] / 1e9
        roof["frac_of_measured"] = achieved / peaks["smem_atomic_lane_updates_per_s"]
    return roof


def host_e2e(gp, torch, w, run_shape, steps, barrier, world, two_tier, norm_only=False):
    """The same step through the host-buffer entry points: pinned host memory in and out,
    copies inside the timed region.  norm_only: only the normalised profiles (the scorer's
    input) come back, a third of the bytes."""
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    h_t, h_f, h_o = pin(w.times), pin(w.flux), pin(w.offsets)
    h_sum = h_cnt = h_norm = None
    if two_tier:
        h_mean = torch.empty(run_shape, dtype=torch.float32, pin_memory=True)
        h_norm = torch.empty(run_shape, dtype=torch.float32, pin_memory=True)
    else:
        h_norm = torch.empty(run_shape, dtype=torch.float32, pin_memory=True)
        if not w.fused_normalize and not norm_only:
            h_sum = torch.empty(run_shape, dtype=torch.float32, pin_memory=True)
            h_cnt = torch.empty(run_shape, dtype=torch.int32, pin_memory=True)

    def step_host():
        if two_tier:
            # no host entry point for the two-tier path: the user's calls are the device API
            # with torch copies (pinned host -> device, merged profiles -> pinned host)
            dt_, df_, do_ = (h_t.cuda(non_blocking=True), h_f.cuda(non_blocking=True),
                             h_o.cuda(non_blocking=True))
            per = gp.gpfc_make_period_grid(w.pmin, w.pmax, w.nperiods, w.grid_mode)
            m_, n_ = gp.gpfc_fold_two_tier(dt_, df_, do_, per, w.nbins, 256)
            h_mean.copy_(m_, non_blocking=True)
            h_norm.copy_(n_, non_blocking=True)
            torch.cuda.synchronize()
            return
        per = gp.gpfc_make_period_grid_host(w.pmin, w.pmax, w.nperiods, w.grid_mode)
        gp.gpfc_fold_batch_host(h_t, h_f, h_o, per, w.nbins, out_sum=h_sum, out_count=h_cnt,
                                out_norm=h_norm)

    step_host()
    barrier()
    t0 = time.perf_counter()
    for _ in range(steps):
        step_host()
    barrier()
    dt = max_over_ranks(time.perf_counter() - t0, world, "cuda")
    nout = int(np.prod(run_shape)) * 4
    e2e = {"value": float(w.point_periods) * world * steps / dt, "unit": UNIT,
           "h2d_bytes_per_step": int(w.n_total * 12 + w.offsets.nbytes),
           "d2h_bytes_per_step": int(nout * (1 if (w.fused_normalize or norm_only) else 3) + w.nperiods * 8),
           "steps": steps, "api": "gpfc_make_period_grid_host + gpfc_fold_batch_host"
                                  + (" (out_norm only)" if norm_only else "")}
    e2e["s_per_step"] = dt / steps
    e2e["d2h_gbs"] = e2e["d2h_bytes_per_step"] / (dt / steps) / 1e9
    if two_tier:
        e2e["d2h_bytes_per_step"] = int(2 * nout)
        e2e["api"] = "torch H2D + gpfc_make_period_grid + gpfc_fold_two_tier + torch D2H"
    return e2e


def gpu_arm(args):
    import torch
    import torch.distributed as dist
    from paper_2312_02063_b200 import binding as gp

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    gp.lib()
    gp.gpfc_init()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    digest = csrc_digest()
    try:
        traffic_db = json.load(open(os.path.join(ROOT, "profiles", "r2_traffic.json")))
    except (OSError, ValueError):
        traffic_db = {}
    peaks = None
    if rank == 0 and not args.no_peaks:
        peaks = gp.gpfc_measure_peaks()

    # ---- the headline workload
    w = make_workload(args, rank)
    run = DeviceRun(gp, torch, w, generated=args.generated_inputs, seed=1000 + rank, nb2=args.nb2,
                    standalone_normalize=args.standalone_normalize)
    generator = run.generator
    ms, prof, paths, clocks = run.timed(args.steps, args.warmup, barrier, world,
                                        ClockSampler(local) if rank == 0 else None)
    pp_step_all = float(w.point_periods) * world
    value = pp_step_all * args.steps / (ms * 1e-3)
    periods_host = run.periods.cpu().numpy()
    shape, two_tier = run.shape, run.two_tier
    sm_max = (clocks or {}).get("sm_max_mhz") or 1965.0
    roof = roofline_of(w, run, prof, sm_max, peaks, traffic_db, digest) if rank == 0 else None
    run.free()

    e2e = None
    if not args.no_e2e:
        e2e = host_e2e(gp, torch, w, shape, max(1, min(args.steps, 3)), barrier, world, two_tier)
        torch.cuda.empty_cache()
        if not two_tier and not w.fused_normalize:
            # the streaming path a scorer would use: only the normalised profiles come back, and
            # the copy of chunk k overlaps the fold of chunk k+1 (gpfc_fold_stream)
            e2n = host_e2e(gp, torch, w, shape, max(1, min(args.steps, 3)), barrier, world, two_tier,
                           norm_only=True)
            fold_s = ms / args.steps * 1e-3
            e2n["device_fold_s_per_step"] = fold_s
            # time hidden by the overlap: fold + copy back to back would take fold_s + bytes / rate
            e2n["copy_s_at_this_rate"] = e2n["d2h_bytes_per_step"] / (e2e["d2h_gbs"] * 1e9)
            e2n["hidden_s_per_step"] = max(0.0, fold_s + e2n["copy_s_at_this_rate"] - e2n["s_per_step"])
            e2e["norm_only"] = e2n
            torch.cuda.empty_cache()

    # ---- the other BASELINE.json configs (and the paper's own fold), each after its own
    # warm-up, so that one driver run carries a number for every row of DESIGN.md 7
    others = []
    if args.config == 2 and not (args.curves or args.periods or args.no_others) and world == 1:
        for cid in (1, 3, 4, 5):
            from paper_2312_02063_b200 import workloads
            wo = workloads.make(cid)
            ro = DeviceRun(gp, torch, wo)
            st = 3
            ms_o, prof_o, paths_o, _ = ro.timed(st, 3, barrier, 1)
            rf = roofline_of(wo, ro, prof_o, sm_max, peaks, traffic_db, digest)
            ent = {"config": workload_desc(wo, args), "value": float(wo.point_periods) * st / (ms_o * 1e-3),
                   "unit": UNIT, "steps": st, "warmup": 3, "ms_per_step": ms_o / st,
                   "kernel": rf["kernel"], "kernel_ms": rf["kernel_ms"], "roofline_frac": rf["frac"],
                   "hbm_frac": rf["hbm_bound"]["frac"], "traffic": rf["traffic"],
                   "traffic_stale": rf.get("traffic_stale"), "slow_paths": paths_o,
                   "gpu_launches": int(prof_o["kernel_launches"])}
            if cid == 5:
                ent["paper"] = {"workload_s_paper_gpu": 4.32, "workload_s_here_device": ms_o / st * 1e-3,
                                "cite": "PAPER.md:125-142 Table 1 (RTX 3090 Ti): 0.66 s kernels + 3.66 s "
                                        "device memory for 70,000 epochs x 100,000 periods"}
            others.append(ent)
            ro.free()
            del wo, ro

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    if peaks:
        roof["fp64_pairs_per_s"] = peaks["fp64_mul_add_pairs_per_s"]
        roof["inner_loop_ceiling_pp_per_s"] = peaks["fold_loop_pp_per_s"]   # fold_lp loop alone
        roof["alternatives_lane_updates_per_s"] = {
            "cas_float_atomicAdd": peaks["smem_cas_float_lane_updates_per_s"],
            "lds_add_sts_private_rows": peaks["smem_lds_sts_lane_updates_per_s"]}

    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
           "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": workload_desc(w, args), "clocks": clocks, "roofline": roof,
           "gpu_launches": int(prof["kernel_launches"]), "slow_paths": paths,
           "csrc_digest": digest}
    if two_tier:
        # the paper's profiled fold, same workload, RTX 3090 Ti (context, not target)
        out["vs_baseline"] = value / (70000.0 * 100000.0 / 4.32)
        out["paper"] = {"workload_s_paper_total": 5.00, "workload_s_paper_gpu_kernels_plus_device_memory": 4.32,
                        "workload_s_here_device": ms / args.steps * 1e-3,
                        "vs_baseline_denominator": "7e9 point-periods / 4.32 s (Table 1: 0.66 s kernels "
                        "+ 3.66 s device memory), PAPER.md:130-131", "hardware_paper": "RTX 3090 Ti"}
    if e2e:
        out["e2e"] = e2e
        if two_tier:
            out["paper"]["workload_s_here_e2e"] = 70000.0 * 100000.0 / e2e["value"]
    if generator:
        out["generator"] = generator
        out["data"] = "synthetic, generated on the device (gpfc_make_light_curves)"
    if others:
        out["other_configs"] = others
    if not args.no_cpu:
        out["cpu_baseline"] = cpu_baseline(w, periods_host)
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        reference_arm(args)
    else:
        gpu_arm(args)


if __name__ == "__main__":
    main()
