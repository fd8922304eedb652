#!/usr/bin/env python
"""bench.py -- the driver's benchmark contract for libtkm.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

Metric (BASELINE.json): (lambda x fold) path fits per second.

Default line = BASELINE.json configs[1] (smoothed-hinge kernel SVM, n=2000, p=50, 5 folds, 50 lambdas x 5 sigma
values), the configuration the metric is quoted on.  One STEP is one pass of the whole hot path over that
workload: for each of the 5 bandwidths  S1 Gram -> S2 spectral setup -> S9 exact CV, with the S3-S8 sweeps of
the 5 bandwidths (50 x (5+1) columns each) run together as groups of one launch sequence (tkm_fit_path_multi),
and S10 coefficients in the e2e leg.  `value` = columns fitted per second by the WHOLE step (setup included), X
and y resident in HBM before the timed region; `fits_per_s_sweep_only` = SURVEY.md 8(d)'s B / t_sweep; `e2e` =
the same through tkm_train_tune_host from pinned HOST buffers.  The same JSON line carries `large_config`: one
pass of BASELINE.json configs[3] (the largest full-kernel single-GPU configuration, n = 20000, 900 columns) with
its own stage times, roofline and clocks (outside the timed region of `value`; `--no-large` skips it), and
`single_tf32_increments` (tf32_delta = 3: one step of the same workload with single-TF32 increment products).

Other workloads (`--workload`, one GPU, one JSON line each with the same keys):
  config2 | config3 | config4      BASELINE.json configs[2..4] at full size
  nystrom_covtype | nystrom_mnist8m46   Nystrom at the row counts of the paper's Table 4
  loo_config1                      leave-one-out form of Algorithm 1 (V = n) on configs[1]'s data (8(f) N2)
  narrow_config2 | narrow_config3  configs[2]/[3] with `--narrow-L` in {1,2,4} lambdas: the HBM-bound narrow batch
  gemm_probe                       the two contraction kernels alone on a list of shapes (calibration / evidence)

N > 1 (torchrun): the path has no exchange step -- every rank runs the same-size workload on its own seeded
data set (independent problems, "weak" scaling); the only communication is the barrier and the max-over-ranks
of the device time.

`--impl reference` times the FP64 CPU oracle (oracle/, test infrastructure) on a bounded sample of the default
workload on the host cores; rank 0 only.
"""
from __future__ import annotations

import argparse
import csv
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

import workloads as wl  # noqa: E402

METRIC = "lambda_x_fold_path_fits_per_s"
UNIT = "fits/s"
STOP_TOL = {"f64": 1e-12}                   # DESIGN.md "Tolerances" (the default line); --tol for the other workloads
MAXIT = 200000
# Stop tolerance of the smoothing rounds 0..R-2, which only produce warm starts for the last round (the
# result is the minimiser at the final smoothing level, whatever the start): DESIGN.md "Schedule".  The oracle
# arm uses the same value (oracle.fit_path(warm_tol=...)).
WARM_TOL = 1e-3
# Delta form of the contractions (tkm_loss_opts.tf32_delta): the FP64 state advances by 3xTF32
# increments on the tcgen05 tensor cores, with exact FP64 DMMA contractions and the stop test on the last iteration
# of every 16-iteration batch and in the narrow tail.  Same fixed point and the same 1e-10 parity bar as the
# all-FP64 sweep.  This is how the "fp32" configurations of BASELINE.json run: FP64 state + 3xTF32 increments.
TF32_DELTA = 2           # default line (configs[1])
TF32_DELTA_LARGE = 2     # configs[2..4], Nystrom, leave-one-out
# nominal dense tensor ratios to bf16 (B200_PROFILING.md / B300_MICROARCH.md tables): FP64 45 TF,
# TF32 1125 TF, bf16 2250 TF.  3xTF32 does three MMAs per useful one.
NOMINAL_RATIO = {"f64": 45.0 / 2250.0, "f32": (1125.0 / 2250.0) / 3.0}
DMMA_FLOP_PER_CLK_SM = 128.0     # DMMA.8x8x4: 4 per 16 clocks per SM = 128 flop/clk/SM
N_SM = 148
# dram bytes per launch of the kernels, from committed `ncu --set full` captures: profiles/traffic.csv
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "traffic.csv")
# columns of the bounded CPU sample: all V+1 hold-out settings x these lambda indices, one sigma
CPU_SAMPLE_LAMBDA_IDX = (0, 12, 24, 36, 49)
CPU_SAMPLE_SIGMA_IDX = 2
FAMILY = ["gemm_f64_tma_kernel GEMM-A (FP64 DMMA, loss epilogue)", "gemm_f64_tma_kernel GEMM-B (FP64 DMMA, spectral epilogue)",
          "gemm_tf32x3_kernel GEMM-A (tcgen05 3xTF32 delta form, loss epilogue)",
          "gemm_tf32x3_kernel GEMM-B (tcgen05 3xTF32 delta form, spectral epilogue)"]


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm=d["hbm_gbs"], bf16_burst=d["bf16_tflops"], bf16_sus=d["bf16_tflops_sustained"],
                    src="measured")
    return dict(hbm=6650.0, bf16_burst=1590.0, bf16_sus=1400.0, src="fallback")


def traffic_table():
    """kernel key -> (dram bytes per launch, source) from profiles/traffic.csv (written from ncu captures)."""
    out = {}
    if os.path.exists(TRAFFIC_CSV):
        with open(TRAFFIC_CSV) as f:
            for row in csv.DictReader(ln for ln in f if not ln.startswith("#")):
                out[row["key"]] = (float(row["dram_bytes_per_launch"]), row["source"])
    return out


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    PERIOD_MS = 200    # --clock-period-ms; 0 = no sampler (experiments only: the line then has no clocks evidence)

    def __init__(self, index):
        self.index, self.proc, self.lines, self.t0 = index, None, [], 0.0

    def mark(self):
        """Start of the timed region: only lines that arrive from now on are used.  The sampler itself is started
        BEFORE the warm-up steps: nvidia-smi's own start-up (NVML initialisation, about a second on a fresh box) holds
        driver locks that stretch host-paced stages (cuSOLVER's Dsyevd: 135 -> 445 ms per step in the first run on a
        box when it was started at the edge of the timed region)."""
        self.t0 = time.monotonic()

    def start(self):
        if self.PERIOD_MS <= 0:
            return
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", str(int(self.PERIOD_MS))],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def wait_ready(self, timeout=8.0):
        """Block until nvidia-smi has printed its first line (its start-up is over) or `timeout` seconds passed."""
        t_end = time.monotonic() + timeout
        while self.proc and not self.lines and time.monotonic() < t_end and self.proc.poll() is None:
            time.sleep(0.05)

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append((time.monotonic(), ln.strip()))

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for (t_arr, ln) in self.lines:
            if t_arr < self.t0:
                continue
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                pw.append(float(f[2]))
            except ValueError:
                continue
            for nme, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ----------------------------------------------------------------------------------------- oracle arm
def oracle_sample_step(w):
    """One bounded sample of the workload on the CPU oracle: one sigma, 5 lambdas x (V+1) columns,
    Gram + eigh + path + exact CV, same stop and warm-start tolerances as the GPU arm.
    Returns (#columns fitted, seconds, column-iterations)."""
    import oracle as o
    t0 = time.perf_counter()
    sigma = float(w.sigmas[CPU_SAMPLE_SIGMA_IDX])
    foldid = o.make_folds(w.n, w.V, w.fold_seed)
    K = o.gram_rbf(w.X, sigma)
    spec = o.spectral_setup(K)
    L, V = w.L, w.V
    cols = [v * L + l for v in range(V + 1) for l in CPU_SAMPLE_LAMBDA_IDX if l < L]
    res = o.fit_path(spec, w.y, w.loss, w.lambdas, foldid, V, taus=w.taus, smooth0=w.smooth0, eta=w.eta,
                     rounds=w.rounds, tol=STOP_TOL["f64"], maxit=MAXIT, columns=cols, warm_tol=WARM_TOL)
    o.exact_cv(spec, res, w.y, foldid, w.loss, w.taus)
    return len(cols), time.perf_counter() - t0, int(res.iters.sum())


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
    except Exception:
        return os.cpu_count() or 1


def sample_text(w, ncol, secs=None, its=None):
    s = ("sigma index %d, lambda indices %s x %d hold-out settings = %d of %d columns per step, full n; Gram + eigh + "
         "path + exact CV; same stop / warm-start tolerances as the GPU arm; the 5 sampled lambdas span the grid "
         "evenly, so the sample averages more iterations per column than the full grid (about 1.5x: a skew against "
         "the oracle)" % (CPU_SAMPLE_SIGMA_IDX, list(CPU_SAMPLE_LAMBDA_IDX), w.V + 1, ncol, w.B * len(w.sigmas)))
    if secs is not None:
        s += "; %.1f s, %d column-iterations" % (secs, its)
    return s


def run_reference(args, w, rank):
    if rank != 0:
        return
    for _ in range(args.warmup):
        oracle_sample_step(w)
    t0 = time.perf_counter()
    fits = 0
    for _ in range(args.steps):
        c, _, _ = oracle_sample_step(w)
        fits += c
    dt = time.perf_counter() - t0
    val = fits / dt
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(w),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
                             "sample": sample_text(w, fits // max(args.steps, 1))},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_config(w):
    """The workload as both arms run it (the GPU-only launch knobs are in `launch_config`)."""
    return {"workload": "BASELINE.json configs[1]: smoothed-hinge kernel SVM, n=%d, p=%d, %d folds, %d lambdas "
                        "1e2..1e-5 x %d sigma (median x {0.25,0.5,1,2,4}), delta 1 -> 1/512 in %d rounds, f64"
                        % (w.n, w.p, w.V, w.L, len(w.sigmas), w.rounds),
            "n": w.n, "p": w.p, "folds": w.V, "lambdas": w.L, "sigmas": len(w.sigmas),
            "columns_per_step": w.B * len(w.sigmas), "stop_tol": STOP_TOL["f64"], "warm_start_rounds_tol": WARM_TOL,
            "maxit": MAXIT, "value_is": "columns / whole step (Gram + eigendecompositions + sweep + exact CV); "
                                        "fits_per_s_sweep_only = columns / sweep (SURVEY.md 8(d))",
            "l2": "flushed between steps (256 MiB memset)", "parallelism": "independent replicas, no collective"}


# ----------------------------------------------------------------------------------------- roofline helpers
def tensor_peaks(pk, sm_mhz):
    """Peaks a contraction is reported against.  `contract` = measured bf16 sustained x nominal ratio (the
    contract's rule: another dtype's measured peak x the guide's ratio); `issue` = DMMA issue ceiling at the sampled
    SM clock."""
    mhz = sm_mhz if sm_mhz else 1965.0
    return {"f64_contract": pk["bf16_sus"] * NOMINAL_RATIO["f64"],
            "f64_issue": DMMA_FLOP_PER_CLK_SM * N_SM * mhz * 1e6 / 1e12,
            "tf32x3_contract": pk["bf16_sus"] * NOMINAL_RATIO["f32"],
            "src": "%s bf16 sustained %.1f TF/s" % (pk["src"], pk["bf16_sus"])}


def library_probes(tkm):
    """Measured dense peaks on this box, this process: cuBLAS DGEMM and cuBLAS TF32 (torch.matmul, 8192^3, best
    of 5), and the library's own DMMA kernel through tkm_gemm_probe at the same shape."""
    import torch
    out = {}
    N = 8192

    def best_ms(fn, reps=5):
        fn()
        torch.cuda.synchronize()
        best = 1e30
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            e1.synchronize()
            best = min(best, e0.elapsed_time(e1))
        return best

    a = torch.randn(N, N, device="cuda", dtype=torch.float64)
    b = torch.randn(N, N, device="cuda", dtype=torch.float64)
    c = torch.empty_like(a)
    out["cublas_dgemm_tflops"] = 2.0 * N ** 3 / (best_ms(lambda: torch.matmul(a, b, out=c)) * 1e-3) / 1e12
    del a, b, c
    old = torch.backends.cuda.matmul.allow_tf32
    torch.backends.cuda.matmul.allow_tf32 = True
    a = torch.randn(N, N, device="cuda", dtype=torch.float32)
    b = torch.randn(N, N, device="cuda", dtype=torch.float32)
    c = torch.empty_like(a)
    out["cublas_tf32_tflops"] = 2.0 * N ** 3 / (best_ms(lambda: torch.matmul(a, b, out=c)) * 1e-3) / 1e12
    torch.backends.cuda.matmul.allow_tf32 = old
    del a, b, c
    torch.cuda.empty_cache()
    out["tkm_dmma_probe_tflops"] = 2.0 * N ** 3 / (tkm.tkm_gemm_probe(-1, 1, N, N, N, iters=3) * 1e-3) / 1e12
    out["shape"] = "8192^3, best of 5 (cuBLAS through torch.matmul: probes only, never on the product path)"
    return out


L2_BYTES = 126e6     # B200 L2 (B200_PROFILING.md): a U operand set larger than this streams from HBM every launch


def family_rooflines(prof, tp, traffic, probes=None, geom=None, hbm_peak=None, tkeys=None, single_tf32=False):
    """One roofline object per kernel family with sampled launches.  prof: dict(ms, flops, launches) arrays of 4.
    geom = (n, r, G): with it every object also carries the HBM side of the same launches (`hbm`: algorithmic bytes
    = G n r 8 for the U operand of the G groups + live (n + r) 8 for the moving operand and the result, over the
    measured copy bandwidth) and `binding` = the side the roofline model says binds at the launches' arithmetic
    intensity (flops per algorithmic byte against the ridge point peak flops / peak bandwidth; "tensor" whenever
    the U operands of one launch fit in L2)."""
    out = []
    for i in range(4):
        nl = int(prof["launches"][i])
        if nl == 0:
            continue
        ms, fl = float(prof["ms"][i]), float(prof["flops"][i])
        ach = (fl / 1e12) / (ms / 1e3) if ms > 0 else 0.0
        f64 = i < 2
        # tf32_delta = 3: one TF32 MMA per useful product and 4-byte operands (hi parts only)
        peak = tp["f64_contract"] if f64 else tp["tf32x3_contract"] * (3.0 if single_tf32 else 1.0)
        tr = traffic.get((tkeys or {}).get(i, "fam%d" % i))
        d = {"bound": "tensor", "kernel": FAMILY[i].replace("3xTF32", "1xTF32") if single_tf32 else FAMILY[i],
             "achieved": ach, "peak": peak, "unit": "TFLOP/s",
             "frac": ach / peak, "traffic": tr[0] if tr else None, "traffic_source": tr[1] if tr else None,
             "peak_source": tp["src"] + (" x nominal f64/bf16 ratio %.4f" % NOMINAL_RATIO["f64"] if f64 else
                                         (" x nominal tf32/bf16 ratio 0.5 (one MMA per useful product)" if single_tf32 else
                                          " x nominal tf32/bf16 ratio 0.5 / 3 MMAs per useful product")),
             "sampled_launches": nl, "avg_launch_ms": ms / nl, "avg_flops_per_launch": fl / nl, "sampled_ms": ms,
             "family": i}
        if f64:
            d["peak_dmma_issue"] = tp["f64_issue"]
            d["frac_of_issue"] = ach / tp["f64_issue"]
        if geom and hbm_peak and fl > 0:
            n, r, G = geom
            live = fl / nl / (2.0 * n * r)
            u_bytes = G * n * r * (4.0 if (single_tf32 and not f64) else 8.0)
            by = u_bytes + live * (n + r) * 8.0
            gbs = by / (ms / nl / 1e3) / 1e9
            ai, ridge = fl / nl / by, peak * 1e12 / (hbm_peak * 1e9)
            d["hbm"] = {"achieved": gbs, "peak": hbm_peak, "unit": "GB/s", "frac": gbs / hbm_peak,
                        "algorithmic_bytes_per_launch": by, "avg_live_columns": live,
                        "flops_per_byte": ai, "ridge_flops_per_byte": ridge}
            d["binding"] = "hbm" if (ai < ridge and u_bytes > L2_BYTES) else "tensor"
        if probes:
            pm = probes["cublas_dgemm_tflops"] if f64 else probes["cublas_tf32_tflops"] / (1.0 if single_tf32 else 3.0)
            d["peak_measured"] = pm
            d["frac_of_measured"] = ach / pm
            d["peak_measured_source"] = ("cuBLAS DGEMM 8192^3 on this box" if f64 else
                                         "cuBLAS TF32 GEMM 8192^3 on this box / 3 MMAs per useful product")
        out.append(d)
    return out


def merge_families(fams, idx):
    """Sum families (e.g. DMMA GEMM-A + GEMM-B = the FP64 kernel) into one roofline object."""
    sel = [f for f in fams if f["family"] in idx]
    if not sel:
        return None
    ms = sum(f["sampled_ms"] for f in sel)
    fl = sum(f["avg_flops_per_launch"] * f["sampled_launches"] for f in sel)
    nl = sum(f["sampled_launches"] for f in sel)
    d = dict(max(sel, key=lambda f: f["sampled_ms"]))
    ach = fl / 1e12 / (ms / 1e3)
    d.update(kernel=" + ".join(f["kernel"] for f in sel), achieved=ach, frac=ach / d["peak"], sampled_launches=nl,
             avg_launch_ms=ms / nl, avg_flops_per_launch=fl / nl, sampled_ms=ms)
    if "peak_dmma_issue" in d:
        d["frac_of_issue"] = ach / d["peak_dmma_issue"]
    if "peak_measured" in d:
        d["frac_of_measured"] = ach / d["peak_measured"]
    if all("hbm" in f for f in sel):
        by = sum(f["hbm"]["algorithmic_bytes_per_launch"] * f["sampled_launches"] for f in sel)
        h = dict(d["hbm"])
        gbs = by / (ms / 1e3) / 1e9
        h.update(achieved=gbs, frac=gbs / h["peak"], algorithmic_bytes_per_launch=by / nl, flops_per_byte=fl / by,
                 avg_live_columns=sum(f["hbm"]["avg_live_columns"] * f["sampled_launches"] for f in sel) / nl)
        d["hbm"] = h
        d["binding"] = max(sel, key=lambda f: f["sampled_ms"])["binding"]
    return d


def binding_side(d):
    """The roofline object the bench line carries: `bound` is the side that binds the sampled launches (see
    family_rooflines); the other side's figures stay in the object under `tensor_side` / `hbm_side`."""
    if d is None or d.get("binding") != "hbm":
        if d is not None and "hbm" in d:
            d = dict(d)
            d["hbm_side"] = d.pop("hbm")
        return d
    h = d["hbm"]
    t = {k: d[k] for k in ("achieved", "peak", "unit", "frac", "peak_source", "frac_of_issue", "peak_dmma_issue",
                           "peak_measured", "frac_of_measured", "peak_measured_source") if k in d}
    o = {k: v for k, v in d.items() if k not in t and k != "hbm"}
    o.update(bound="hbm", achieved=h["achieved"], peak=h["peak"], unit="GB/s", frac=h["frac"],
             peak_source="MEASURED_PEAKS.json copy bandwidth",
             algorithmic_bytes_per_launch=h["algorithmic_bytes_per_launch"],
             avg_live_columns=h["avg_live_columns"], flops_per_byte=h["flops_per_byte"],
             ridge_flops_per_byte=h["ridge_flops_per_byte"], tensor_side=t)
    return o


def time_weighted(prof2, tp, single_tf32=False):
    """All launches of one sweep (profile = 2): useful flops the device counted / total kernel time, per family."""
    out = {}
    for name, idx, peak, issue in (("fp64_dmma", (0, 1), tp["f64_contract"], tp["f64_issue"]),
                                   ("tcgen05_1xtf32" if single_tf32 else "tcgen05_3xtf32", (2, 3),
                                    tp["tf32x3_contract"] * (3.0 if single_tf32 else 1.0), None)):
        ms = float(sum(prof2["ms"][i] for i in idx))
        fl = float(sum(prof2["flops"][i] for i in idx))
        nl = int(sum(prof2["launches"][i] for i in idx))
        if nl == 0:
            continue
        ach = fl / 1e12 / (ms / 1e3)
        out[name] = {"achieved": ach, "frac": ach / peak, "launches": nl, "kernel_ms": ms,
                     "useful_flops": fl}
        if issue:
            out[name]["frac_of_issue"] = ach / issue
    out["note"] = ("every contraction launch of one extra step timed with CUDA events (outside the timed region); flops "
                   "= 2 n r per column-iteration still unconverged at the launch, counted on the device")
    return out


# ----------------------------------------------------------------------------------------- single-problem runner
def run_problem(tkm, w, *, tf32_delta, tol, warm_tol, profile=1, nystrom_streamed=False, loo=False, lam_idx=None,
                clocks_index=0, gap_tol=0.0, delta_min_live=0):
    """One pass of S1..S9 over ONE (X, sigma) problem on the current device; X, y resident.  Returns a dict of stage
    times (ms), column-iterations, sampled kernel families and clocks."""
    import torch
    sigma = float(w.sigmas[0])
    lambdas = w.lambdas if lam_idx is None else w.lambdas[np.asarray(lam_idx)]
    V = w.n if loo else w.V
    foldid = np.arange(w.n, dtype=np.int32) if loo else tkm.tkm_make_folds(w.n, V, w.fold_seed)
    X, y = torch.from_numpy(w.X).cuda(), torch.from_numpy(w.y).cuda()
    taus = w.taus if len(w.taus) else None

    def ev():
        e = torch.cuda.Event(enable_timing=True)
        e.record()
        return e

    mon = ClockSampler(clocks_index)
    mon.start()
    mon.wait_ready()            # nvidia-smi's start-up stays outside the pass
    mon.mark()
    torch.cuda.reset_peak_memory_stats()
    e0 = ev()
    if w.m_landmarks:
        idx = wl.landmarks(w.n, w.m_landmarks, w.landmark_seed)
        if nystrom_streamed:
            e1 = e0
            spec = tkm.tkm_spectral_setup_nystrom_x(X, sigma, idx)
        else:
            Xl = X[torch.from_numpy(idx).cuda()]
            K_nm, K_mm = tkm.tkm_gram(X, sigma, Xl), tkm.tkm_gram(Xl, sigma)
            e1 = ev()
            spec = tkm.tkm_spectral_setup(nystrom=(K_nm, K_mm, idx))
            del K_nm, K_mm
        gram_bytes = w.n * w.m_landmarks * 8 + w.m_landmarks ** 2 * 8
    else:
        K = tkm.tkm_gram(X, sigma)
        e1 = ev()
        spec = tkm.tkm_spectral_setup(K)
        del K
        gram_bytes = w.n * w.n * 8
    e2 = ev()
    path = tkm.tkm_fit_path(spec, y, w.loss, lambdas, foldid, V, tol, MAXIT, smooth0=w.smooth0, eta=w.eta,
                            rounds=w.rounds, taus=taus, warm_tol=warm_tol, tf32_delta=tf32_delta, profile=profile,
                            gap_tol=gap_tol, delta_min_live=delta_min_live)
    e3 = ev()
    cv = tkm.tkm_exact_cv(path, y, foldid, w.T, len(lambdas), V)
    e4 = ev()
    e4.synchronize()
    clocks = mon.stop()
    if path.status != 0:
        raise RuntimeError("columns hit maxit: the timed work is not the stated work")
    out = dict(gram_ms=e0.elapsed_time(e1), setup_ms=e1.elapsed_time(e2), sweep_ms=e2.elapsed_time(e3),
               cv_ms=e3.elapsed_time(e4), col_iters=int(path.total_col_iters), B=path.B, r=spec.r, n=w.n,
               prof=path.profile(), profile_mode=profile, tf32_delta=tf32_delta, clocks=clocks, gram_bytes=gram_bytes, best_l=[int(b) for b in cv[3]],
               peak_mem_gb=torch.cuda.max_memory_allocated() / 1e9, iters_max=int(path.info()["iters"].max()))
    path.close()
    spec.close()
    torch.cuda.empty_cache()
    return out


def problem_summary(res, pk, traffic, what, knobs, probes=None, tkeys=None):
    tp = tensor_peaks(pk, res["clocks"].get("sm_mhz"))
    n, r = res["n"], res["r"]
    fams = family_rooflines(res["prof"], tp, traffic, probes, geom=(n, r, 1), hbm_peak=pk["hbm"], tkeys=tkeys,
                            single_tf32=knobs.get("tf32_delta") == 3)
    sweep_s = res["sweep_ms"] / 1e3
    total_ms = res["gram_ms"] + res["setup_ms"] + res["sweep_ms"] + res["cv_ms"]

    def dominance(f):
        # profile = 1 samples ONE exact and ONE delta iteration per batch, but a batch of 16 (or 32) iterations holds
        # one exact iteration and 15 (31) delta iterations: the tcgen05 families stand for 15 x their sampled time
        return f["sampled_ms"] * (15.0 if f["family"] >= 2 and res.get("profile_mode") != 2
                                  else 1.0)

    d = {"workload": what, "columns": res["B"], "launch_config": knobs,
         "fits_per_s": res["B"] / (total_ms / 1e3), "fits_per_s_sweep_only": res["B"] / sweep_s,
         "stages_ms": {"gram": res["gram_ms"], "eig_setup": res["setup_ms"], "sweep": res["sweep_ms"],
                       "exact_cv": res["cv_ms"]},
         "col_iters": res["col_iters"], "max_iters_of_a_column": res["iters_max"],
         "sweep_useful_tflops": 4.0 * n * r * res["col_iters"] / sweep_s / 1e12,
         "gram_gbs": res["gram_bytes"] / (res["gram_ms"] / 1e3) / 1e9 if res["gram_ms"] > 0 else None,
         "gram_frac_of_hbm": res["gram_bytes"] / (res["gram_ms"] / 1e3) / 1e9 / pk["hbm"] if res["gram_ms"] > 0 else None,
         "roofline": binding_side(max(fams, key=dominance)) if fams else None,
         "roofline_families": [binding_side(f) for f in fams],
         "peak_device_memory_gb": res["peak_mem_gb"], "clocks": res["clocks"], "selected_lambda_index": res["best_l"]}
    return d


def narrow_hbm_roofline(res, pk):
    """Narrow live batch: both FP64 contractions stream U once per launch; algorithmic bytes per launch =
    n r 8 (the U operand) + live (r + n) 8 (moving operand in, result out), from the sampled launches."""
    pr = res["prof"]
    out = []
    n, r = res["n"], res["r"]
    for i in (0, 1, 2, 3):     # 2, 3: the tcgen05 delta-form contractions (hi + lo FP32 operands: the same bytes)
        nl = int(pr["launches"][i])
        if not nl:
            continue
        live = pr["flops"][i] / nl / (2.0 * n * r)          # average live columns of the sampled launches
        ub = 4.0 if (i >= 2 and res.get("tf32_delta") == 3) else 8.0   # single-TF32 mode reads the hi parts only
        by = n * r * ub + live * (r + n) * ub + (live * (n if i == 2 else r) * 4.0 if i >= 2 else 0.0)
        ms = pr["ms"][i] / nl
        name = FAMILY[i].replace("3xTF32", "1xTF32") if res.get("tf32_delta") == 3 else FAMILY[i]
        out.append({"bound": "hbm", "kernel": name, "achieved": by / (ms / 1e3) / 1e9, "peak": pk["hbm"],
                    "unit": "GB/s", "frac": by / (ms / 1e3) / 1e9 / pk["hbm"], "traffic": None,
                    "avg_live_columns": live, "avg_launch_ms": ms, "algorithmic_bytes_per_launch": by,
                    "sampled_launches": nl})
    return out


GEMM_PROBE_SHAPES = [(64, 256, 2000), (64, 2000, 2000), (128, 2000, 2000), (300, 2000, 2000), (64, 18944, 2000),
                     (300, 10000, 10000), (512, 10000, 10000), (1100, 10000, 10000), (300, 20000, 20000),
                     (900, 20000, 20000), (600, 100000, 4096), (600, 4096, 100000)]


def run_gemm_probe(args):
    """`--workload gemm_probe`: the two contraction kernels alone, Dt[N][M] = P[N][K] Q[M][K]^T on random operands
    (N slots, M rows of U, K contraction depth), `--probe-iters` back-to-back launches timed with CUDA events:
    the tcgen05 3xTF32 pair kernel (tkm_tf32x3_gemm_nt) and the FP64 DMMA kernel (tkm_gemm_probe)."""
    import torch
    import paper_2606_06742_b200 as tkm
    tkm.lib()
    torch.cuda.set_device(0)
    pk = peaks()
    rows = []
    for (N, M, K) in GEMM_PROBE_SHAPES:
        P = torch.randn((N, K), device="cuda", dtype=torch.float64)
        Q = torch.randn((M, K), device="cuda", dtype=torch.float64)
        _, ms = tkm.tkm_tf32x3_gemm_nt(P, Q, iters=args.probe_iters)
        del P, Q
        torch.cuda.empty_cache()
        ms64 = tkm.tkm_gemm_probe(-1, 1, N, M, K, iters=max(2, args.probe_iters // 4)) if N * M * K <= 4e11 else None
        fl = 2.0 * N * M * K
        rows.append({"N": N, "M": M, "K": K, "tcgen05_3xtf32_us": 1e3 * ms, "tcgen05_useful_tflops": fl / ms / 1e9,
                     "tcgen05_frac_of_contract_peak": fl / ms / 1e9 / (pk["bf16_sus"] * NOMINAL_RATIO["f32"]),
                     "dmma_f64_us": None if ms64 is None else 1e3 * ms64,
                     "dmma_tflops": None if ms64 is None else fl / ms64 / 1e9})
    print(json.dumps({"workload": "gemm_probe", "iters": args.probe_iters, "peaks": pk,
                      "tf32x3_contract_peak_tflops": pk["bf16_sus"] * NOMINAL_RATIO["f32"], "shapes": rows}))


def run_setup_probe(args):
    """`--workload setup_probe`: wall time of the spectral set-up alone on configs[1]'s five Gram matrices, call by
    call (`--probe-iters` calls each): all five at once (tkm_spectral_setup_multi), one after the other
    (tkm_spectral_setup x 5), a single one through the multi entry, and -- as a library yardstick, never on the
    product path -- torch.linalg.eigh x 5.  The spread of the per-call times is the point (profiles/r02_host_stalls.md)."""
    import torch
    import paper_2606_06742_b200 as tkm
    tkm.lib()
    torch.cuda.set_device(0)
    w = wl.config1(seed=1001)
    X = torch.from_numpy(w.X).cuda()

    def timed(fn, G):
        Ks = tkm.tkm_gram_multi(X, w.sigmas[:G])
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        out = fn(Ks)
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) * 1e3
        for o in out:
            if hasattr(o, "close"):
                o.close()
        return dt

    cases = [("setup_multi_5", lambda Ks: tkm.tkm_spectral_setup_multi(Ks), 5),
             ("setup_single_x5", lambda Ks: [tkm.tkm_spectral_setup(K) for K in Ks], 5),
             ("setup_multi_1", lambda Ks: tkm.tkm_spectral_setup_multi(Ks), 1),
             ("torch_linalg_eigh_x5", lambda Ks: [torch.linalg.eigh(K) for K in Ks], 5)]
    out = {"workload": "setup_probe", "n": w.n, "calls": args.probe_iters, "unit": "ms of wall time per call"}
    for name, fn, G in cases:
        timed(fn, G)
        ts = [timed(fn, G) for _ in range(args.probe_iters)]
        out[name] = {"median": float(np.median(ts)), "min": min(ts), "max": max(ts), "each": [round(t, 1) for t in ts]}
    print(json.dumps(out))


def run_single(args):
    """`--workload` other than config1: one GPU, one problem, one JSON line."""
    import torch
    import paper_2606_06742_b200 as tkm
    tkm.lib()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (libtkm has no CPU fallback)")
    torch.cuda.set_device(0)
    name = args.workload
    pk, traffic = peaks(), traffic_table()
    kw = dict(tf32_delta=TF32_DELTA_LARGE if args.tf32_delta < 0 else args.tf32_delta, tol=args.tol, warm_tol=WARM_TOL,
              profile=2 if args.profile_all else 1, gap_tol=args.gap_tol, delta_min_live=args.delta_min_live)
    if name.startswith("nystrom_"):
        w = wl.nystrom_paper_shape(name[len("nystrom_"):])
        kw["nystrom_streamed"] = True
        what = ("%s: Nystrom smoothed-hinge SVM with the shape of the paper's Table-4 data set (synthetic rows), n=%d, "
                "p=%d, m=%d landmarks, %d folds, %d lambdas 1e2..1e-5" % (name, w.n, w.p, w.m_landmarks, w.V, w.L))
    elif name == "loo_config1":
        w = wl.config1(sigma_mults=(1.0,))
        if args.loo_lambdas:
            w.lambdas = w.lambdas[np.linspace(0, w.L - 1, args.loo_lambdas).round().astype(int)]
        kw["loo"] = True
        what = ("loo_config1: leave-one-out form of Algorithm 1 (PAPER.md:178-224, V = n) on configs[1]'s data, median "
                "bandwidth: n=%d, %d lambdas, B = L (n + 1) = %d columns" % (w.n, w.L, w.L * (w.n + 1)))
    elif name.startswith("narrow_"):
        cfg = int(name[-1])
        w = wl.CONFIGS[cfg]()
        frac = {1: [0.5], 2: [0.4, 0.7], 4: [0.3, 0.5, 0.7, 0.9]}[args.narrow_L]
        kw["lam_idx"] = [int(round(f * (w.L - 1))) for f in frac]
        kw["tf32_delta"] = TF32_DELTA_LARGE if args.tf32_delta < 0 else args.tf32_delta   # 0: the all-FP64 DMMA stream
        what = ("%s: BASELINE.json configs[%d] at full n = %d with %d lambda(s) (grid indices %s): B = %d columns, the "
                "HBM-bound narrow batch of SURVEY.md 8(d)" % (name, cfg, w.n, args.narrow_L, kw["lam_idx"],
                                                               w.T * args.narrow_L * (w.V + 1)))
    else:
        cfg = int(name[-1])
        w = wl.CONFIGS[cfg]()
        what = "BASELINE.json configs[%d] at full size: n=%d, p=%d, %d folds, %d lambdas%s%s" % (
            cfg, w.n, w.p, w.V, w.L, ", tau %s" % list(w.taus) if len(w.taus) else "",
            ", Nystrom m=%d" % w.m_landmarks if w.m_landmarks else "")
    res = None
    for it in range(args.warmup + args.steps):
        res = run_problem(tkm, w, **kw)          # the last pass is reported (a pass takes seconds to a minute)
    knobs = {"tf32_delta": kw["tf32_delta"], "stop_tol": args.tol, "warm_start_rounds_tol": WARM_TOL,
             "gap_tol": args.gap_tol, "profile": kw["profile"], "delta_min_live": args.delta_min_live,
             "l2": "inputs larger than L2" if w.n * res["r"] * 8 > 126e6 else "not flushed"}
    tkeys = {2: "config3_tcgen05_full_width", 3: "config3_tcgen05_full_width"} if name == "config3" else None
    d = problem_summary(res, pk, traffic, what, knobs, tkeys=tkeys)
    total_ms = sum(d["stages_ms"].values())
    line = {"metric": METRIC, "value": d["fits_per_s"], "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": what, "columns_per_step": d["columns"],
                       "value_is": "columns / (Gram + setup + sweep + exact CV)"}}
    line.update({k: v for k, v in d.items() if k != "workload"})
    if name.startswith("narrow_"):
        line["roofline_hbm"] = narrow_hbm_roofline(res, pk)
        if line["roofline_hbm"]:
            line["roofline"] = max(line["roofline_hbm"], key=lambda f: f["avg_launch_ms"])
    if args.profile_all:
        line["time_weighted"] = time_weighted(res["prof"], tensor_peaks(pk, res["clocks"].get("sm_mhz")),
                                              single_tf32=kw["tf32_delta"] == 3)
    line["gpu_launches"] = int(tkm.tkm_launch_count())
    print(json.dumps(line))


# ----------------------------------------------------------------------------------------- CUDA arm, default line
def run_ours(args, w, rank, world):
    import torch
    import paper_2606_06742_b200 as tkm
    from paper_2606_06742_b200 import ranks
    tkm.lib()   # raises if libtkm.so is missing: there is no fallback
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (libtkm has no CPU fallback)")
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    tol = STOP_TOL["f64"]
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X = torch.from_numpy(w.X).cuda()
    y = torch.from_numpy(w.y).cuda()
    Xh = torch.from_numpy(w.X).pin_memory()
    yh = torch.from_numpy(w.y).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    prof = dict(ms=np.zeros(4), flops=np.zeros(4), launches=np.zeros(4, dtype=np.int64), col_iters=0)
    stage = np.zeros(4)
    e2e_stage = np.zeros(5)     # summed over the e2e steps: copy-in, gram, eig, sweep, cv + coefficients + copy-out (ms)

    def ev():
        e = torch.cuda.Event(enable_timing=True)
        e.record()
        return e

    def step_device(collect, profile=1, mode=None):
        """One pass of the hot path: S1 + S2 per bandwidth, S3-S8 for all bandwidths as groups of one
        sweep (tkm_fit_path_multi), S9 per bandwidth."""
        flush.zero_()
        e0 = ev()
        Ks = tkm.tkm_gram_multi(X, w.sigmas)                               # one distance pass, 5 exp + writes
        e1 = ev()
        specs = tkm.tkm_spectral_setup_multi(Ks)                           # the 5 decompositions overlap
        del Ks
        e2 = ev()
        paths = tkm.tkm_fit_path_multi(specs, y, w.loss, w.lambdas, foldid, w.V, tol, MAXIT, smooth0=w.smooth0,
                                       eta=w.eta, rounds=w.rounds, warm_tol=WARM_TOL,
                                       tf32_delta=TF32_DELTA if mode is None else mode,
                                       profile=profile, delta_min_live=args.delta_min_live)
        e3 = ev()
        best = [int(tkm.tkm_exact_cv(path, y, foldid, w.T, w.L, w.V)[3][0]) for path in paths]
        e4 = ev()
        pr = None
        if collect:
            e4.synchronize()
            pr = paths[0].profile()
            pr["col_iters"] = sum(path.total_col_iters for path in paths)
            pr["stage"] = np.array([e0.elapsed_time(e1), e1.elapsed_time(e2), e2.elapsed_time(e3), e3.elapsed_time(e4)])
            if any(path.status != 0 for path in paths):
                raise RuntimeError("columns hit maxit: the timed work is not the stated work")
        for path in paths:
            path.close()
        for spec in specs:
            spec.close()
        return best, pr

    def step_e2e():
        flush.zero_()
        r = tkm.tkm_train_tune_host(Xh.numpy(), yh.numpy(), np.asarray(w.sigmas, dtype=np.float64), w.loss, w.lambdas,
                                    foldid, w.V, tol, MAXIT, smooth0=w.smooth0, eta=w.eta, rounds=w.rounds,
                                    warm_tol=WARM_TOL, tf32_delta=TF32_DELTA)
        if r["status"] != 0:
            raise RuntimeError("columns hit maxit in the e2e leg")
        e2e_stage[:] += r["stage_ms"]
        nb_in = Xh.numel() * 8 + yh.numel() * 8
        nb_out = r["cv_loss"].nbytes + r["cv_err"].nbytes + r["cv_mean"].nbytes + r["best_l"].nbytes + \
            r["alpha"].nbytes + r["beta0"].nbytes
        return nb_in, nb_out

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(ms):
        return ranks.max_over_ranks(ms, dist, device="cuda")

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    for _ in range(args.warmup):
        step_device(False)
    if rank == 0:
        sampler.wait_ready()
    barrier()
    sampler.mark()
    tkm.tkm_launch_count_reset()
    s_ev = ev()
    step_marks = [s_ev]
    for _ in range(args.steps):
        _, pr = step_device(True)
        step_marks.append(ev())
        for k in ("ms", "flops", "launches"):
            prof[k] += pr[k]
        prof["col_iters"] += pr["col_iters"]
        stage += pr["stage"]
    e_ev = ev()
    barrier()
    launches = tkm.tkm_launch_count()
    ms_total = max_over_ranks(s_ev.elapsed_time(e_ev))
    clocks = sampler.stop() if rank == 0 else None

    # e2e leg: host buffers -> tkm_train_tune_host -> host results
    step_e2e()
    barrier()
    e2e_stage[:] = 0.0
    s_ev = ev()
    for _ in range(args.steps):
        nb_in, nb_out = step_e2e()
    e_ev = ev()
    barrier()
    ms_e2e = max_over_ranks(s_ev.elapsed_time(e_ev))

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    fits_per_step = w.B * len(w.sigmas)
    ms_per_step = ms_total / args.steps
    value = world * fits_per_step / (ms_per_step / 1e3)
    pk, traffic = peaks(), traffic_table()
    tp = tensor_peaks(pk, clocks.get("sm_mhz") if clocks else None)
    probes = library_probes(tkm) if world == 1 else None
    fams = family_rooflines(prof, tp, traffic, probes, geom=(w.n, w.n, len(w.sigmas)), hbm_peak=pk["hbm"],
                            single_tf32=TF32_DELTA == 3)
    # the FP64 DMMA kernel (both epilogues) and the tcgen05 kernel (both delta forms): the dominant one -- the larger
    # share of the sampled kernel time -- is `roofline`
    roof_f64, roof_tf32 = merge_families(fams, (0, 1)), merge_families(fams, (2, 3))
    if roof_f64 is not None:
        tr = traffic.get("config1_dmma_full_width")
        roof_f64["traffic"], roof_f64["traffic_source"] = (tr[0], tr[1]) if tr else (None, None)
    if roof_tf32 is not None:
        tr = traffic.get("config1_tcgen05_full_width")
        roof_tf32["traffic"], roof_tf32["traffic_source"] = (tr[0], tr[1]) if tr else (None, None)
    if TF32_DELTA >= 2 and roof_tf32 is not None:
        roofline, roofline_other = roof_tf32, roof_f64
    else:
        roofline, roofline_other = roof_f64, roof_tf32
    sweep_s = stage[2] / 1e3
    stage_sum = float(stage.sum()) / args.steps
    gram_gbs = len(w.sigmas) * w.n * w.n * 8 / (stage[0] / args.steps / 1e3) / 1e9
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(w),
            "launch_config": {"tf32_delta": TF32_DELTA, "sampled_kernel_events": "profile=1 in the timed region"},
            "stages_ms_per_step": {"gram": stage[0] / args.steps, "eig_setup": stage[1] / args.steps,
                                   "sweep": stage[2] / args.steps, "exact_cv": stage[3] / args.steps},
            "ms_per_step_outside_stages": ms_per_step - stage_sum,
            "ms_of_each_step": [round(a.elapsed_time(b), 2) for a, b in zip(step_marks[:-1], step_marks[1:])],
            "exact_cv_ms_per_grid": stage[3] / args.steps / len(w.sigmas),
            "fits_per_s_sweep_only": args.steps * fits_per_step / sweep_s,
            "col_iters_per_step": prof["col_iters"] / args.steps,
            "sweep_useful_tflops": 4.0 * w.n * w.n * prof["col_iters"] / sweep_s / 1e12,
            "gram_gbs": gram_gbs, "gram_frac_of_hbm": gram_gbs / pk["hbm"],
            "roofline": binding_side(roofline), "roofline_other_kernel": binding_side(roofline_other), "clocks": clocks, "gpu_launches": int(launches),
            "e2e": {"value": world * fits_per_step / (ms_e2e / args.steps / 1e3), "unit": UNIT,
                    "h2d_bytes_per_step": int(nb_in), "d2h_bytes_per_step": int(nb_out),
                    "ms_per_step": ms_e2e / args.steps,
                    "stages_ms_per_step": {k: float(v) / args.steps for k, v in zip(("h2d", "gram", "eig_setup", "sweep",
                                                                                      "cv_coef_d2h"), e2e_stage)},
                    "ms_per_step_outside_stages": (ms_e2e - float(e2e_stage.sum())) / args.steps}}
    if world == 1:
        line["peaks_measured_here"] = probes
        # every launch of one more step, outside the timed region: the time-weighted fractions
        _, pr2 = step_device(True, profile=2)
        line["roofline_time_weighted"] = time_weighted(pr2, tp, single_tf32=TF32_DELTA == 3)
        if TF32_DELTA == 2:
            # beyond BASELINE.json's "3xTF32 split": the same step with single-TF32 increment products (tf32_delta = 3,
            # include/tkm.h) -- one warm-up and one measured step outside the timed region; NOT part of `value`
            step_device(False, mode=3)
            b3, pr3 = step_device(True, mode=3)
            line["single_tf32_increments"] = {
                "what": "tf32_delta = 3: increments contracted in one TF32 product (hi parts only: half the operand bytes, "
                        "a third of the MMAs); FP64 state, exact restarts and stop tests unchanged, same 1e-10 parity "
                        "tests (tests/test_gpu_parity.py); an option, not the configuration of `value`",
                "sweep_ms": float(pr3["stage"][2]), "fits_per_s_sweep_only": fits_per_step / (float(pr3["stage"][2]) / 1e3),
                "step_ms": float(pr3["stage"].sum()), "fits_per_s": fits_per_step / (float(pr3["stage"].sum()) / 1e3),
                "col_iters": int(pr3["col_iters"]), "selected_lambda_index": b3}
        if not args.no_large:
            # the largest full-kernel single-GPU configuration of BASELINE.json: one pass, its own roofline and clocks
            del X, y, flush
            torch.cuda.empty_cache()
            w3 = wl.config3()
            r3 = run_problem(tkm, w3, tf32_delta=TF32_DELTA_LARGE, tol=1e-10, warm_tol=WARM_TOL, profile=1,
                             clocks_index=local)
            line["large_config"] = problem_summary(
                r3, pk, traffic, "BASELINE.json configs[3]: kernel quantile regression tau in {0.1,0.5,0.9} on one U, "
                "n=20000, p=28, 5 folds, 50 lambdas 1e1..1e-6, gamma 1 -> 1/512 in 4 rounds; ONE pass (no warm-up "
                "pass, outside the timed region of `value`)",
                {"tf32_delta": TF32_DELTA_LARGE, "stop_tol": 1e-10, "warm_start_rounds_tol": WARM_TOL,
                 "l2": "inputs larger than L2 (U Lam and U^T: 3.2 GB each)"}, probes,
                tkeys={2: "config3_tcgen05_full_width", 3: "config3_tcgen05_full_width"})
            if TF32_DELTA_LARGE == 2:
                # the same pass with single-TF32 increment products (tf32_delta = 3): an option, reported beside
                r3s = run_problem(tkm, w3, tf32_delta=3, tol=1e-10, warm_tol=WARM_TOL, profile=1, clocks_index=local)
                line["large_config"]["single_tf32_increments"] = {
                    "sweep_ms": r3s["sweep_ms"], "fits_per_s_sweep_only": r3s["B"] / (r3s["sweep_ms"] / 1e3),
                    "col_iters": r3s["col_iters"], "selected_lambda_index": r3s["best_l"], "clocks": r3s["clocks"]}
        ncol, secs, its = oracle_sample_step(w)
        line["cpu_baseline"] = {"value": ncol / secs, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
                                "sample": sample_text(w, ncol, secs, its)}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--dtype", default="f64", choices=["f64"])
    ap.add_argument("--workload", default="config1",
                    choices=["config1", "config2", "config3", "config4", "nystrom_covtype", "nystrom_mnist8m46",
                             "loo_config1", "narrow_config2", "narrow_config3", "gemm_probe", "setup_probe"],
                    help="config1 = BASELINE.json's metric configuration (the bench line, which also carries configs[3] "
                         "as `large_config`); the others are single-GPU measurements of one problem "
                         "(use --steps 1 --warmup 0 or 1: a pass takes seconds to a minute)")
    ap.add_argument("--tol", type=float, default=1e-10, help="stop tolerance of the --workload runs other than config1")
    ap.add_argument("--tf32-delta", type=int, default=-1, help="override the delta-form mode of a --workload run")
    ap.add_argument("--gap-tol", type=float, default=0.0,
                    help="outer control of PAPER.md:220-222 (reading G23) for a --workload run; 0 = fixed schedule")
    ap.add_argument("--delta-min-live", type=int, default=0,
                    help="live columns at or below which a delta-form sweep runs all-FP64 (0 = the library's cost model)")
    ap.add_argument("--narrow-L", type=int, default=1, choices=[1, 2, 4])
    ap.add_argument("--loo-lambdas", type=int, default=0, help="loo_config1: use this many lambdas of the grid (0 = all 50)")
    ap.add_argument("--probe-iters", type=int, default=20, help="gemm_probe: launches per shape")
    ap.add_argument("--profile-all", action="store_true", help="time every contraction launch (profile = 2)")
    ap.add_argument("--clock-period-ms", type=int, default=200,
                    help="nvidia-smi sampling period of the clocks evidence; 0 = no sampler (experiments only)")
    ap.add_argument("--no-large", action="store_true", help="default line: skip the configs[3] pass (`large_config`)")
    args = ap.parse_args()
    ClockSampler.PERIOD_MS = args.clock_period_ms
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.workload != "config1":
        if args.impl != "ours" or world != 1 or args.gpus != 1:
            raise SystemExit("--workload %s: one GPU, --impl ours only" % args.workload)
        if args.workload == "setup_probe":
            return run_setup_probe(args)
        return run_gemm_probe(args) if args.workload == "gemm_probe" else run_single(args)
    if args.tf32_delta >= 0:
        global TF32_DELTA
        TF32_DELTA = args.tf32_delta
    from paper_2606_06742_b200.ranks import replica_seed
    w = wl.config1(seed=replica_seed(1001, rank if args.impl == "ours" else 0))
    if args.impl == "reference":
        run_reference(args, w, rank)
    else:
        run_ours(args, w, rank, world)


if __name__ == "__main__":
    main()
