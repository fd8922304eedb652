#!/usr/bin/env python
"""bench.py -- the driver's benchmark contract for libtkm.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--dtype f64]

Metric (BASELINE.json): (lambda x fold) path fits per second on BASELINE.json configs[1]
(smoothed-hinge kernel SVM, n=2000, p=50, 5 folds, 50 lambdas x 5 sigma values).  One STEP is one pass
of the whole hot path over that workload: for each of the 5 bandwidths  S1 Gram -> S2 spectral setup
-> S9 exact CV, with the S3-S8 sweeps of the 5 bandwidths (50 x (5+1) columns each) run together as groups
of one launch sequence (tkm_fit_path_multi), and S10 coefficients in the e2e leg.
`value` = columns fitted per second by the whole job, X and y resident in HBM before the timed
region; `e2e` = the same through tkm_train_tune_host from pinned HOST buffers.

N > 1 (torchrun): the path has no exchange step -- every rank runs the same-size workload on its own
seeded data set (independent problems, "weak" scaling); the only communication is the barrier and the
max-over-ranks of the device time.

`--impl reference` times the FP64 CPU oracle (oracle/, test infrastructure) on a bounded sample of
the same workload on the host cores; rank 0 only.
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

import workloads as wl  # noqa: E402

METRIC = "lambda_x_fold_path_fits_per_s"
UNIT = "fits/s"
STOP_TOL = {"f64": 1e-12, "f32": 1e-6}
MAXIT = 200000
# Stop tolerance of the smoothing rounds 0..R-2, which only produce warm starts for the last round (the
# result is the minimiser at the final smoothing level, whatever the start): DESIGN.md "Schedule".
WARM_TOL = 1e-3
# Delta form of the U^T contraction (tkm_loss_opts.tf32_delta = 1): zeta advances by 3xTF32 increments on the
# tcgen05 tensor cores, with the exact FP64 DMMA contraction and the stop test on the last iteration of every
# 16-iteration batch and in the narrow tail.  Same fixed point and the same 1e-10 parity bar as the all-FP64
# sweep.  Mode 2 (both contractions) is 4 % faster still at n = 2000 and 3.2x at n = 20000, but
# it makes a bandwidth-bound tcgen05 kernel the dominant one; mode 1 keeps the FP64 DMMA GEMM dominant.
TF32_DELTA = 1
# nominal dense tensor ratios to bf16 (B200_PROFILING.md / B300_MICROARCH.md tables): FP64 45 TF,
# TF32 1125 TF, bf16 2250 TF.  3xTF32 does three MMAs per useful one.
NOMINAL_RATIO = {"f64": 45.0 / 2250.0, "f32": (1125.0 / 2250.0) / 3.0}
# dram bytes per launch of the dominant kernel from the committed ncu --set full capture
# (profiles/): filled in by hand after each capture, None until one exists.
NCU_TRAFFIC_BYTES_PER_LAUNCH = 218.0e6   # profiles/r01c: full-width launch, dram read + write
NCU_TRAFFIC_TF32_BYTES_PER_LAUNCH = 271.0e6  # profiles/r01e: tcgen05 ZetaEpi kernel, full-width launch
# columns of the bounded CPU sample: all V+1 hold-out settings x these lambda indices, one sigma
CPU_SAMPLE_LAMBDA_IDX = (0, 12, 24, 36, 49)
CPU_SAMPLE_SIGMA_IDX = 2


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return dict(hbm=d["hbm_gbs"], bf16_burst=d["bf16_tflops"], bf16_sus=d["bf16_tflops_sustained"],
                    src="measured")
    return dict(hbm=6650.0, bf16_burst=1590.0, bf16_sus=1400.0, src="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

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
        for ln in self.lines:
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
def oracle_sample_step(w, want_all=False):
    """One bounded sample of the workload on the CPU oracle: one sigma, 5 lambdas x (V+1) columns,
    Gram + eigh + path + exact CV.  Returns (#columns fitted, seconds)."""
    import oracle as o
    t0 = time.perf_counter()
    sigma = float(w.sigmas[CPU_SAMPLE_SIGMA_IDX])
    foldid = o.make_folds(w.n, w.V, w.fold_seed)
    K = o.gram_rbf(w.X, sigma)
    spec = o.spectral_setup(K)
    L, V = w.L, w.V
    cols = [v * L + l for v in range(V + 1) for l in CPU_SAMPLE_LAMBDA_IDX if l < L]
    res = o.fit_path(spec, w.y, w.loss, w.lambdas, foldid, V, taus=w.taus, smooth0=w.smooth0, eta=w.eta,
                     rounds=w.rounds, tol=STOP_TOL["f64"], maxit=MAXIT, columns=cols)
    o.exact_cv(spec, res, w.y, foldid, w.loss, w.taus)
    return len(cols), time.perf_counter() - t0, int(res.iters.sum())


def blas_threads():
    try:
        from threadpoolctl import threadpool_info
        return max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
    except Exception:
        return os.cpu_count() or 1


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
    sample = ("sigma index %d, lambda indices %s x %d hold-out settings = %d of %d columns per step, "
              "full n; Gram + eigh + path + exact CV" % (CPU_SAMPLE_SIGMA_IDX, list(CPU_SAMPLE_LAMBDA_IDX),
                                                        w.V + 1, fits // max(args.steps, 1), w.B * len(w.sigmas)))
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": workload_config(w, "f64", warm_tol=STOP_TOL["f64"]),
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_config(w, dtype, warm_tol=None):
    return {"workload": "BASELINE.json configs[1]: smoothed-hinge kernel SVM, n=%d, p=%d, %d folds, %d lambdas "
                        "1e2..1e-5 x %d sigma (median x {0.25,0.5,1,2,4}), delta 1 -> 1/512 in %d rounds, %s"
                        % (w.n, w.p, w.V, w.L, len(w.sigmas), w.rounds, dtype),
            "n": w.n, "p": w.p, "folds": w.V, "lambdas": w.L, "sigmas": len(w.sigmas),
            "columns_per_step": w.B * len(w.sigmas), "stop_tol": STOP_TOL[dtype], "warm_start_rounds_tol": WARM_TOL if warm_tol is None else warm_tol,
            "tf32_delta": TF32_DELTA if warm_tol is None else 0, "maxit": MAXIT,
            "l2": "flushed between steps (256 MiB memset)", "parallelism": "independent replicas, no collective"}


# ----------------------------------------------------------------------------------------- CUDA arm
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
    dt = args.dtype
    sweep_dt = tkm.F64 if dt == "f64" else tkm.F32
    tol = STOP_TOL[dt]
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X = torch.from_numpy(w.X).cuda()
    y = torch.from_numpy(w.y).cuda()
    Xh = torch.from_numpy(w.X).pin_memory()
    yh = torch.from_numpy(w.y).pin_memory()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    prof = dict(ms=np.zeros(4), flops=np.zeros(4), launches=np.zeros(4, dtype=np.int64), col_iters=0)
    stage = np.zeros(4)
    e2e_stage = np.zeros(5)     # last e2e step: copy-in, gram, eig, sweep, cv + coefficients + copy-out (ms)

    def ev():
        e = torch.cuda.Event(enable_timing=True)
        e.record()
        return e

    def step_device(collect):
        """One pass of the hot path: S1 + S2 per bandwidth, S3-S8 for all bandwidths as groups of one
        sweep (tkm_fit_path_multi), S9 per bandwidth."""
        flush.zero_()
        e0 = ev()
        Ks = tkm.tkm_gram_multi(X, w.sigmas)                               # one distance pass, 5 exp + writes
        e1 = ev()
        specs = tkm.tkm_spectral_setup_multi(Ks, sweep_dtype=sweep_dt)     # the 5 decompositions overlap
        del Ks
        e2 = ev()
        paths = tkm.tkm_fit_path_multi(specs, y, w.loss, w.lambdas, foldid, w.V, tol, MAXIT, smooth0=w.smooth0,
                                       eta=w.eta, rounds=w.rounds, warm_tol=WARM_TOL, tf32_delta=TF32_DELTA, profile=True)
        e3 = ev()
        best = [int(tkm.tkm_exact_cv(path, y, foldid, w.T, w.L, w.V)[3][0]) for path in paths]
        e4 = ev()
        if collect:
            e4.synchronize()
            stage[0] += e0.elapsed_time(e1)
            stage[1] += e1.elapsed_time(e2)
            stage[2] += e2.elapsed_time(e3)
            stage[3] += e3.elapsed_time(e4)
            pr = paths[0].profile()
            prof["ms"] += pr["ms"]
            prof["flops"] += pr["flops"]
            prof["launches"] += pr["launches"]
            prof["col_iters"] += sum(path.total_col_iters for path in paths)
            if any(path.status != 0 for path in paths):
                raise RuntimeError("columns hit maxit: the timed work is not the stated work")
        for path in paths:
            path.close()
        for spec in specs:
            spec.close()
        return best

    def step_e2e():
        flush.zero_()
        r = tkm.tkm_train_tune_host(Xh.numpy(), yh.numpy(), np.asarray(w.sigmas, dtype=np.float64), w.loss, w.lambdas,
                                    foldid, w.V, tol, MAXIT, smooth0=w.smooth0, eta=w.eta, rounds=w.rounds,
                                    warm_tol=WARM_TOL, tf32_delta=TF32_DELTA, sweep_dtype=sweep_dt)
        if r["status"] != 0:
            raise RuntimeError("columns hit maxit in the e2e leg")
        e2e_stage[:] = r["stage_ms"]
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

    for _ in range(args.warmup):
        step_device(False)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    barrier()
    tkm.tkm_launch_count_reset()
    s_ev = ev()
    for _ in range(args.steps):
        step_device(True)
    e_ev = ev()
    barrier()
    launches = tkm.tkm_launch_count()
    ms_total = max_over_ranks(s_ev.elapsed_time(e_ev))
    clocks = sampler.stop() if rank == 0 else None

    # e2e leg: host buffers -> tkm_train_tune_host -> host results
    step_e2e()
    barrier()
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
    pk = peaks()

    def family(idx, name, peak_tf, peak_src, traffic):
        ms, fl, nl = float(prof["ms"][idx].sum()), float(prof["flops"][idx].sum()), int(prof["launches"][idx].sum())
        ach = (fl / 1e12) / (ms / 1e3) if ms > 0 else 0.0
        return {"bound": "tensor", "kernel": name, "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s",
                "frac": ach / peak_tf, "traffic": traffic, "peak_source": peak_src, "sampled_launches": nl,
                "avg_launch_ms": ms / max(1, nl), "avg_flops_per_launch": fl / max(1, nl),
                "sampled_ms": ms}

    # FP64 DMMA kernel: peak = measured bf16 sustained x nominal FP64/bf16 ratio
    roof_f64 = family([0, 1], "gemm_f64_tma_kernel (FP64 DMMA: exact iterations and the narrow tail; GEMM-A loss "
                      "epilogue + GEMM-B spectral epilogue)", pk["bf16_sus"] * NOMINAL_RATIO["f64"],
                      "%s bf16 sustained %.1f TF/s x nominal f64/bf16 ratio %.4f" %
                      (pk["src"], pk["bf16_sus"], NOMINAL_RATIO["f64"]), NCU_TRAFFIC_BYTES_PER_LAUNCH)
    # tcgen05 3xTF32 kernel: every useful product costs three TF32 MMAs; achieved counts the USEFUL flops only
    roof_tf32 = family([2, 3], "gemm_tf32x3_kernel (tcgen05 3xTF32 delta forms: F+ = Fbar - U Lam da with loss "
                       "epilogue, zeta += U^T dz with rho epilogue)", pk["bf16_sus"] * NOMINAL_RATIO["f32"],
                       "%s bf16 sustained %.1f TF/s x nominal tf32/bf16 ratio 0.5 / 3 MMAs per useful product" %
                       (pk["src"], pk["bf16_sus"]), NCU_TRAFFIC_TF32_BYTES_PER_LAUNCH)
    # the dominant kernel family is the one with the larger share of the sweep: per batch of 16 iterations the
    # delta forms run 15 tcgen05 pairs and one DMMA pair, the all-FP64 sweep 16 DMMA pairs
    if TF32_DELTA == 2 and roof_tf32["sampled_launches"]:
        roofline, roofline_other = roof_tf32, roof_f64
    else:
        roofline, roofline_other = roof_f64, (roof_tf32 if roof_tf32["sampled_launches"] else None)
    sweep_s = stage[2] / 1e3
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": dt, "data": "synthetic", "config": workload_config(w, dt),
            "stages_ms_per_step": {"gram": stage[0] / args.steps, "eig_setup": stage[1] / args.steps,
                                   "sweep": stage[2] / args.steps, "exact_cv": stage[3] / args.steps},
            "exact_cv_ms_per_grid": stage[3] / args.steps / len(w.sigmas),
            "fits_per_s_sweep_only": args.steps * fits_per_step / sweep_s,
            "col_iters_per_step": prof["col_iters"] / args.steps,
            "sweep_useful_tflops": 4.0 * w.n * w.n * prof["col_iters"] / sweep_s / 1e12,
            "gram_gbs": len(w.sigmas) * w.n * w.n * 8 / (stage[0] / args.steps / 1e3) / 1e9,
            "roofline": roofline, "roofline_other_kernel": roofline_other, "clocks": clocks, "gpu_launches": int(launches),
            "e2e": {"value": world * fits_per_step / (ms_e2e / args.steps / 1e3), "unit": UNIT,
                    "h2d_bytes_per_step": int(nb_in), "d2h_bytes_per_step": int(nb_out),
                    "ms_per_step": ms_e2e / args.steps,
                    "last_step_stages_ms": {k: float(v) for k, v in zip(("h2d", "gram", "eig_setup", "sweep",
                                                                          "cv_coef_d2h"), e2e_stage)}}}
    if world == 1:
        ncol, secs, its = oracle_sample_step(w)
        line["cpu_baseline"] = {"value": ncol / secs, "unit": UNIT, "cores": blas_threads(), "kind": "oracle",
                                "sample": "sigma index %d, lambda indices %s x %d hold-out settings = %d of %d columns, "
                                          "full n, Gram + eigh + path + exact CV, %.1f s, %d column-iterations"
                                          % (CPU_SAMPLE_SIGMA_IDX, list(CPU_SAMPLE_LAMBDA_IDX), w.V + 1, ncol,
                                             fits_per_step, secs, its)}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


# ------------------------------------------------------------- secondary workload: Nystrom at the paper's row counts
def run_nystrom_scale(args):
    """`--workload nystrom_covtype | nystrom_mnist8m46` (not the headline line): streamed Nystrom
    setup + sweep + exact CV at the row counts of the paper's Table 4, one GPU, X and y resident.  One JSON line with
    the same metric; `roofline` holds the four contraction-kernel families as sampled inside the sweep."""
    import torch
    import paper_2606_06742_b200 as tkm
    tkm.lib()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device (libtkm has no CPU fallback)")
    torch.cuda.set_device(0)
    w = wl.nystrom_paper_shape(args.workload[len("nystrom_"):])
    sigma = float(w.sigmas[0])
    idx = wl.landmarks(w.n, w.m_landmarks, w.landmark_seed)
    foldid = tkm.tkm_make_folds(w.n, w.V, w.fold_seed)
    X, y = torch.from_numpy(w.X).cuda(), torch.from_numpy(w.y).cuda()
    pk = peaks()

    def ev():
        e = torch.cuda.Event(enable_timing=True)
        e.record()
        return e

    tot = np.zeros(3)
    prof = dict(ms=np.zeros(4), flops=np.zeros(4), launches=np.zeros(4, dtype=np.int64))
    col_iters = 0
    mon = ClockSampler(0)
    for it in range(args.warmup + args.steps):
        if it == args.warmup:
            mon.start()
        e0 = ev()
        spec = tkm.tkm_spectral_setup_nystrom_x(X, sigma, idx)
        e1 = ev()
        path = tkm.tkm_fit_path(spec, y, w.loss, w.lambdas, foldid, w.V, args.tol, MAXIT, smooth0=w.smooth0, eta=w.eta,
                                rounds=w.rounds, warm_tol=WARM_TOL, tf32_delta=2, profile=True)
        e2 = ev()
        tkm.tkm_exact_cv(path, y, foldid, 1, w.L, w.V)
        e3 = ev()
        e3.synchronize()
        if path.status != 0:
            raise RuntimeError("columns hit maxit: the timed work is not the stated work")
        if it >= args.warmup:
            tot += [e0.elapsed_time(e1), e1.elapsed_time(e2), e2.elapsed_time(e3)]
            pr = path.profile()
            for k in prof:
                prof[k] += pr[k]
            col_iters += path.total_col_iters
        r = spec.r
        path.close()
        spec.close()
    clocks = mon.stop()
    tot /= args.steps
    names = ["gemm_f64_tma_kernel GEMM-A (FP64 DMMA)", "gemm_f64_tma_kernel GEMM-B (FP64 DMMA, K-split)",
             "gemm_tf32x3_kernel GEMM-A (tcgen05 3xTF32)", "gemm_tf32x3_kernel GEMM-B (tcgen05 3xTF32, K-split)"]
    f64_tf, tf32x3_tf = pk["bf16_sus"] * NOMINAL_RATIO["f64"], pk["bf16_sus"] * NOMINAL_RATIO["f32"]   # as in run_ours
    peak = [f64_tf, f64_tf, tf32x3_tf, tf32x3_tf]
    fam = [{"kernel": names[i], "bound": "tensor", "achieved": float(prof["flops"][i] / prof["ms"][i] / 1e9), "peak": peak[i],
            "unit": "TFLOP/s", "frac": float(prof["flops"][i] / prof["ms"][i] / 1e9 / peak[i]),
            "sampled_launches": int(prof["launches"][i]), "avg_launch_ms": float(prof["ms"][i] / prof["launches"][i]),
            "traffic": None} for i in range(4) if prof["launches"][i]]
    print(json.dumps({
        "metric": "lambda_x_fold_path_fits_per_s", "value": w.B / (tot.sum() / 1e3), "unit": "fits/s", "n_gpus": 1,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(tot.sum()), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s: Nystrom smoothed-hinge SVM with the shape of the paper's Table-4 data set (synthetic "
                               "rows), n=%d, p=%d, m=%d landmarks (r=%d), %d folds, %d lambdas 1e2..1e-5; secondary "
                               "workload, not BASELINE.json's metric configuration" % (args.workload, w.n, w.p,
                                                                                        w.m_landmarks, r, w.V, w.L),
                   "columns_per_step": w.B, "stop_tol": args.tol, "warm_start_rounds_tol": WARM_TOL, "tf32_delta": 2,
                   "l2": "inputs larger than L2 (U alone is %.1f GB)" % (w.n * r * 8 / 1e9)},
        "stages_ms_per_step": {"nystrom_setup_streamed": float(tot[0]), "sweep": float(tot[1]), "exact_cv": float(tot[2])},
        "col_iters_per_step": col_iters / args.steps,
        "sweep_useful_tflops": 4.0 * w.n * r * col_iters / args.steps / (tot[1] / 1e3) / 1e12,
        "roofline": fam, "clocks": clocks}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--workload", default="config1", choices=["config1", "nystrom_covtype", "nystrom_mnist8m46"],
                    help="config1 = BASELINE.json's metric configuration (the bench line); the nystrom_* workloads are "
                         "secondary single-GPU measurements (use --steps 1 --warmup 1: a step takes 20-100 s)")
    ap.add_argument("--tol", type=float, default=1e-10, help="stop tolerance of the nystrom_* workloads")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.workload != "config1":
        if args.impl != "ours" or world != 1 or args.gpus != 1:
            raise SystemExit("--workload %s: one GPU, --impl ours only" % args.workload)
        return run_nystrom_scale(args)
    from paper_2606_06742_b200.ranks import replica_seed
    w = wl.config1(seed=replica_seed(1001, rank if args.impl == "ours" else 0))
    if args.impl == "reference":
        run_reference(args, w, rank)
    else:
        run_ours(args, w, rank, world)


if __name__ == "__main__":
    main()
