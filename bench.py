#!/usr/bin/env python
"""bench.py -- throughput of the DIA hot path on B200 (contract: see the task prompt / DESIGN.md section 8).

Workload (BASELINE.json configs[4], the one the metric is quoted on): one 4096x4096 float32 reference
(200000 stars) resident on the device, 16 seeded target epochs, 19x19 kernel + B0 per epoch, Gaussian
likelihood with the noise model of Eq. 6 (sigma0 = 5, G = 1).

A "step" is one pass of the whole hot path over the batch: one dia_fit call in lock-step mode
(force_adam_iters = 8, force_lbfgs_iters = 3), i.e. per epoch 8 Adam updates, the switch, 3 L-BFGS
updates -- every one a fused loss+gradient evaluation (stage -> model -> residual -> variance -> loss ->
weights -> kernel gradient -> block partials), the FP64 second-level reduction, the on-device optimiser
step and its convergence bookkeeping, for all 16 epochs inside one CUDA-graph launch.
  metric / value : loss+gradient evaluations per second (one evaluation = one epoch, 4096^2, m = 19),
                   counted from the n_evals the device reports, inputs resident in HBM
  e2e            : the same through dia_fit_host (C ABI; Handle.fit_host marshals) -- pinned host I / theta0 copied in, theta-hat and the
                   result structs copied out, inside the timed region
  roofline       : the fused kernel against the FP32 FMA pipe ("alu"); its launch duration is measured with
                   CUDA events around back-to-back dia_eval_loss_grad launches of the same batch
  cpu_baseline   : the FP64 oracle (oracle/) on the host cores, one evaluation of epoch 0 (rank 0, N = 1)
  fits           : one free-running fit of the batch with the paper's settings (fits/s, iteration counts)

python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--no-fit]
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

CONFIG_INDEX = 4
N, M, E_PER_GPU = 4096, 19, 16
STEP_ADAM, STEP_LBFGS = 8, 3
METRIC = "loss+grad evaluations per second (4096^2 image, 19x19 kernel + B0, per epoch)"
UNIT = "evals/s"
SM_COUNT, FP32_LANES_PER_SM = 148, 128          # B200 (B200_PROFILING.md: 148 SMs; 128 FP32 lanes per SM)
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "dram_traffic.csv")


def measured_traffic(kernel: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel` over the 16-epoch batch, from the last
    matching row of profiles/dram_traffic.csv (one row per committed `ncu --set full` capture: kernel, capture file,
    commit, bytes read, bytes written); None when no capture is recorded."""
    try:
        import csv
        rows = list(csv.reader(l for l in open(TRAFFIC_CSV) if l.strip() and not l.startswith("#")))
        rows = [r for r in rows[1:] if r[0] == kernel]
        return (float(rows[-1][3]) + float(rows[-1][4]), rows[-1][1], rows[-1][2]) if rows else (None, None, None)
    except Exception:
        return None, None, None


def useful_fma(n=N, m=M, epochs=1):
    """2 m^2 FMA per valid pixel: m^2 forward + m^2 gradient."""
    return 2.0 * m * m * (n - m + 1) ** 2 * epochs


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons while the timed region runs."""

    def __init__(self, index=0):
        self.index, self.rows, self.proc = index, [], None

    def __enter__(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
            except Exception:
                continue
            for k, nm in enumerate(names):
                if len(r) > 3 + k and r[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        sm_busy = [x for x in sm if x > 0.6 * mx] or sm
        return {"sm_mhz": float(np.median(sm_busy)) if sm_busy else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


# --------------------------------------------------------------------------------------------------
# workload
# --------------------------------------------------------------------------------------------------
def build_workload(first_epoch: int, n_epochs: int, n: int = N, m: int = M):
    """Reference of config 4 and target epochs [first_epoch, first_epoch + n_epochs) (seeded per epoch)."""
    from workloads import CONFIGS, make_reference, make_target, theta_init
    cfg = CONFIGS[CONFIG_INDEX]
    R = make_reference(cfg, n)
    I = np.empty((n_epochs, n, n), np.float32)
    th0 = np.empty((n_epochs, m * m + 1), np.float32)
    global TRUE_WIDTHS                      # sigma of each planted kernel (second moment), for the Gaussian-init series
    TRUE_WIDTHS = []
    h = (m - 1) // 2
    r2 = (np.arange(m)[:, None] - h) ** 2 + (np.arange(m)[None, :] - h) ** 2
    for e in range(n_epochs):
        I[e], th_true, _, _ = make_target(cfg, first_epoch + e, R, m)
        th0[e] = theta_init(R, I[e], m)
        K = np.asarray(th_true[:m * m], np.float64).reshape(m, m)
        TRUE_WIDTHS.append(float(np.sqrt((K * r2).sum() / (2.0 * K.sum()))))
    return cfg, R, I, th0


TRUE_WIDTHS = []


def oracle_fit_and_b08_times():
    """the oracle's own fit (dia_ref_fit, paper settings) and the classical B08 normal-equation solve
    (3 iterations) timed on the host cores, on the configs they finish in seconds (c0, c1)."""
    import oracle
    from workloads import make_workload
    out = {}
    for c in (0, 1):
        w = make_workload(c)
        rc = oracle.RefConfig(w.n, w.n, w.m, sigma0=w.sigma0, gain=w.gain)
        t0 = time.perf_counter()
        th_b = oracle.b08_solve(rc, w.R, w.I[0], n_iters=3)
        t_b08 = time.perf_counter() - t0
        entry = {"n": w.n, "m": w.m, "b08_solve_3_iterations_s": t_b08, "b08_photometric_scale": float(th_b[:-1].sum())}
        if c == 0:
            t0 = time.perf_counter()
            _, res = oracle.fit(rc, w.R, w.I, w.theta0, oracle.RefFitOpts.default())
            entry.update({"oracle_fit_s": time.perf_counter() - t0, "oracle_fit_evals": int(res[0].n_evals)})
        out[f"c{c}"] = entry
    return {"classical_and_fit": out}


def oracle_eval_rate(cfg, R, I0, th0, crop: int, repeats: int = 1):
    """Times the FP64 oracle (as it stands) on a crop x crop corner of one epoch; returns
    (full-size-equivalent evaluations per second, seconds per call, threads used)."""
    import oracle
    Rc, Ic = np.ascontiguousarray(R[:crop, :crop]), np.ascontiguousarray(I0[:crop, :crop])
    rc = oracle.RefConfig(crop, crop, M, sigma0=cfg.sigma0, gain=cfg.gain)
    best = float("inf")
    for _ in range(repeats):
        t0 = time.perf_counter()
        oracle.eval_loss_grad(rc, Rc, Ic, th0)
        best = min(best, time.perf_counter() - t0)
    frac = (crop - M + 1) ** 2 / float((N - M + 1) ** 2)
    return frac / best, best, oracle.num_threads()


def oracle_single_thread_rate():
    """the oracle timed single-threaded beside the OpenMP figure.  The thread count of the oracle is
    fixed when its library loads, so this runs `bench.py --impl reference` once more in a child process with
    OMP_NUM_THREADS=1 (two steps of a 1024^2 evaluation, scaled to full-size evaluations per second)."""
    try:
        env = dict(os.environ, OMP_NUM_THREADS="1", RANK="0", WORLD_SIZE="1")
        out = subprocess.run([sys.executable, os.path.abspath(__file__), "--impl", "reference", "--steps", "2", "--warmup", "1"],
                             env=env, capture_output=True, text=True, timeout=600)
        d = json.loads(out.stdout.strip().splitlines()[-1])
        return {"value": d["value"], "unit": UNIT, "cores": d["cpu_baseline"]["cores"], "sample": d["cpu_baseline"]["sample"]}
    except Exception as exc:      # noqa: BLE001 -- a reported baseline, never fatal
        return {"error": repr(exc)}


def stamp_batch_rate(dia, dev, n_stamps=296, n=142, m=19):
    """Throughput of the one-reference-per-epoch mode on synthetic stamps of the paper's stamp shape
    (142^2 images, 19x19 kernel): batched evaluations and a lock-step fit."""
    import torch
    from workloads import CONFIGS, make_reference, make_target, theta_init
    cfg = CONFIGS[2]
    big = make_reference(cfg, 1024)                        # crowded field; stamps are crops of it
    rng = np.random.default_rng(7)
    R = np.empty((n_stamps, n, n), np.float32); I = np.empty_like(R); th0 = np.empty((n_stamps, m * m + 1), np.float32)
    for k in range(n_stamps):
        y, x = rng.integers(0, 1024 - n, 2)
        R[k] = big[y:y + n, x:x + n]
        I[k], _, _, _ = make_target(CONFIGS[0], 1000 + k, R[k], m)
        th0[k] = theta_init(R[k], I[k], m)
    dR, dI, dth = (torch.from_numpy(a).to(dev) for a in (R, I, th0))
    h = dia.Handle(dR, m, max_epochs=n_stamps, sigma0=CONFIGS[0].sigma0, gain=CONFIGS[0].gain)
    loss = torch.empty(n_stamps, dtype=torch.float64, device=dev)
    grad = torch.empty((n_stamps, m * m + 1), dtype=torch.float64, device=dev)
    for _ in range(3):
        h.eval_loss_grad(dI, dth, loss=loss, grad=grad)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    a.record()
    for _ in range(20):
        h.eval_loss_grad(dI, dth, loss=loss, grad=grad)
    b.record()
    torch.cuda.synchronize()
    ms_eval = a.elapsed_time(b) / 20
    opts = dia.FitOpts.default(force_adam_iters=100, force_lbfgs_iters=20)
    h.fit(dI, dth, opts)
    torch.cuda.synchronize()
    a.record()
    _, res = h.fit(dI, dth, opts)
    b.record()
    torch.cuda.synchronize()
    ms_fit = a.elapsed_time(b)
    h.close()
    fma = useful_fma(n, m, n_stamps)
    return {"n_stamps": n_stamps, "n": n, "m": m, "evals_per_s": n_stamps / (ms_eval * 1e-3),
            "ms_per_batched_eval": ms_eval, "tflops_useful": 2.0 * fma / (ms_eval * 1e-3) / 1e12,
            "lockstep_fit": {"iterations": res[0].n_evals, "ms": ms_fit,
                             "stamp_iterations_per_s": n_stamps * res[0].n_evals / (ms_fit * 1e-3)},
            "note": "one reference per epoch (dia_config.n_refs == max_epochs), one launch sequence for the batch"}


def other_configs(dia, dev):
    """BASELINE configs[0..3] (parity-test shapes): evaluations/s of a stand-alone dia_eval_loss_grad and one
    free-running fit with the paper's settings, for context beside the headline workload."""
    import torch
    from workloads import make_workload
    out = []
    for c in (0, 1, 2, 3):
        w = make_workload(c)
        to = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        loss_kind = dia.LOSS_HUBER if w.loss == "huber" else dia.LOSS_GAUSSIAN
        h = dia.Handle(to(w.R), w.m, max_epochs=1, loss=loss_kind, sigma0=w.sigma0, gain=w.gain, flat=to(w.flat))
        I, th0, mk = to(w.I), to(w.theta0), to(w.mask)
        L = torch.empty(1, dtype=torch.float64, device=dev)
        G = torch.empty((1, w.m * w.m + 1), dtype=torch.float64, device=dev)
        for _ in range(5):
            h.eval_loss_grad(I, th0, mask=mk, loss=L, grad=G)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        a.record()
        for _ in range(50):
            h.eval_loss_grad(I, th0, mask=mk, loss=L, grad=G)
        b.record()
        torch.cuda.synchronize()
        ms_eval = a.elapsed_time(b) / 50
        opts = dia.FitOpts.default()
        h.fit(I, th0, opts, mask=mk)
        torch.cuda.synchronize()
        a.record()
        _, res = h.fit(I, th0, opts, mask=mk)
        b.record()
        torch.cuda.synchronize()
        ms_fit = a.elapsed_time(b)
        h.close()
        out.append({"config": c, "n": w.n, "m": w.m, "loss": w.loss, "evals_per_s": 1e3 / ms_eval,
                    "us_per_eval": 1e3 * ms_eval, "frac_fp32_nominal": 2.0 * useful_fma(w.n, w.m) / (ms_eval * 1e-3) / 1e12 /
                    (SM_COUNT * FP32_LANES_PER_SM * 2 * 1.965e9 / 1e12),
                    "fits_per_s": 1e3 / ms_fit, "ms_per_fit": ms_fit, "lr_b0": float(opts.lr_b0),
                    "adam_met_switch_rule": bool(res[0].n_adam < opts.max_adam_iters),
                    "n_adam": res[0].n_adam, "n_lbfgs": res[0].n_lbfgs,
                    "status": res[0].status, "photometric_scale": round(res[0].photometric_scale, 5)})
    return out


def sweeps(dia, dev):
    """--sweep: the shapes of the paper's speed tests (Fig. 8: image size at m = 19 and 25, PAPER.md:604, 620;
    Fig. 9: kernel size on a 1024^2 crop) on crops of the c4 pair; stand-alone single-epoch
    dia_eval_loss_grad.  GB/s counts the algorithmic bytes 4 n^2 (1 + E) (R once, every I once)."""
    import torch
    from workloads import make_workload
    w = make_workload(4, n_epochs=1)
    peak = SM_COUNT * FP32_LANES_PER_SM * 2 * 1.965e9 / 1e12
    hbm_peak = float(measured_peaks().get("hbm_gbs") or 6650.0)   # MEASURED_PEAKS.json, else B200_PROFILING.md's fallback
    cases = [(n, m, 1) for m in (19, 25) for n in (512, 1024, 2048, 4096)]
    cases += [(1024, m, 1) for m in (1, 3, 5, 7, 11, 15, 23, 31, 39, 47)] + [(4096, 47, 1)]
    # small kernels on a batch larger than L2 (16 copies of the target: 1 GiB): the HBM-side regime of SURVEY.md 8(d)
    cases += [(4096, m, 16) for m in (1, 3, 5, 7)]
    out = []
    for n, m, E in cases:
        R = torch.from_numpy(np.ascontiguousarray(w.R[:n, :n])).to(dev)
        I = torch.from_numpy(np.ascontiguousarray(w.I[:, :n, :n])).to(dev).repeat(E, 1, 1).contiguous()
        th = torch.full((E, m * m + 1), 1.0 / (m * m), dtype=torch.float32, device=dev)
        th[:, -1] = 0.0
        h = dia.Handle(R, m, max_epochs=E, sigma0=w.sigma0, gain=w.gain)
        L = torch.empty(E, dtype=torch.float64, device=dev)
        G = torch.empty((E, m * m + 1), dtype=torch.float64, device=dev)
        for _ in range(5):
            h.eval_loss_grad(I, th, loss=L, grad=G)
        ms = float("inf")
        for _ in range(3):           # best of three series: at 10-20 us per call host launch jitter shows
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            a.record()
            for _ in range(50):
                h.eval_loss_grad(I, th, loss=L, grad=G)
            b.record()
            torch.cuda.synchronize()
            ms = min(ms, a.elapsed_time(b) / 50)
        h.close()
        out.append({"n": n, "m": m, "epochs": E, "us_per_eval": round(1e3 * ms / E, 2), "evals_per_s": round(1e3 * E / ms, 1),
                    "tflops": round(2.0 * useful_fma(n, m, E) / (ms * 1e-3) / 1e12, 3),
                    "frac_fp32_nominal": round(2.0 * useful_fma(n, m, E) / (ms * 1e-3) / 1e12 / peak, 4),
                    "algorithmic_GBps": round(4.0 * n * n * (1 + E) / (ms * 1e-3) / 1e9, 1),
                    "frac_hbm_measured": round(4.0 * n * n * (1 + E) / (ms * 1e-3) / 1e9 / hbm_peak, 4)})
    return out


def run_sweep(args):
    import torch
    if not torch.cuda.is_available():
        print("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle", file=sys.stderr)
        return 2
    import paper_2104_13715_b200 as dia
    dia.load_library()
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    with ClockSampler(dev.index or 0) as clocks:
        rows = sweeps(dia, dev)
    print(json.dumps({"sweep": rows, "clocks": clocks.summary(), "data": "synthetic (crops of the c4 pair)",
                      "note": "L2-resident for n <= 2048 (the pair fits the 126 MB L2): repeated evaluations of one pair, as in a fit"}),
          flush=True)
    return 0


def run_reference(args):
    """--impl reference: the CPU oracle on the host cores, rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    crop = 1024
    cfg, R, I, th0 = build_workload(0, 1, n=crop)      # same recipe and stellar density at the sample size
    import oracle
    rc = oracle.RefConfig(crop, crop, M, sigma0=cfg.sigma0, gain=cfg.gain)
    frac = (crop - M + 1) ** 2 / float((N - M + 1) ** 2)
    for _ in range(args.warmup):
        oracle.eval_loss_grad(rc, R, I[0], th0[0])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.eval_loss_grad(rc, R, I[0], th0[0])
    dt = time.perf_counter() - t0
    value = args.steps * frac / dt
    sample = (f"each step = one FP64 oracle loss+gradient evaluation of a {crop}x{crop} field of the config-4 recipe "
              f"({frac:.4f} of the 4096^2 valid pixels); value scaled to full-size evaluations per second")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE configs[4]: 4096^2 reference, 19x19 kernel + B0, Gaussian likelihood",
                       "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# --------------------------------------------------------------------------------------------------
# GPU arm
# --------------------------------------------------------------------------------------------------
def run_gpu(args):
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the engine has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    import paper_2104_13715_b200 as dia
    from paper_2104_13715_b200.sharding import epoch_shard, max_over_ranks

    # weak scaling: every rank owns E_PER_GPU epochs of a (world * E_PER_GPU)-epoch batch; R is replicated
    first, last = epoch_shard(E_PER_GPU * world, world, rank)
    E = last - first
    cfg, R, I, th0 = build_workload(first, E)
    hI = torch.from_numpy(I).pin_memory()
    hth0 = torch.from_numpy(th0).pin_memory()
    dR = torch.from_numpy(R).to(dev)
    dI = hI.to(dev)
    dth0 = hth0.to(dev)
    h = dia.Handle(dR, M, max_epochs=E, loss=dia.LOSS_GAUSSIAN, noise=dia.NOISE_MODEL, sigma0=cfg.sigma0,
                   gain=cfg.gain)
    step_opts = dia.FitOpts.default(force_adam_iters=STEP_ADAM, force_lbfgs_iters=STEP_LBFGS)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        a.record()
        out = None
        for _ in range(steps):
            out = fn()
        b.record()
        barrier()
        ms = a.elapsed_time(b)
        if world > 1:
            ms = max_over_ranks(ms, device=dev)
        return ms, out

    # ---- device-resident steps (value)
    for _ in range(args.warmup):
        h.fit(dI, dth0, step_opts)
    with ClockSampler(local_rank) as clocks:
        ms, (_, res) = timed(lambda: h.fit(dI, dth0, step_opts), args.steps)
    evals_per_step_rank = sum(r.n_evals for r in res)
    iters = max(r.n_evals for r in res)
    total_evals = evals_per_step_rank * world          # every rank runs the same lock-step counts
    value = total_evals * args.steps / (ms * 1e-3)
    lpe = h.info()["launches_per_eval"]                # (pack_const,) eval_kernel, fit_step_kernel per iteration
    launches = args.steps * (1 + lpe * iters)          # + fit_init_kernel once per fit

    # ---- end to end through host buffers
    for _ in range(max(1, args.warmup // 2)):
        h.fit_host(hI, hth0, step_opts)
    ms_e2e, (_, res_e, h2d, d2h) = timed(lambda: h.fit_host(hI, hth0, step_opts), args.steps)
    e2e_value = sum(r.n_evals for r in res_e) * world * args.steps / (ms_e2e * 1e-3)

    # ---- the dominant kernel alone: back-to-back batched evaluations (eval_kernel + the small reduce kernel)
    loss = torch.empty(E, dtype=torch.float64, device=dev)
    grad = torch.empty((E, M * M + 1), dtype=torch.float64, device=dev)
    n_eval_launch, n_series = 50, 5            # back-to-back launches between two events, median of 5 series
    for _ in range(3):
        h.eval_loss_grad(dI, dth0, loss=loss, grad=grad)
    series = sorted(timed(lambda: h.eval_loss_grad(dI, dth0, loss=loss, grad=grad), n_eval_launch)[0] / n_eval_launch
                    for _ in range(n_series))
    ms_kernel = series[n_series // 2]
    flop_per_launch = 2.0 * useful_fma(epochs=E)
    achieved_tflops = flop_per_launch / (ms_kernel * 1e-3) / 1e12
    info = h.info()

    line = None
    if rank == 0:
        peaks = measured_peaks()
        sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))
        nominal_tflops = SM_COUNT * FP32_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
        measured_fma = dia.dia_measure_fp32_peak()
        patterns = {name: 2.0 * dia.dia_measure_fp32_pattern(k) / 1e12 for k, name in
                    enumerate(("pipe_peak_one_vector_register", "forward_ffma2_uniform_multiplicand",
                               "gradient_ffma2_vector_operands", "scalar_ffma_three_vector_registers"))}
        kernel_name = f"dia::eval_kernel<{M}, false, false, true>"
        traffic, traffic_file, traffic_commit = measured_traffic(kernel_name)
        roof = {"bound": "alu", "achieved": achieved_tflops, "peak": nominal_tflops, "unit": "TFLOP/s",
                "frac": achieved_tflops / nominal_tflops, "traffic": traffic,
                "traffic_source": f"profiles/dram_traffic.csv: {traffic_file} at commit {traffic_commit}",
                "ms_per_launch_series": series, "pattern_peaks_tflops": patterns,
                "peak_kind": f"nominal FP32 FMA pipe: {SM_COUNT} SMs x {FP32_LANES_PER_SM} lanes x 2 FLOP x "
                             f"{sm_max_mhz:.0f} MHz (DESIGN.md section 8)",
                "peak_measured": 2.0 * measured_fma / 1e12,
                "frac_of_measured": achieved_tflops / (2.0 * measured_fma / 1e12),
                "peak_measured_kind": "register-only FFMA microbenchmark run in this process (dia_measure_fp32_peak: FFMAs "
                                      "reading one vector register; the kernel's own operand patterns are in pattern_peaks_tflops)",
                "kernel": kernel_name, "ms_per_launch": ms_kernel,
                "flop_per_launch": flop_per_launch,
                "how": f"CUDA events around {n_eval_launch} back-to-back dia_eval_loss_grad launches of the "
                       f"{E}-epoch batch (pack_const + eval_kernel + reduce_partials_kernel), median of {n_series} series, "
                       f"useful FLOP = 4 m^2 per valid pixel",
                "hbm_gbs_algorithmic": (4.0 * N * N * (1 + E)) / (ms_kernel * 1e-3) / 1e9,
                "hbm_peak_gbs_measured": peaks.get("hbm_gbs")}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "BASELINE configs[4]: 4096^2 reference resident on device, 16 target epochs "
                                       "per GPU, 19x19 kernel + B0 per epoch, Gaussian likelihood, Eq. 6 noise "
                                       "(sigma0=5, G=1)",
                           "n": N, "m": M, "epochs_per_gpu": E, "global_epochs": E * world,
                           "step": f"one dia_fit call in lock-step mode: {STEP_ADAM} Adam + {STEP_LBFGS} L-BFGS "
                                   f"iterations = {iters} fused loss+gradient evaluations per epoch",
                           "parallelism": f"epochs sharded over {world} GPU(s), reference replicated, no collective",
                           "l2": "inputs (1 GiB of targets per GPU per evaluation) are larger than the 126 MB L2",
                           "grid_blocks": info["grid_blocks"], "smem_bytes": info["smem_bytes"]},
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                        "ms_per_step": ms_e2e / args.steps},
                "gpu_launches": launches, "clocks": clocks.summary(), "roofline": roof}

    # ---- one free-running fit of the batch with the paper's settings (fits/s)
    if not args.no_fit:
        fit_opts = dia.FitOpts.default()
        ms_fit, (th_hat, res_f) = timed(lambda: h.fit(dI, dth0, fit_opts), 1)
        if rank == 0:
            line["fits"] = {"value": E * world / (ms_fit * 1e-3), "unit": "fits/s", "ms_per_batch": ms_fit,
                            "epochs": E * world, "settings": "paper defaults: Adam lr 1e-3 / 10, switch 1e-6, L-BFGS "
                                                             "lr 1 history 100, stop 1e-8 (PAPER.md:242-244)",
                            "n_adam": [r.n_adam for r in res_f], "n_lbfgs": [r.n_lbfgs for r in res_f],
                            "n_evals": [r.n_evals for r in res_f], "status": [r.status for r in res_f],
                            "photometric_scale": [round(r.photometric_scale, 5) for r in res_f]}
        # second series (the paper's other panel): Gaussian initial kernel of the true width
        from workloads import gaussian_kernel_init
        thg = np.stack([gaussian_kernel_init(M, TRUE_WIDTHS[e], float(th0[e][-1])) for e in range(E)])
        dthg = torch.from_numpy(thg).to(dev)
        ms_fit_g, (_, res_g) = timed(lambda: h.fit(dI, dthg, fit_opts), 1)
        if rank == 0:
            line["fits"]["gaussian_init"] = {"value": E * world / (ms_fit_g * 1e-3), "unit": "fits/s", "ms_per_batch": ms_fit_g,
                                             "init": "symmetric Gaussian of each epoch's planted width, sum 1; B0 as in the "
                                                     "flat-kernel series",
                                             "n_adam": [r.n_adam for r in res_g], "n_lbfgs": [r.n_lbfgs for r in res_g],
                                             "n_evals": [r.n_evals for r in res_g], "status": [r.status for r in res_g],
                                             "photometric_scale": [round(r.photometric_scale, 5) for r in res_g]}
        # Hessian at the fitted theta of epoch 0 (Eq. 15): np rows, max_epochs rows per launch
        h.hessian(dI[0], th_hat[0])
        ms_h, H_hat = timed(lambda: h.hessian(dI[0], th_hat[0]), 1)
        # covariance and uncertainties from it (Eq. 16-17): FP64 Cholesky factorisation and solves on the device
        h.covariance(H_hat)
        ms_c, (_, sig_hat, cov_info) = timed(lambda: h.covariance(H_hat), 1)
        if rank == 0:
            rows = M * M + 1
            ci = cov_info.cpu().tolist()
            # dia_hessian is one tensor-core contraction X' diag(h) X over the valid pixels (hess_tc_kernel):
            # "useful" counts the dense np x np x pixels product once (2 flops per multiply-add); the kernel computes the
            # upper block triangle of the 128-padded matrix in four split-float16 terms
            n_valid = (N - M + 1) ** 2
            g_ = -(-rows // 128)
            executed = 2.0 * 4 * (g_ * (g_ + 1) // 2) * 128 * 128 * n_valid        # four split terms, upper block triangle
            tensor_peak = float(peaks.get("bf16_tflops") or 2250.0)                 # fp16 = bf16 rate (nominal ratio 1); burst figure
            line["fits"]["hessian"] = {"ms": ms_h, "rows": rows, "launches": 3,
                                       "useful_tflops": 2.0 * rows * rows * n_valid / (ms_h * 1e-3) / 1e12,
                                       "roofline": {"bound": "tensor", "achieved": executed / (ms_h * 1e-3) / 1e12, "peak": tensor_peak,
                                                    "unit": "TFLOP/s", "frac": executed / (ms_h * 1e-3) / 1e12 / tensor_peak,
                                                    "traffic": 139.1e6,
                                                    "note": "executed float16 MMA work of hess_tc_kernel (4 terms x 6 blocks of 128 x 128 per "
                                                            "valid pixel) over the whole dia_hessian call, against MEASURED_PEAKS.json's "
                                                            "cuBLAS bf16 burst figure (else the nominal 2250); traffic: dram bytes of the "
                                                            "ncu capture in profiles/r02_tc_hessian.md"},
                                       "path": "tcgen05 kind::f16, float16 hi/lo split (4 terms), FP32 in TMEM per tile row, "
                                               "FP64 per tile",
                                       "work_model": "2 np^2 flops per valid pixel"}
            line["fits"]["covariance"] = {"ms": ms_c, "np": rows, "launches": 2 * (-(-rows // 32)) + 3, "valid": ci[0],
                                          "sigma_P": ci[2], "sigma_B0": float(sig_hat[M * M])}

    # ---- small kernels on the same resident batch: the HBM side of the roofline
    if rank == 0 and not args.no_stamps:
        hbm_peak = float(peaks.get("hbm_gbs") or 6650.0)
        line["small_kernels"] = []
        for ms_ in (1, 3, 5):
            hs = dia.Handle(dR, ms_, max_epochs=E, sigma0=cfg.sigma0, gain=cfg.gain)
            ths = torch.full((E, ms_ * ms_ + 1), 1.0 / (ms_ * ms_), dtype=torch.float32, device=dev)
            ths[:, -1] = 0.0
            Ls = torch.empty(E, dtype=torch.float64, device=dev)
            Gs = torch.empty((E, ms_ * ms_ + 1), dtype=torch.float64, device=dev)
            for _ in range(3):
                hs.eval_loss_grad(dI, ths, loss=Ls, grad=Gs)
            ev_a, ev_b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)   # rank 0 only:
            torch.cuda.synchronize()                                                                  # no barrier here
            ev_a.record()
            for _ in range(20):
                hs.eval_loss_grad(dI, ths, loss=Ls, grad=Gs)
            ev_b.record()
            torch.cuda.synchronize()
            ms_s = ev_a.elapsed_time(ev_b)
            hs.close()
            gbs = 4.0 * N * N * (1 + E) / (ms_s / 20 * 1e-3) / 1e9
            tfl = 4.0 * ms_ * ms_ * (N - ms_ + 1) ** 2 * E / (ms_s / 20 * 1e-3) / 1e12
            # m = 5 sits between the roofs (100 FLOP per 8 bytes): both fractions are given, the larger one binds
            fh = gbs / hbm_peak
            ff = tfl / (SM_COUNT * FP32_LANES_PER_SM * 2 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12)
            line["small_kernels"].append({"m": ms_, "epochs": E, "us_per_epoch": 1e3 * ms_s / 20 / E,
                                          "evals_per_s": E * 20 / (ms_s * 1e-3), "bound": "hbm" if fh >= ff else "alu",
                                          "algorithmic_GBps": gbs, "hbm_peak_gbs": hbm_peak, "frac": max(fh, ff),
                                          "frac_hbm": fh, "tflops_useful": tfl, "frac_fp32_nominal": ff,
                                          "kernel": f"dia::eval_small_kernel<{ms_}, false>"})

    # ---- many small image pairs, one reference each (the paper's stamp workloads)
    if rank == 0 and not args.no_stamps:
        line["stamps"] = stamp_batch_rate(dia, dev)
        line["stamps_m27"] = stamp_batch_rate(dia, dev, m=27)     # median kernel size of the paper's real-data fits
        line["other_configs"] = other_configs(dia, dev)

    # ---- the oracle beside it (rank 0, N = 1 only)
    if rank == 0 and world == 1 and not args.no_cpu:
        crop = N                                   # one whole epoch: ~40 core-seconds of FP64 work
        v, sec, cores = oracle_eval_rate(cfg, R, I[0], th0[0], crop, repeats=3)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"FP64 oracle loss+gradient evaluation of epoch 0 at the full {crop}x{crop} size, "
                                          f"best of 3 calls ({sec:.2f} s per call, OpenMP over all host cores)"}
        line["cpu_baseline"]["host_cores_available"] = len(os.sched_getaffinity(0))
        line["cpu_baseline"]["single_thread"] = oracle_single_thread_rate()
        line["cpu_baseline"].update(oracle_fit_and_b08_times())
    h.close()
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-fit", action="store_true", help="skip the free-running fit (fits/s)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the oracle cpu_baseline leg")
    ap.add_argument("--no-stamps", action="store_true", help="skip the many-small-pairs leg")
    ap.add_argument("--sweep", action="store_true", help="image-size and kernel-size sweeps (the paper's Fig. 8-9 shapes) only")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
