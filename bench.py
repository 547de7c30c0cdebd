#!/usr/bin/env python
"""bench.py -- one JSON line for the driver.

Workload: BASELINE.json configs[3], 32^3x64 (2.1M sites), eps=0.8 warm links, kappa=0.1248,
csw=1.8, Gaussian source.  One STEP is one pass of the whole hot path
in fp64 with 18-real links:
    gauge pack -> clover build + inverse -> source pack -> prepare -> even-odd CGNE to 1e-10
    (dslash with fused clover epilogues + fused BLAS-1) -> reconstruct -> true residual -> unpack.
value  = algorithmic HBM bytes of every kernel of the step / step time (GB/s), whole job.
roofline = the dominant kernel (dslash with fused clover epilogue), timed per launch with CUDA
events on the launching stream inside the timed region.
Also reported (extra keys): the standalone dslash sweep (fp32/fp64 x 18/12 reals) that the
headline target is stated on, and the solve's iterations / seconds / residuals.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
N > 1: one replica per GPU under torchrun ("replicas only": the path has no exchange step).
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

WORKLOAD = 4  # BASELINE.json configs[3] (1-based numbering in synth.CONFIGS)
METRIC = "Wilson-clover dslash GB/s (whole even-odd CGNE solve, algorithmic bytes / time)"
MATPC = 2  # symmetric even-odd preconditioning from the right (reading A10): 32 CGNE iterations at configs[3]
           # (asymmetric: 54) and the recurrence residual is the even half of the true residual
FLOPS_PER_SITE = 1320.0


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(mx)) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def dslash_alg_bytes(recon, prec, Vh):
    return (8 * recon + 48) * prec * Vh


# ------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands, on the host cores, bounded sample
# ------------------------------------------------------------------------------------------------
def oracle_sample(steps, warmup):
    """Each step = one full-lattice hopping-term application (two parity sweeps) at the workload's
    size in fp64 by the CPU oracle.  Returns (GB/s with the dslash algorithmic bytes, ms/step)."""
    import oracle
    from paper_2411_08461_b200 import synth
    cfg = synth.CONFIGS[WORKLOAD]
    dims = cfg["dims"]
    U = synth.gauge(dims, cfg["eps"], cfg["seed"])
    psi = synth.source(dims, "gaussian", cfg["src_seed"])
    orc = oracle.Oracle(dims, U, -1)
    del U
    for _ in range(warmup):
        orc.dslash(psi)
    t0 = time.perf_counter()
    for _ in range(steps):
        orc.dslash(psi)
    dt = (time.perf_counter() - t0) / steps
    Vh = int(np.prod(dims)) // 2
    gbs = 2 * dslash_alg_bytes(18, 8, Vh) / dt / 1e9
    return gbs, dt * 1e3, oracle.threads()


def oracle_legs(config, n_apply, iters):
    """The oracle as it stands on the host cores (SURVEY.md §8(d) "CPU baseline"; invert is where the
    time goes): clover build, hopping term, clover apply and the even-odd CGNE solve (asymmetric Schur complement,
    the oracle's own) at BASELINE config `config`.  The solve is timed for iters[0] and iters[1] iterations; the
    difference gives seconds per iteration (prepare, reconstruction and true residual cancel)."""
    import oracle
    from paper_2411_08461_b200 import synth
    cfg = synth.CONFIGS[config]
    dims = cfg["dims"]
    U = synth.gauge(dims, cfg["eps"], cfg["seed"])
    psi = synth.source(dims, "gaussian", cfg["src_seed"])
    orc = oracle.Oracle(dims, U, -1)
    del U
    t0 = time.perf_counter()
    orc.set_clover(cfg["kappa"], cfg["csw"])
    t_build = time.perf_counter() - t0
    orc.dslash(psi)
    t0 = time.perf_counter()
    for _ in range(n_apply):
        orc.dslash(psi)
    t_d = (time.perf_counter() - t0) / n_apply
    t0 = time.perf_counter()
    for _ in range(n_apply):
        orc.clover_apply(psi)
    t_c = (time.perf_counter() - t0) / n_apply
    ts = []
    for n in iters:
        t0 = time.perf_counter()
        orc.invert(psi, 1e-10, n, "cgne", 0)
        ts.append(time.perf_counter() - t0)
    V = int(np.prod(dims))
    per_it = (ts[1] - ts[0]) / (iters[1] - iters[0])
    return {"config": config, "dims": list(dims), "threads": oracle.threads(),
            "clover_build_s": t_build,
            "dslash_full_lattice_ms": t_d * 1e3, "dslash_GBps": 2 * dslash_alg_bytes(18, 8, V // 2) / t_d / 1e9,
            "clover_apply_full_lattice_ms": t_c * 1e3, "clover_apply_GBps": 120 * 8 * V / t_c / 1e9,
            "cgne_seconds_per_iteration": per_it, "cgne_timed_iterations": list(iters),
            "cgne_fixed_seconds": ts[0] - iters[0] * per_it}


def oracle_leg_subprocess(config, n_apply, iters, threads=None):
    """oracle_legs in a child process (OMP_NUM_THREADS must be set before the oracle library loads)."""
    env = dict(os.environ)
    if threads is not None:
        env["OMP_NUM_THREADS"] = str(threads)
    cmd = [sys.executable, os.path.abspath(__file__), "--impl", "cpu-leg", "--cpu-leg",
           "%d,%d,%d,%d" % (config, n_apply, iters[0], iters[1])]
    out = subprocess.run(cmd, env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True, timeout=900)
    for ln in reversed(out.stdout.strip().splitlines()):
        if ln.startswith("{"):
            return json.loads(ln)
    return {"error": (out.stderr or out.stdout)[-300:]}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    gbs, ms, cores = oracle_sample(max(1, args.steps), min(args.warmup, 1))
    sample = "per step: one full-lattice fp64 hopping-term application (2 parity sweeps) at 32^3x64 by the CPU oracle"
    line = {
        "impl": "reference", "metric": METRIC, "value": gbs, "unit": "GB/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[3]: 32^3x64, eps=0.8 links seed 4, Gaussian source seed 104",
                   "sample": sample},
        "cpu_baseline": {"value": gbs, "unit": "GB/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": gbs, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------
# GPU arm
# ------------------------------------------------------------------------------------------------
def time_batched(torch, fn, n=20, reps=7, warm=6):
    """Median over `reps` of (device time of n back-to-back asynchronous launches) / n, CUDA events on the launching
    stream.  The host runs ahead of the device, so no launch gap is inside the interval (an event pair around ONE
    launch issued from Python contains 10-30 us of host latency: 10 % of a 140 us kernel)."""
    for i in range(warm):
        fn(i)
    torch.cuda.synchronize()
    ts = []
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(n):
            fn(i)
        e1.record()
        e1.synchronize()
        ts.append(e0.elapsed_time(e1) * 1e-3 / n)
    return float(np.median(ts))


def dslash_sweep(torch, lqcd, U, psi, dims, device, peak):
    """Standalone dslash (bare hopping term, scale 1) at the workload size for the four
    (precision, reconstruction) variants.  Inputs (links 0.4-1.2 GB) exceed L2 (126 MB)."""
    out = {}
    for prec, recon in ((4, 18), (4, 12), (8, 18), (8, 12)):
        ctx = lqcd.Context(dims, prec, recon, -1, device)
        g = ctx.gauge_pack(ctx.to_device(U))
        nat = ctx.spinor_pack(ctx.to_device(psi))
        dst = ctx.new_spinor(2)
        t = time_batched(torch, lambda i: ctx.dslash(ctx.parity(dst, i & 1), ctx.parity(nat, 1 - (i & 1)), g, i & 1))
        by = dslash_alg_bytes(recon, prec, ctx.Vh)
        out["fp%d_recon%d" % (8 * prec, recon)] = {
            "us": t * 1e6, "GBps": by / t / 1e9, "frac_of_measured_peak": by / t / 1e9 / peak,
            "frac_of_8TBps": by / t / 8e12, "GFLOPs": FLOPS_PER_SITE * ctx.Vh / t / 1e9,
            "bytes_per_site": by // ctx.Vh}
        ctx.close()
        del g, nat, dst
    return out


def kernel_sweep(torch, lqcd, synth, U, psi, dims, device, peak):
    """The other bandwidth-bound kernels of the path at the workload size (north_star: HBM GB/s for clover apply and
    the BLAS-1 kernels beside dslash): clover / clover-inverse apply (120 w B/site) and the fused BLAS-1 entry points
    (vectors streamed x 24 w B/site).  One-parity fields of 100-600 MB: larger than L2 together.  The two reduction
    kernels return their scalars to the host, so their time includes that read-back."""
    cfg = synth.CONFIGS[WORKLOAD]
    out = {}
    for prec in (4, 8):
        ctx = lqcd.Context(dims, prec, 18, -1, device)
        g = ctx.gauge_pack(ctx.to_device(U))
        A, Ai = ctx.clover_build(g, cfg["csw"], cfg["kappa"])
        nat = ctx.spinor_pack(ctx.to_device(psi))
        x, y = ctx.parity(nat, 0), ctx.parity(nat, 1)
        z, w = ctx.new_spinor(1), ctx.new_spinor(1)
        z.copy_(x)
        w.copy_(y)
        site = ctx.Vh * prec
        runs = (("clover_apply", lambda i: ctx.clover_apply(z if i & 1 else w, x if i & 1 else y, A, i & 1), 120),
                ("clover_inverse_apply", lambda i: ctx.clover_apply(z if i & 1 else w, x if i & 1 else y, Ai, i & 1), 120),
                ("blas_xpay", lambda i: ctx.blas_xpay(x if i & 1 else y, 0.5, z if i & 1 else w), 72),
                ("blas_caxpbypz", lambda i: ctx.blas_caxpbypz(0.5 + 0.1j, x, 0.25 - 0.2j, y, z if i & 1 else w), 96),
                ("blas_axpy_norm", lambda i: ctx.blas_axpy_norm(1e-3, x if i & 1 else y, z if i & 1 else w), 72),
                ("blas_cdot", lambda i: ctx.blas_cdot(x if i & 1 else z, y if i & 1 else w), 48))
        row = {}
        for name, fn, reals in runs:
            t = time_batched(torch, fn)
            row[name] = {"us": t * 1e6, "GBps": reals * site / t / 1e9, "frac_of_measured_peak": reals * site / t / 1e9 / peak,
                         "bytes_per_site": reals * prec}
            if name in ("blas_axpy_norm", "blas_cdot"):
                row[name]["includes_host_readback"] = True  # the call returns its scalars: stream sync inside
        out["fp%d" % (8 * prec)] = row
        ctx.close()
        del g, A, Ai, nat, z, w
    return out


def mrhs_sweep(torch, lqcd, U, psi, dims, device, peak, nrhs=12):
    """Standalone multi-RHS dslash (lqcd_dslash_mrhs, 12 columns) at the workload size.  Algorithmic
    bytes per site: links once for all columns, every column's input and output once:
    (8R + nrhs*48)*w.  Reported per column beside the single-RHS time of the same variant."""
    out = {}
    for prec, recon in ((4, 18), (4, 12), (8, 18), (8, 12)):
        ctx = lqcd.Context(dims, prec, recon, -1, device)
        g = ctx.gauge_pack(ctx.to_device(U))
        nat = ctx.spinor_pack(ctx.to_device(psi))
        n = ctx.spinor_bytes // prec
        src = [torch.cat([ctx.parity(nat, p)] * nrhs) for p in (0, 1)]
        dst = ctx.new_spinor(nrhs)
        t = time_batched(torch, lambda i: ctx.dslash_mrhs(dst, src[1 - (i & 1)], g, i & 1, nrhs), n=6, reps=5, warm=4)
        by = (8 * recon + nrhs * 48) * prec * ctx.Vh
        out["fp%d_recon%d" % (8 * prec, recon)] = {
            "nrhs": nrhs, "us": t * 1e6, "us_per_column": t * 1e6 / nrhs, "GBps": by / t / 1e9,
            "frac_of_measured_peak": by / t / 1e9 / peak, "GFLOPs": FLOPS_PER_SITE * ctx.Vh * nrhs / t / 1e9,
            "bytes_per_site_and_column": by / ctx.Vh / nrhs}
        ctx.close()
        del g, nat, src, dst
    return out


def extras(torch, lqcd, synth, U, b, ctx, gauge, device):
    """SURVEY.md §8(f) rows measured beside the headline (not part of `value`):
    mixed   : the same 32^3x64 system to the same fp64 tolerance by fp64 defect correction around fp32
              reconstruct-12 solves (lqcd_invert_mixed), CGNE and BiCGStab;
    propagator : BASELINE configs[2] (16^3x32, fp32, reconstruct-12): the 12 spin-colour columns of a
              point-source propagator by CGNE to 1e-6, 12 single solves vs one lqcd_invert_multi."""
    out = {}
    cfg = synth.CONFIGS[WORKLOAD]
    kappa, csw = cfg["kappa"], cfg["csw"]
    A, Ai = ctx.clover_build(gauge, csw, kappa)
    lo = lqcd.Context(cfg["dims"], 4, 12, -1, device)
    g_lo = lo.gauge_pack(lo.to_device(U))
    A_lo, Ai_lo = lo.clover_build(g_lo, csw, kappa)
    b_dev = ctx.to_device(b)
    mixed = {}
    for solver in ("cgne", "bicgstab"):
        for _ in range(2):
            # CGNE: right-preconditioned symmetric form (no clover apply per iteration); BiCGStab applies only
            # Mhat, never its adjoint, and the left form is two fused launches
            mp = MATPC if solver == "cgne" else 1
            _, r64 = ctx.invert(b_dev, gauge, A, Ai, kappa, tol=1e-10, maxiter=2000, solver=solver, matpc=mp)
            _, rmx = ctx.invert_mixed(lo, b_dev, gauge, A, Ai, g_lo, A_lo, Ai_lo, kappa, tol=1e-10,
                                      inner_tol=1e-5, maxiter=2000, solver=solver, matpc=mp)
        mixed[solver] = {"fp64_seconds": r64.seconds, "fp64_iterations": r64.iterations,
                         "mixed_seconds": rmx.seconds, "mixed_inner_iterations": rmx.iterations,
                         "mixed_true_resid": rmx.true_resid, "fp64_true_resid": r64.true_resid,
                         "speedup": r64.seconds / rmx.seconds}
    # the same with a 16-bit-storage inner context (prec = 2: int16 + per-site norms, fp32 arithmetic), and its dslash
    # against its own roofline: (8R + 48) reals x 2 B + two 4 B spinor norms per output site
    hf = lqcd.Context(cfg["dims"], 2, 12, -1, device)
    g_h = hf.gauge_pack(hf.to_device(synth.round_fp32(U)))
    A_h, Ai_h = hf.clover_to_half(A_lo), hf.clover_to_half(Ai_lo)
    for solver in ("cgne", "bicgstab"):
        mp = MATPC if solver == "cgne" else 1
        for _ in range(2):
            _, r16 = ctx.invert_mixed(hf, b_dev, gauge, A, Ai, g_h, A_h, Ai_h, kappa, tol=1e-10, inner_tol=2e-3,
                                      maxiter=4000, solver=solver, matpc=mp)
        mixed[solver].update({"mixed16_seconds": r16.seconds, "mixed16_inner_iterations": r16.iterations,
                              "mixed16_true_resid": r16.true_resid, "mixed16_status": r16.status,
                              "mixed16_speedup_vs_fp64": mixed[solver]["fp64_seconds"] / r16.seconds})
    peak = measured_peaks()[0]
    nat_h = hf.spinor_pack(hf.to_device(synth.round_fp32(b)))
    dst_h = hf.new_spinor(2)
    th = time_batched(torch, lambda i: hf.dslash(hf.parity(dst_h, i & 1), hf.parity(nat_h, 1 - (i & 1)), g_h, i & 1))
    by_h = ((8 * 12 + 48) * 2 + 8) * hf.Vh
    mixed["dslash_16bit_recon12"] = {"us": th * 1e6, "GBps": by_h / th / 1e9, "frac_of_measured_peak": by_h / th / 1e9 / peak,
                                     "bytes_per_site": by_h // hf.Vh, "GFLOPs": FLOPS_PER_SITE * hf.Vh / th / 1e9}
    hf.close()
    del g_h, A_h, Ai_h, nat_h, dst_h
    out["mixed_precision_32x64"] = mixed
    # 12-column point-source propagator at the headline size to the fp64 tolerance: 12 mixed
    # solves one after the other vs one batched mixed solve (lqcd_invert_multi_mixed), BiCGStab
    dims = cfg["dims"]
    cols = np.stack([synth.source(dims, "point", spin=sp, colour=c) for sp in range(4) for c in range(3)])
    B = ctx.to_device(cols)
    ws, _ = ctx.workspace_multi(12, "bicgstab")
    ws_lo, _ = lo.workspace_multi(12, "bicgstab")
    for _ in range(2):
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record()
        r1 = [ctx.invert_mixed(lo, B[j], gauge, A, Ai, g_lo, A_lo, Ai_lo, kappa, tol=1e-10, inner_tol=1e-5,
                               maxiter=2000, solver="bicgstab", matpc=1, workspace=ws, workspace_lo=ws_lo)[1]
              for j in range(12)]
        e1.record()
        _, rs, rc = ctx.invert_multi_mixed(lo, B, gauge, A, Ai, g_lo, A_lo, Ai_lo, kappa, tol=1e-10, inner_tol=1e-5,
                                           maxiter=2000, solver="bicgstab", matpc=1, workspace=ws,
                                           workspace_lo=ws_lo)
        e2.record()
        torch.cuda.synchronize()
    out["propagator_32x64_mixed_bicgstab"] = {
        "single_solves_ms": e0.elapsed_time(e1), "batched_ms": e1.elapsed_time(e2),
        "speedup": e0.elapsed_time(e1) / e1.elapsed_time(e2),
        "inner_iterations_single": [r.iterations for r in r1], "inner_iterations_batched": [r.iterations for r in rs],
        "status": rc, "worst_true_resid_single": max(r.true_resid for r in r1),
        "worst_true_resid_batched": max(r.true_resid for r in rs)}
    del B, ws, ws_lo
    lo.close()
    del A, Ai, g_lo, A_lo, Ai_lo
    c3 = synth.CONFIGS[3]
    dims = c3["dims"]
    U3 = synth.gauge(dims, c3["eps"], c3["seed"])
    p = lqcd.Context(dims, 4, 12, -1, device)
    g3 = p.gauge_pack(p.to_device(U3))
    A3, Ai3 = p.clover_build(g3, c3["csw"], c3["kappa"])
    cols = np.stack([synth.source(dims, "point", spin=sp, colour=c) for sp in range(4) for c in range(3)])
    B = p.to_device(cols)
    ws1, _ = p.workspace("cgne")          # one workspace for the single solves, one for the batched call: like for like
    ws12, _ = p.workspace_multi(12, "cgne")
    for _ in range(2):
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        e0.record()
        its = [p.invert(B[j], g3, A3, Ai3, c3["kappa"], tol=1e-6, solver="cgne", matpc=MATPC, workspace=ws1)[1].iterations
               for j in range(12)]
        e1.record()
        _, rs, rc = p.invert_multi(B, g3, A3, Ai3, c3["kappa"], tol=1e-6, solver="cgne", matpc=MATPC, workspace=ws12)
        e2.record()
        torch.cuda.synchronize()
    out["propagator_16x32_fp32_recon12"] = {
        "single_solves_ms": e0.elapsed_time(e1), "batched_ms": e1.elapsed_time(e2),
        "speedup": e0.elapsed_time(e1) / e1.elapsed_time(e2), "iterations_single": its,
        "iterations_batched": [r.iterations for r in rs], "status": rc,
        "worst_true_resid": max(r.true_resid for r in rs)}
    p.close()
    del g3, A3, Ai3, B
    # BASELINE configs[4] (48^3x96, 10.6M sites, fp32 reconstruct-12): capacity and bandwidth of dslash and
    # clover-inverse apply, and a BiCGStab solve to 1e-6 (symmetric form from the left: BiCGStab never applies the adjoint)
    c5 = synth.CONFIGS[5]
    dims = c5["dims"]
    U5 = synth.gauge(dims, c5["eps"], c5["seed"])
    b5 = synth.source(dims, c5["source"], c5["src_seed"])
    q = lqcd.Context(dims, 4, 12, -1, device)
    g5 = q.gauge_pack(q.to_device(U5))
    del U5
    A5, Ai5 = q.clover_build(g5, c5["csw"], c5["kappa"])
    nat = q.spinor_pack(q.to_device(b5))
    dst = q.new_spinor(2)
    peak = measured_peaks()[0]
    td = time_batched(torch, lambda i: q.dslash(q.parity(dst, i & 1), q.parity(nat, 1 - (i & 1)), g5, i & 1), n=10, reps=5)
    tc = time_batched(torch, lambda i: q.clover_apply(q.parity(dst, i & 1), q.parity(nat, i & 1), Ai5, i & 1), n=10, reps=5)
    bd, bc = dslash_alg_bytes(12, 4, q.Vh), 120 * 4 * q.Vh
    for _ in range(2):
        _, r5 = q.invert(q.to_device(b5), g5, A5, Ai5, c5["kappa"], tol=1e-6, maxiter=2000, solver="bicgstab", matpc=1)
    out["capacity_48x96_fp32_recon12"] = {
        "device_bytes_fields": int(q.gauge_bytes + 2 * q.clover_bytes + 2 * 2 * q.spinor_bytes),
        "dslash": {"us": td * 1e6, "GBps": bd / td / 1e9, "frac_of_measured_peak": bd / td / 1e9 / peak,
                   "frac_of_8TBps": bd / td / 8e12, "GFLOPs": FLOPS_PER_SITE * q.Vh / td / 1e9},
        "clover_inverse_apply": {"us": tc * 1e6, "GBps": bc / tc / 1e9, "frac_of_measured_peak": bc / tc / 1e9 / peak},
        "bicgstab_1e-6": {"seconds": r5.seconds, "iterations": r5.iterations, "true_resid": r5.true_resid,
                          "status": r5.status}}
    q.close()
    return out


def small_solves(torch, lqcd, synth, device):
    """Solve wall time at BASELINE configs 1-3 (the lattices that fit in L2, where the host's share of an iteration
    shows): device seconds of the whole lqcd_invert call (CUDA events inside the library), iterations, launches."""
    out = {}
    runs = ((1, 8, 18, "point", "cgne", 0, 1e-10), (2, 8, 18, "z2", "bicgstab", 1, 1e-10), (2, 4, 18, "z2", "bicgstab", 1, 1e-6),
            (3, 4, 12, "gaussian", "cgne", MATPC, 1e-6), (3, 4, 12, "gaussian", "bicgstab", 1, 1e-6))
    for n, prec, recon, kind, solver, matpc, tol in runs:
        c = synth.CONFIGS[n]
        U = synth.gauge(c["dims"], c["eps"], c["seed"])
        b = synth.source(c["dims"], kind, c["src_seed"])
        ctx = lqcd.Context(c["dims"], prec, recon, -1, device)
        g = ctx.gauge_pack(ctx.to_device(U))
        A, Ai = ctx.clover_build(g, c["csw"], c["kappa"])
        bd = ctx.to_device(b)
        ws, _ = ctx.workspace(solver)
        best = None
        for _ in range(5):
            _, r = ctx.invert(bd, g, A, Ai, c["kappa"], tol=tol, maxiter=2000, solver=solver, matpc=matpc, workspace=ws)
            if best is None or r.seconds < best.seconds:
                best = r
        out["config%d_fp%d_recon%d_%s" % (n, 8 * prec, recon, solver)] = {
            "dims": list(c["dims"]), "tol": tol, "matpc": matpc, "us": best.seconds * 1e6, "iterations": best.iterations,
            "us_per_iteration": best.seconds * 1e6 / max(best.iterations, 1), "kernel_launches": best.kernel_launches,
            "true_resid": best.true_resid, "status": best.status, "graph_blocks_replayed": ctx.graph_launch_count()}
        ctx.close()
    return out


def reduce_over_ranks(dist, dt, sums, device):
    """Multi-replica aggregation: MAX of the device time over ranks, SUM of the work counters.
    dist = torch.distributed (initialised) or None for a single process."""
    if dist is None:
        return dt, list(sums)
    import torch
    t = torch.tensor([dt], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    s = torch.tensor(list(sums), device=device, dtype=torch.float64)
    dist.all_reduce(s, op=dist.ReduceOp.SUM)
    return float(t.item()), [float(v) for v in s.tolist()]


def run_gpu(args):
    import torch
    from paper_2411_08461_b200 import lqcd, synth
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    peak, peak_src = measured_peaks()

    cfg = synth.CONFIGS[WORKLOAD]
    dims = cfg["dims"]
    kappa, csw, tol = cfg["kappa"], cfg["csw"], 1e-10
    U = synth.gauge(dims, cfg["eps"], cfg["seed"])            # same seeded field on every replica
    b = synth.source(dims, cfg["source"], cfg["src_seed"] + rank)
    ctx = lqcd.Context(dims, 8, 18, -1, local)
    U_dev, b_dev = ctx.to_device(U), ctx.to_device(b)
    gauge = ctx.empty(ctx.gauge_bytes)
    ws, _ = ctx.workspace("cgne")
    lib, P, S = ctx.lib, lqcd._p, lqcd._stream
    results = []

    def step():
        ctx._check(lib.lqcd_gauge_pack(ctx.h, P(gauge), P(U_dev), S()))
        x, res = ctx.invert(b_dev, gauge, None, None, kappa, csw=csw, tol=tol, maxiter=2000,
                            solver="cgne", matpc=MATPC, workspace=ws)
        results.append(res)
        return x

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()

    for _ in range(max(args.warmup, 3)):
        step()
    results.clear()
    sampler = ClockSampler(local)
    ctx.profile_enable(True)
    ctx.profile_read()
    barrier()
    sampler.start()
    l0, a0 = ctx.launch_count(), ctx.algorithmic_bytes()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    clocks = sampler.stop()
    ctx.profile_enable(False)
    dt = e0.elapsed_time(e1) * 1e-3
    launches = ctx.launch_count() - l0
    alg = ctx.algorithmic_bytes() - a0
    n_ds, ds_ms, ds_bytes = ctx.profile_read()
    dt, (alg, launches) = reduce_over_ranks(dist, dt, [alg, float(launches)], "cuda")
    value = alg / dt / 1e9
    res = results[-1]

    # ---- end to end through the host-buffer entry points (pinned host inputs, result read back)
    U_h = torch.from_numpy(U).pin_memory()
    b_h = torch.from_numpy(b).pin_memory()
    x_h = torch.empty_like(b_h).pin_memory()
    g_scr = ctx.empty(U_h.numel() * 16)
    h_scr, _ = ctx.host_scratch("cgne")
    A, Ai = ctx.empty(ctx.clover_bytes), ctx.empty(ctx.clover_bytes)

    def step_e2e():
        # one C-ABI call from host buffers: uploads on the context's copy stream (the source goes up while the
        # links are packed and the clover field is built), solve, download
        return ctx.solve_host(x_h, b_h, U_h, gauge, A, Ai, csw, kappa, g_scr, h_scr, tol=tol, maxiter=2000,
                              solver="cgne", matpc=MATPC)[1]

    step_e2e()
    barrier()
    a0 = ctx.algorithmic_bytes()
    e0.record()
    n_e2e = max(1, min(args.steps, 3))
    for _ in range(n_e2e):
        r2 = step_e2e()
    e1.record()
    barrier()
    dt2 = e0.elapsed_time(e1) * 1e-3
    alg2 = ctx.algorithmic_bytes() - a0
    dt2, (alg2,) = reduce_over_ranks(dist, dt2, [alg2], "cuda")
    e2e = {"value": alg2 / dt2 / 1e9, "unit": "GB/s",
           "h2d_bytes_per_step": int(U_h.numel() * 16 + b_h.numel() * 16),
           "d2h_bytes_per_step": int(x_h.numel() * 16), "ms_per_step": dt2 / n_e2e * 1e3,
           "true_resid": r2.true_resid}

    # The driver keeps the standard keys (roofline, cpu_baseline, e2e, config, clocks) and only the NAMES of the others,
    # and it stores the tail of stdout: the large blocks come first in the line, and the figures the targets are stated
    # on are repeated, compact, inside `roofline` and `cpu_baseline`.
    line = {}
    roofline = {"bound": "hbm", "achieved": ds_bytes / (ds_ms * 1e-3) / 1e9 if ds_ms > 0 else None,
                "peak": peak, "unit": "GB/s",
                "frac": (ds_bytes / (ds_ms * 1e-3) / 1e9 / peak) if ds_ms > 0 else None,
                "traffic": traffic_from_profile(), "traffic_source": "committed ncu --set full capture under profiles/ (not this run)",
                "kernel": "dslash_kernel<double,18,*,EPI 1|9|10> (fused clover and CG epilogues)",
                "launches_timed": n_ds, "avg_launch_us": ds_ms * 1e3 / max(n_ds, 1),
                "alg_bytes_per_launch": ds_bytes / max(n_ds, 1), "peak_source": peak_src,
                "frac_of_8TBps": (ds_bytes / (ds_ms * 1e-3) / 8e12) if ds_ms > 0 else None,
                "solve_32x64_fp64_cgne": {"seconds": res.seconds, "iterations": res.iterations, "true_resid": res.true_resid}}
    cpu = None
    if rank == 0 and not args.no_sweep:
        line["dslash"] = dslash_sweep(torch, lqcd, U, b, dims, local, peak)
        line["kernels"] = kernel_sweep(torch, lqcd, synth, U, b, dims, local, peak)
        # north_star's target: Wilson-clover dslash at 32^3x64 in fp32 >= 70 % of HBM bandwidth
        roofline["headline_dslash_fp32"] = {
            k: {f: line["dslash"]["fp32_" + k][f] for f in ("us", "GBps", "frac_of_measured_peak", "frac_of_8TBps", "GFLOPs")}
            for k in ("recon18", "recon12")}
        roofline["clover_apply_frac"] = {k: line["kernels"][k]["clover_apply"]["frac_of_measured_peak"] for k in ("fp32", "fp64")}
    if rank == 0 and world == 1 and not args.no_extras:
        nr = extras(torch, lqcd, synth, U, b, ctx, gauge, local)
        nr["dslash_mrhs_32x64"] = mrhs_sweep(torch, lqcd, U, b, dims, local, peak)
        nr["small_lattice_solves"] = small_solves(torch, lqcd, synth, local)
        line["next_rows"] = nr
        roofline["dslash_mrhs_32x64_frac"] = {k: v["frac_of_measured_peak"] for k, v in nr["dslash_mrhs_32x64"].items()}
        roofline["mixed_precision_32x64_cgne_ms"] = {k: nr["mixed_precision_32x64"]["cgne"][k + "_seconds"] * 1e3
                                                     for k in ("fp64", "mixed", "mixed16")}
        roofline["dslash_16bit_recon12_frac"] = nr["mixed_precision_32x64"]["dslash_16bit_recon12"]["frac_of_measured_peak"]
        roofline["propagator_32x64_mixed_bicgstab_ms"] = nr["propagator_32x64_mixed_bicgstab"]["batched_ms"]
        roofline["propagator_16x32_fp32_cgne_ms"] = nr["propagator_16x32_fp32_recon12"]["batched_ms"]
        roofline["worst_true_resid_fp32_1e-6"] = max(nr["propagator_16x32_fp32_recon12"]["worst_true_resid"],
                                                      nr["capacity_48x96_fp32_recon12"]["bicgstab_1e-6"]["true_resid"])
    if rank == 0 and world == 1 and not args.no_cpu:
        # the oracle on the host cores: all threads at the workload size, one thread at 16^3x32 (1/16 of the volume)
        full = oracle_leg_subprocess(WORKLOAD, 3, (2, 5))
        one = oracle_leg_subprocess(3, 2, (2, 4), threads=1)
        # iterations of the oracle's own solve (asymmetric CGNE) = those of the GPU's (equal to +-1, tests/test_gpu_solvers.py)
        ctx._check(lib.lqcd_gauge_pack(ctx.h, P(gauge), P(U_dev), S()))
        _, ra = ctx.invert(b_dev, gauge, None, None, kappa, csw=csw, tol=tol, maxiter=2000, solver="cgne", matpc=0, workspace=ws)
        est = None
        if "error" not in full:
            est = full["cgne_fixed_seconds"] + ra.iterations * full["cgne_seconds_per_iteration"]
        cpu = {"value": full.get("dslash_GBps"), "unit": "GB/s", "cores": full.get("threads"), "kind": "oracle",
               "sample": "32^3x64 fp64 on all host threads: clover build, 3 full-lattice hopping-term applications, 3 clover "
                         "applies, even-odd CGNE (asymmetric) timed at 2 and 5 iterations; value = dslash algorithmic bytes / time",
               "all_threads_32x64": full,
               "cgne_solve_seconds_estimated": est,
               "cgne_solve_estimate": "fixed + seconds/iteration x %d iterations (the GPU's count for the same asymmetric CGNE to 1e-10; "
                                      "GPU: %.4f s)" % (ra.iterations, ra.seconds),
               "one_thread_16x32": one}
    line.update({
        "metric": METRIC, "value": value, "unit": "GB/s", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "configs[3]: 32^3x64 (2.1M sites), eps=0.8 links seed 4, kappa=0.1248, "
                               "csw=1.8, Gaussian source seed 104; fp64, 18-real links, antiperiodic t",
                   "step": "gauge pack + clover build/inverse + even-odd CGNE to 1e-10 (symmetric Schur complement, "
                           "right-preconditioned: 1 - k^2 D_eo A_oo^-1 D_oe A_ee^-1, 32 iterations; the asymmetric one takes 54) + reconstruct + "
                           "true residual",
                   "l2": "inputs larger than L2 (links 1.2 GB, clover 2x1.2 GB, spinors 0.2 GB each)",
                   "parallelism": "replicas only (one independent solve per GPU)",
                   "value_definition": "sum over all kernels of the step of their algorithmic HBM bytes / step time"},
        "roofline": roofline,
        "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "solve": {"solver": "cgne", "tol": tol, "iterations": res.iterations, "seconds": res.seconds,
                  "iter_resid": res.iter_resid, "true_resid": res.true_resid, "status": res.status,
                  "dslash_count": res.dslash_count, "kernel_launches": res.kernel_launches},
    })
    if cpu is not None:
        line["cpu_baseline"] = cpu
    if rank == 0:
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


def traffic_from_profile():
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel (fp64 dslash
    with fused clover epilogue) from the committed `ncu --set full` raw page under profiles/
    (newest round first), averaged over the captured launches; None if no capture is committed."""
    import csv
    import glob
    for path in sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_dslash_full_raw.csv")), reverse=True):
        try:
            rows = list(csv.reader(open(path)))
            hdr, units = rows[0], rows[1]
            ik, ir, iw = hdr.index("Kernel Name"), hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
            scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
            tot = [float(r[ir]) * scale[units[ir]] + float(r[iw]) * scale[units[iw]]
                   for r in rows[2:] if r[ik].startswith("void dslash_kernel<double, 18")]
            if tot:
                return sum(tot) / len(tot)
        except Exception:
            continue
    return None


def spawn_command(args, port=None):
    """`python bench.py --gpus N` outside torchrun: the same command line under torch.distributed.run, one rank per GPU."""
    import socket
    if port is None:
        with socket.socket() as so:
            so.bind(("127.0.0.1", 0))
            port = so.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__),
           "--gpus", str(args.gpus), "--steps", str(args.steps), "--warmup", str(args.warmup), "--impl", args.impl]
    for flag, on in (("--no-sweep", args.no_sweep), ("--no-extras", args.no_extras), ("--no-cpu", args.no_cpu)):
        if on:
            cmd.append(flag)
    return cmd


def run_selftest(args):
    """Launch plumbing only (tests/test_bench_dist.py): every rank joins a gloo group, rank 0 prints the world size."""
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        dist.init_process_group("gloo")
        t = torch.ones(1)
        dist.all_reduce(t)
        world = int(t.item())
    if int(os.environ.get("RANK", "0")) == 0:
        print(json.dumps({"impl": "selftest", "n_gpus": world}))
    if dist.is_initialized():
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference", "cpu-leg", "selftest"])
    ap.add_argument("--cpu-leg", default="", help="internal: config,applications,iters0,iters1 of one oracle leg")
    ap.add_argument("--no-sweep", action="store_true", help="skip the standalone dslash sweep")
    ap.add_argument("--no-extras", action="store_true", help="skip the SURVEY 8(f) rows (mixed precision, batched propagator)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the CPU-oracle baseline leg")
    ap.add_argument("--mrhs-only", action="store_true", help="only the standalone multi-RHS dslash sweep (profiling runs)")
    ap.add_argument("--propagator-only", action="store_true",
                    help="only the batched 12-column mixed-precision BiCGStab propagator at 32^3x64 (profiling runs)")
    args = ap.parse_args()
    if args.impl == "cpu-leg":
        c, n, i0, i1 = (int(v) for v in args.cpu_leg.split(","))
        print(json.dumps(oracle_legs(c, n, (i0, i1))))
        return 0
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return subprocess.call(spawn_command(args))  # N ranks, one per GPU; rank 0 prints the line with n_gpus = N
    if args.impl == "selftest":
        return run_selftest(args)
    if args.propagator_only:
        import torch
        from paper_2411_08461_b200 import lqcd, synth
        cfg = synth.CONFIGS[WORKLOAD]
        dims, kappa, csw = cfg["dims"], cfg["kappa"], cfg["csw"]
        U = synth.gauge(dims, cfg["eps"], cfg["seed"])
        ctx, lo = lqcd.Context(dims, 8, 18, -1, 0), lqcd.Context(dims, 4, 12, -1, 0)
        g, g_lo = ctx.gauge_pack(ctx.to_device(U)), lo.gauge_pack(lo.to_device(U))
        (A, Ai), (A_lo, Ai_lo) = ctx.clover_build(g, csw, kappa), lo.clover_build(g_lo, csw, kappa)
        B = ctx.to_device(np.stack([synth.source(dims, "point", spin=sp, colour=c) for sp in range(4) for c in range(3)]))
        ws, _ = ctx.workspace_multi(12, "bicgstab")
        ws_lo, _ = lo.workspace_multi(12, "bicgstab")
        for _ in range(2):
            _, rs, rc = ctx.invert_multi_mixed(lo, B, g, A, Ai, g_lo, A_lo, Ai_lo, kappa, tol=1e-10, inner_tol=1e-5, maxiter=2000,
                                               solver="bicgstab", matpc=1, workspace=ws, workspace_lo=ws_lo)
        print(json.dumps({"propagator_32x64_mixed_bicgstab_batched_ms": rs[0].seconds * 1e3, "status": rc,
                          "inner_iterations": [r.iterations for r in rs], "launches": rs[0].kernel_launches}))
        return 0
    if args.mrhs_only:
        import torch
        from paper_2411_08461_b200 import lqcd, synth
        cfg = synth.CONFIGS[WORKLOAD]
        U = synth.gauge(cfg["dims"], cfg["eps"], cfg["seed"])
        b = synth.source(cfg["dims"], cfg["source"], cfg["src_seed"])
        print(json.dumps({"dslash_mrhs_32x64": mrhs_sweep(torch, lqcd, U, b, cfg["dims"], 0, measured_peaks()[0])}))
        return 0
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
