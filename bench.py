#!/usr/bin/env python
"""bench.py -- throughput of the LinMin hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--cubes C]

One "step" = one pass of the whole hot path (projection, IPLS, exact finish, uncertainty
propagation, residual, output store) over the workload.  At N = 1 the workload is BASELINE.json
configs[4] ("throughput": L = 128, R = 32, N = 16,777,216 = 128 OMEGA-like cubes, per-pixel sigma),
synthetic and seeded (paper_1402_2518_b200/synth.py).  With --gpus N > 1 (under torchrun, or plain: bench.py then
starts its own N ranks through torch.distributed.run on 127.0.0.1 and refuses when fewer devices are visible) every
rank owns its own 128 cubes ("weak" scaling; pixels are independent, no collective on the data path).
`value` = spectra/s with inputs resident in HBM; `e2e` = the same through linmin_unmix_host with
pinned HOST buffers (H2D and D2H inside the timed region).  `--impl reference` times the CPU fp64
oracle (oracle/) on a bounded sample of the same workload.  Prints ONE JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from concurrent.futures import ThreadPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1402_2518_b200.shard import cube_block, launch_plan, max_over_ranks  # noqa: E402
from paper_1402_2518_b200.synth import CONFIGS, make_cube, make_library  # noqa: E402

METRIC = "unmixed spectra/sec"
UNIT = "spectra/s"
CUBE = 128 * 1024
# FP32 roofline denominator: 148 SMs x 128 FP32 lanes x 2 flop x 1.965 GHz
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
SEED = CONFIGS["throughput"]["seed"]


def flops_model(L, R, it, piv, k):
    """Algorithmic flops per pixel; it, piv, k are the per-pixel counts the kernels
    report in info_out.  Returns (ipls_kernel_flops, finish_kernel_flops), each summed over pixels."""
    it = it.astype(np.float64); piv = piv.astype(np.float64); k = k.astype(np.float64)
    proj = 2.0 * L * R
    ipls = it * (R ** 3 / 3.0 + 8.0 * R ** 2 + 30.0 * R)
    fin = (piv + 1.0) * (2.0 * L * k * k + 2.0 * L * k + 2.0 * L * R)
    unc = 2.0 * L * k * k + 3.0 * L * k
    res = 2.0 * L * k + 3.0 * L
    return float((proj + ipls).sum()), float((fin + unc + res).sum())


def executed_ipls_flops(L, R, it):
    """What one iteration of the IPLS kernel executes as useful flops: R^3/3 for the factorisation and
    five triangular solves (5 R^2) -- G a is carried by the Newton identity instead of a mat-vec -- against the
    R^3/3 + 8 R^2 + 30 R of the SURVEY's model."""
    it = it.astype(np.float64)
    return float((2.0 * L * R + it * (R ** 3 / 3.0 + 5.0 * R ** 2)).sum())


def gen_cubes(first_cube, n_cubes, Y_out, S_out, threads):
    """Fill Y_out, S_out (numpy views, (n_cubes*CUBE, L)) with cubes first_cube.. of config 4."""
    cfg = CONFIGS["throughput"]
    A64, _ = make_library(cfg, np.random.Generator(np.random.PCG64(SEED)))

    def one(c):
        rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([SEED, first_cube + c])))
        Y, s, _, _ = make_cube(cfg, A64, rng, CUBE)
        Y_out[c * CUBE:(c + 1) * CUBE] = Y
        S_out[c * CUBE:(c + 1) * CUBE] = s

    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(one, range(n_cubes)))
    return A64.astype(np.float32)


class ClockSampler:
    """nvidia-smi sampling DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1])); smax.append(float(f[2])); power.append(float(f[3]))
            except ValueError:
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "samples": len(sm),
                "power_w_max": float(max(power)), "reasons": sorted(reasons)}


def host_threads():
    """Threads for the oracle legs: the host cores this process may use.  Passed explicitly, because torchrun
    presets OMP_NUM_THREADS=1 for its workers and the oracle would otherwise run on one core there."""
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:
        return max(1, os.cpu_count() or 1)


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle as it stands, on a bounded sample of the same workload."""
    if rank != 0:
        return
    import oracle
    oracle.build()
    n = 32768 if args.sample is None else args.sample
    cfg = CONFIGS["throughput"]
    A64, _ = make_library(cfg, np.random.Generator(np.random.PCG64(SEED)))
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([SEED, 0])))
    Y, s, _, _ = make_cube(cfg, A64, rng, CUBE)
    Y, s = Y[:n], s[:n]
    A = A64.astype(np.float32)
    cores = host_threads()
    for _ in range(args.warmup):
        oracle.solve(A, Y[: max(1, n // 8)], s[: max(1, n // 8)], nthreads=cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.solve(A, Y, s, nthreads=cores)
    dt = (time.perf_counter() - t0) / args.steps
    v = n / dt
    sample = f"first {n} pixels of cube 0 of config 4 per step"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "throughput (config 4): L=128, R=32, per-pixel sigma; " + sample},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def time_calls(torch, fn, reps=3):
    fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


def run_extras(linmin, torch, dev, A4, Yd, Sd):
    """Not the headline: (a) BASELINE.json configs[2] and [3] (R = 64, R = 256: the any-size kernels), whole config,
    with the per-kernel split and the fraction of the FP32 peak in SURVEY 8(d) flops; (b) the NEXT-row options of
    SURVEY.md 8(f) on the first 2^20 pixels of the timed workload."""
    from paper_1402_2518_b200.synth import make_workload
    out = {"configs": {}, "options": {}}
    for name in ("crism", "stress"):
        w = make_workload(name)
        At, Yt, St = (torch.from_numpy(x).to(dev) for x in (w.A, w.Y, w.sigma))
        lib = linmin.library_create(At)
        lib.enable_timing(True)
        res = {}

        def call():
            res["o"] = linmin.unmix_lib(lib, Yt, St)
        ms = time_calls(torch, call, reps=2 if name == "stress" else 3)
        ipls_ms, fin_ms = lib.last_timing()
        info = res["o"][3].cpu().numpy()
        it, piv, k = (info >> 8) & 0xff, (info >> 16) & 0xff, (info >> 24) & 0xff
        f_ipls, f_fin = flops_model(w.L, w.R, it, piv, k)
        out["configs"][name] = {"L": w.L, "R": w.R, "N": w.N, "ms": ms, "spectra_per_s": w.N / (ms * 1e-3),
                                "ipls_ms": ipls_ms, "finish_ms": fin_ms, "mean_iterations": float(it.mean()),
                                "ipls_frac_of_fp32_peak": f_ipls / (ipls_ms * 1e-3) / 1e12 / FP32_PEAK_TFLOPS,
                                "whole_frac_of_fp32_peak": (f_ipls + f_fin) / (ms * 1e-3) / 1e12 / FP32_PEAK_TFLOPS}
        lib.destroy()
    n = min(1 << 20, Yd.shape[0])
    Y1, S1 = Yd[:n], Sd[:n]
    Ad = torch.from_numpy(A4).to(dev)
    L = A4.shape[0]
    sd = Sd[0].clone()
    idx = torch.arange(L, device=dev)
    C = (0.6 ** (idx[:, None] - idx[None, :]).abs().float()) * torch.outer(sd, sd)
    C = torch.where((idx[:, None] - idx[None, :]).abs() > 3, torch.zeros_like(C), C) + 0.05 * torch.diag(sd ** 2)
    cases = {"sto (headline path)": dict(), "slo": dict(constraint=linmin.CONSTRAINT_SUM_LOWER_THAN_ONE),
             "pos": dict(constraint=linmin.CONSTRAINT_POSITIVITY_ONLY),
             "sto + diagonal covariance": dict(cov=sd), "sto + full covariance (banded, 7 diagonals)": dict(cov=C.contiguous())}
    for label, kw in cases.items():
        lib = linmin.library_create(Ad, **kw)
        ms = time_calls(torch, lambda: linmin.unmix_lib(lib, Y1, None if "cov" in kw else S1))
        out["options"][label] = {"N": n, "ms": ms, "spectra_per_s": n / (ms * 1e-3)}
        lib.destroy()
    # the one-shot form repeats the once-per-library precompute in every call (include/linmin.h): what that costs on one
    # OMEGA-like cube, unweighted and with the full covariance (Cholesky factor + inverse of an L x L matrix per call)
    n1 = min(CUBE, Yd.shape[0])
    Yc, Sc = Yd[:n1], Sd[:n1]
    out["one_shot"] = {"N": n1}
    for label, kw in (("unweighted", dict()), ("full covariance", dict(cov=C.contiguous()))):
        lib = linmin.library_create(Ad, **kw)
        sg = None if kw else Sc
        ms_h = time_calls(torch, lambda: linmin.unmix_lib(lib, Yc, sg))
        ms_o = time_calls(torch, lambda: linmin.unmix(Ad, Yc, sg, **kw))
        out["one_shot"][label] = {"handle_ms": ms_h, "one_shot_ms": ms_o, "precompute_ms": ms_o - ms_h}
        lib.destroy()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--cubes", type=int, default=CONFIGS["throughput"]["cubes"],
                    help="cubes of 131072 pixels per GPU (default 128 = config 4; fewer only for quick checks)")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--sample", type=int, default=None, help="pixels in the cpu_baseline / reference sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true",
                    help="skip the extra report keys (other configs, NEXT-row options); the headline is unaffected")
    args = ap.parse_args()

    if args.impl == "ours":
        # `python bench.py --gpus N` without torchrun starts its own N ranks (one per GPU, this node)
        import socket
        visible = 0
        if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
            import torch
            visible = torch.cuda.device_count()
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        try:
            kind, cmd = launch_plan(args.gpus, os.environ, visible, [os.path.abspath(__file__)] + sys.argv[1:],
                                    sys.executable, port)
        except ValueError as e:
            raise SystemExit(f"bench.py: {e}")
        if kind == "spawn":
            sys.stdout.flush()
            os.execv(sys.executable, cmd)

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_1402_2518_b200 import build, linmin
    if rank == 0:
        build.build_library()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    if world > 1:
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
        dist.barrier()
    linmin.load()
    dev = torch.device("cuda", local_rank if world > 1 else 0)
    torch.cuda.set_device(dev)

    cfg = CONFIGS["throughput"]
    L, R = cfg["L"], cfg["R"]
    n_cubes = args.cubes
    N = n_cubes * CUBE
    threads = max(1, (os.cpu_count() or 8) // max(1, world))

    # ---- inputs: generated on the host (seeded), kept in pinned memory for the e2e leg
    t_gen = time.perf_counter()
    Yh = torch.empty((N, L), dtype=torch.float32, pin_memory=True)
    Sh = torch.empty((N, L), dtype=torch.float32, pin_memory=True)
    A = gen_cubes(cube_block(rank, n_cubes)[0], n_cubes, Yh.numpy(), Sh.numpy(), threads)
    t_gen = time.perf_counter() - t_gen
    Ad = torch.from_numpy(A).to(dev)
    Yd = Yh.to(dev, non_blocking=True)
    Sd = Sh.to(dev, non_blocking=True)
    out = dict(coeffs=torch.empty((N, R), dtype=torch.float32, device=dev),
               coeff_sigma=torch.empty((N, R), dtype=torch.float32, device=dev),
               resid=torch.empty((N,), dtype=torch.float32, device=dev),
               info=torch.empty((N,), dtype=torch.int32, device=dev))
    torch.cuda.synchronize()
    lib = linmin.library_create(Ad)
    lib.enable_timing(True)

    def step():
        linmin.unmix_lib(lib, Yd, Sd, out=out)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def step_shared():
        linmin.unmix_lib(lib, Yd, Sshared, out=out)

    # second timed mode: ONE shared per-channel sigma[L], the paper's own case (one noise
    # covariance per image) -- half the input bytes
    Sshared = Sd[0].clone()
    for _ in range(max(args.warmup, 3)):
        step_shared()
    barrier()
    evs0, evs1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    evs0.record()
    for _ in range(args.steps):
        step_shared()
    evs1.record()
    barrier()
    ms_shared = max_over_ranks(evs0.elapsed_time(evs1) / args.steps, dev)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local_rank if world > 1 else 0)
    sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ipls_ms, fin_ms = [], []
    barrier()
    ev0.record()
    for _ in range(args.steps):
        step()
        # per-kernel events recorded by the library on the same stream; reading them blocks on this
        # step only, which the next launch would do anyway (same stream, same buffers)
        a, b = lib.last_timing()
        ipls_ms.append(a); fin_ms.append(b)
    ev1.record()
    barrier()
    clocks = sampler.stop()
    ms_total = ev0.elapsed_time(ev1)
    ms_step = ms_total / args.steps
    ms_step = max_over_ranks(ms_step, dev)
    value = world * N / (ms_step * 1e-3)
    launches = lib.last_launches() * args.steps

    # ---- flops actually needed (per-pixel counts reported by the kernels)
    info = out["info"].cpu().numpy()
    it, piv, k = (info >> 8) & 0xff, (info >> 16) & 0xff, (info >> 24) & 0xff
    f_ipls, f_fin = flops_model(L, R, it, piv, k)
    # per-pixel distributions behind the means (rank 0's pixels): index = value, entry = pixel count
    histograms = {
        "iterations": np.bincount(it).tolist(), "pivots": np.bincount(piv).tolist(), "support": np.bincount(k).tolist(),
        "frac_support_above_16": float((k > 16).mean()),       # the pixels finish_sweep hands to finish_fast
        "frac_with_support_change": float((piv > 0).mean()),   # the pixels of finish_sweep's second (repair) pass
        "pixels": int(N),
    }
    ipls_avg = float(np.mean(ipls_ms)); fin_avg = float(np.mean(fin_ms))
    achieved = f_ipls / (ipls_avg * 1e-3) / 1e12
    traffic = None
    whole_dram = None
    tpath = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if os.path.exists(tpath):
        try:
            tj = json.load(open(tpath))
            traffic = tj.get("ipls_kernel_dram_bytes_per_pixel", None)
            keys = [kk for kk in tj if kk.endswith("_dram_bytes_per_pixel")]
            whole_dram = float(sum(tj[kk] for kk in keys)) if keys else None     # every kernel of the step (stored ncu figures)
            if traffic is not None:      # K0 and K1 are timed together: both kernels' bytes
                traffic = (traffic + tj.get("start_r32_kernel_dram_bytes_per_pixel", 0.0)) * N
        except (OSError, ValueError):
            traffic = None
    try:
        from bench_probe.fp32_probe import probe_fp32_peak
        ffma_tf, ffma2_tf = probe_fp32_peak()
    except Exception:  # report helper only: never fail the bench line on it
        ffma_tf, ffma2_tf = None, None
    f_exec = executed_ipls_flops(L, R, it)
    roofline = {
        "bound": "alu", "kernel": "projection + start kernel (K0) and IPLS iteration kernel (K1), timed together", "achieved": achieved,
        "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP32_PEAK_TFLOPS,
        "traffic": traffic,
        "traffic_source": "STORED, not measured by this run: dram bytes per pixel of the ncu --set full capture in "
                          "profiles/ncu_traffic.json x N",
        "peak_source": "derived: 148 SM x 128 FP32 lanes x 2 x 1.965 GHz (DESIGN.md); MEASURED_PEAKS.json has no FP32 figure",
        "peak_measured_TFLOPs": {"ffma": ffma_tf, "ffma2": ffma2_tf,
                                 "how": "libfp32probe.so: register-resident independent FMA chains, 8 CTAs x 256 threads per SM"},
        # the same fraction three ways: SURVEY model / derived peak (the contract), SURVEY model / in-run FFMA2 probe,
        # executed-flop model (R^3/3 + 5 R^2 per iteration) / derived peak
        "frac_vs_probe": (achieved / ffma2_tf) if ffma2_tf else None,
        "frac_executed_flops": f_exec / (ipls_avg * 1e-3) / 1e12 / FP32_PEAK_TFLOPS,
        "kernel_ms": {"ipls": ipls_avg, "finish": fin_avg},
        "algorithmic_flops_per_pixel": {"ipls_kernel": f_ipls / N, "finish_kernel": f_fin / N},
        "whole_step": {"achieved": (f_ipls + f_fin) / (ms_step * 1e-3) / 1e12,
                       "frac": (f_ipls + f_fin) / (ms_step * 1e-3) / 1e12 / FP32_PEAK_TFLOPS},
        "hbm": {"algorithmic_bytes_per_pixel": 4 * L * 2 + 4 * (2 * R + 1) + 4,
                "dram_bytes_per_pixel_whole_step_stored": whole_dram,
                "achieved_GBps": (4 * L * 2 + 4 * (2 * R + 1) + 4) * N / (ms_step * 1e-3) / 1e9},
        "mean_iterations": float(it.mean()), "mean_pivots": float(piv.mean()), "mean_support": float(k.mean()),
    }

    # ---- sampled parity on the timed outputs (full size, this launch configuration)
    parity = None
    cpu_baseline = None
    if rank == 0:
        import oracle
        oracle.build()
        sel = np.arange(0, N, max(1, N // 4096))[:4096]
        Ysel, Ssel = Yh.numpy()[sel], Sh.numpy()[sel]
        ora = oracle.solve(A, Ysel, Ssel)
        sel_t = torch.from_numpy(sel).to(dev)
        cg = out["coeffs"][sel_t].cpu().numpy().astype(np.float64)
        sg = out["coeff_sigma"][sel_t].cpu().numpy().astype(np.float64)
        rg = out["resid"][sel_t].cpu().numpy().astype(np.float64)
        same = ((cg > 0) == (ora.coeffs > 0)).all(1)
        m = ora.coeff_sigma[same] > 1e-6
        parity = {"pixels": int(len(sel)), "max_abs_da": float(np.abs(cg - ora.coeffs).max()),
                  "max_rel_resid": float((np.abs(rg - ora.resid) / ora.resid).max()),
                  "max_rel_sigma_same_support": float((np.abs(sg[same] - ora.coeff_sigma[same])[m] / ora.coeff_sigma[same][m]).max()),
                  "support_mismatches": int((~same).sum())}
        if not args.no_cpu_baseline:
            n = 262144 if args.sample is None else args.sample
            n = min(n, N)
            cores = host_threads()
            t0 = time.perf_counter()
            oracle.solve(A, Yh.numpy()[:n], Sh.numpy()[:n], nthreads=cores)
            dt = time.perf_counter() - t0
            cpu_baseline = {"value": n / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
                            "sample": f"first {n} pixels of the same workload, one pass, {dt:.1f} s"}

    # ---- extra report keys (rank 0, after the timed region): the other BASELINE.json configs through the any-size
    #      kernels, and the NEXT-row options on the config-4 library -- device-resident, CUDA events, 3 calls each
    extras = None
    if rank == 0 and not args.no_extras:
        extras = run_extras(linmin, torch, dev, A, Yd, Sd)

    # ---- end-to-end: host buffers through linmin_unmix_host (H2D + kernels + D2H per step)
    e2e = None
    if args.e2e_steps > 0:
        Ah = torch.from_numpy(A)
        hout = dict(coeffs=torch.empty((N, R), dtype=torch.float32, pin_memory=True),
                    coeff_sigma=torch.empty((N, R), dtype=torch.float32, pin_memory=True),
                    resid=torch.empty((N,), dtype=torch.float32, pin_memory=True))
        # warm-up call over enough pixels to run all three buffer sets of the host pipeline at their full chunk size
        nw = min(N, 8 * CUBE)
        linmin.unmix_host(Ah, Yh[:nw], Sh[:nw], out=dict(coeffs=hout["coeffs"][:nw], coeff_sigma=hout["coeff_sigma"][:nw], resid=hout["resid"][:nw]))
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            linmin.unmix_host(Ah, Yh, Sh, out=hout)
        barrier()
        dt = (time.perf_counter() - t0) / args.e2e_steps
        dt = max_over_ranks(dt, dev)
        e2e = {"value": world * N / dt, "unit": UNIT, "h2d_bytes_per_step": int(2 * N * L * 4 + L * R * 4),
               "d2h_bytes_per_step": int(N * (2 * R + 1) * 4), "ms_per_step": dt * 1e3, "steps": args.e2e_steps,
               "api": "linmin_unmix_host (pinned host buffers, 3-deep chunk pipeline)"}
        if rank == 0:
            same_bits = bool(np.array_equal(hout["coeffs"].numpy()[sel], out["coeffs"][sel_t].cpu().numpy()))
            e2e["matches_device_path_bitwise"] = same_bits

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": f"throughput (BASELINE.json configs[4]): L={L}, R={R}, N={N} per GPU "
                                   f"({n_cubes} OMEGA-like cubes of 131072 px), per-pixel sigma (N x L)",
                       "L": L, "R": R, "N_per_gpu": N, "sigma": "per-pixel",
                       "l2_policy": "inputs (2 x %.1f GB) larger than L2, no flush needed" % (N * L * 4 / 1e9),
                       "precompute": "library handle created once outside the timed region (once-per-library step a0)",
                       "arithmetic": "fp32 IPLS; fp64 k x k factor and residual in the finish",
                       "host_generation_s": t_gen},
            "shared_sigma": {"value": world * N / (ms_shared * 1e-3), "unit": UNIT, "ms_per_step": ms_shared,
                             "what": "same step with ONE shared sigma[L] (sigma_pixel_stride = 0), device-resident"},
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
            "cpu_baseline": cpu_baseline, "parity_sample": parity, "histograms": histograms, "extras": extras,
        }
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
