#!/usr/bin/env python
"""bench.py -- headline benchmark of libtina: fused PFB at P=1024, M=16 (BASELINE.json config 4).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload c4|c5|c5bf16|c5fp16|c2|c3|c3multi|c1|c4fir|c4fft|c5fft|peaks]

One "step" = one pass of the whole hot path (subfilter stage + DFT contraction, one
tina_pfb_batched call) over one batch of synthetic input shaped like config 4:
8 streams x 8192 spectra x 1024 channels, 16 taps (537.9 MB in, 536.9 MB out -- both larger
than the 126 MB L2, so consecutive steps cannot be served from cache; no explicit flush).
Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for the definitions.
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

import tina_inputs as ti  # noqa: E402

METRIC = "pfb_input_gsamples_per_s"
UNIT = "GSamples/s"
FALLBACK_PEAKS = {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            d = json.load(fh)
        d["_source"] = "measured"
        return d
    d = dict(FALLBACK_PEAKS)
    d["_source"] = "fallback"
    return d


def workload_spec(name: str):
    """(kind, dict) for each BASELINE.json config; c4 is the headline."""
    if name == "c4":
        return dict(call="pfb", P=1024, M=16, S=8, F=8192, real=False, prec=0)
    if name == "c5":
        return dict(call="pfb", P=4096, M=8, S=1, F=32761, real=True, prec=0)
    if name == "c5bf16":
        return dict(call="pfb", P=4096, M=8, S=1, F=32761, real=True, prec=1)
    if name == "c5fp16":
        return dict(call="pfb", P=4096, M=8, S=1, F=32761, real=True, prec=2)
    if name == "c1":
        return dict(call="pfb", P=16, M=4, S=1, F=4096, real=False, prec=0)
    if name == "c4fir":   # subfilter stage only (Fig. 3 left column), config-4 shape
        return dict(call="pfb_fir", P=1024, M=16, S=8, F=8192, real=False, prec=0)
    if name == "c4fft":   # config-4 shape through the factorised (32 x 32 Cooley-Tukey) Fourier stage: same result,
        # HBM / FMA bound instead of tensor bound; reported separately from the dense-contraction headline
        return dict(call="pfb_fft", P=1024, M=16, S=8, F=8192, real=False, prec=0)
    if name == "c5fft":   # config 5 (real, P = 4096 = 64 x 64) through the factorised Fourier stage
        return dict(call="pfb_fft", P=4096, M=8, S=1, F=32761, real=True, prec=0)
    if name == "c2":
        return dict(call="dft", B=65536, N=256)
    if name == "c3":
        return dict(call="fir", C=64, L=1 << 20, K=64)
    if name == "c3multi":   # config-3 shape with one tap vector per channel (tina_fir_multi)
        return dict(call="fir_multi", C=64, L=1 << 20, K=64)
    if name == "peaks":     # measured arithmetic ceilings (tina_probe_peak), no workload
        return dict(call="peaks")
    raise SystemExit(f"unknown workload {name}")


def roof_floors(issued_flops, algorithmic_bytes, tensor_tflops, hbm_gbs):
    """Time floors (seconds) of one step under the two roofs: issued tensor flops at `tensor_tflops`, algorithmic bytes
    at `hbm_gbs`.  The larger one is the roof that binds."""
    return issued_flops / (tensor_tflops * 1e12), algorithmic_bytes / (hbm_gbs * 1e9)


def useful_flops_and_bytes(w):
    """Algorithmic flops (DFT contraction, the dominant kernel's tensor work) and HBM bytes
    per step -- SURVEY.md section 8(d) / DESIGN.md "Algorithmic work"."""
    if w["call"] == "pfb_fir":
        P, M, S, F = w["P"], w["M"], w["S"], w["F"]
        esz = 4 if w["real"] else 8
        return S * F * P * (esz // 4) * 2.0 * M, float(S * (F + M - 1) * P * esz + S * F * P * esz + P * M * 4), S * (F + M - 1) * P, S * F
    if w["call"] == "pfb_fft":
        P, M, S, F = w["P"], w["M"], w["S"], w["F"]
        if w["real"]:    # stage 1: 2 P sqrt(P) real MACs, stage 2: 2 x 2 x (P / 2) sqrt(P)
            return S * F * 8.0 * P * 64, float(S * (F + M - 1) * P * 4 + S * F * (P // 2 + 1) * 8 + P * M * 4), S * (F + M - 1) * P, S * F
        return S * F * 8.0 * P * 64, float(S * (F + M - 1) * P * 8 + S * F * P * 8 + P * M * 4), S * (F + M - 1) * P, S * F
    if w["call"] == "pfb":
        P, M, S, F = w["P"], w["M"], w["S"], w["F"]
        frames = S * F
        if w["real"]:
            flops = frames * (2.0 * P * P + 4.0 * P)
            byts = S * (F + M - 1) * P * 4 + frames * (P // 2 + 1) * 8 + P * M * 4
        else:
            flops = frames * 8.0 * P * P
            byts = S * (F + M - 1) * P * 8 + frames * P * 8 + P * M * 4
        samples = S * (F + M - 1) * P
        return flops, float(byts), samples, frames
    if w["call"] == "dft":
        B, N = w["B"], w["N"]
        return B * 8.0 * N * N, B * N * 16.0, B * N, B
    C, L, K = w["C"], w["L"], w["K"]
    return C * (L - K + 1) * 2.0 * K, C * L * 4.0 + C * (L - K + 1) * 4.0, C * L, C


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-i", str(self.index), "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append((time.time(), ln.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        sm, smax, reasons, watts = [], None, set(), []
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.1] or [r for (_, r) in self.rows]
        for r in rows:
            f = [c.strip() for c in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax = float(f[1])
            except ValueError:
                continue
            try:
                watts.append(float(f[2]))
            except ValueError:
                pass
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax,
                "reasons": sorted(reasons), "samples": len(sm),
                "power_w_median": float(np.median(watts)) if watts else None, "power_w_max": float(max(watts)) if watts else None}


def make_inputs(w, seed_offset: int = 0):
    """Seeded synthetic host arrays for the workload (tina_inputs recipes)."""
    if w["call"] in ("pfb", "pfb_fir", "pfb_fft"):
        if (w["P"], w["M"], w["real"]) == (1024, 16, False):
            case = ti.pfb_case(1024, 16, w["F"], streams=w["S"], seed=ti.SEED_BASE + 4 + 100 * seed_offset,
                               tones=3, name="c4")
        else:
            idx = 5 if w["real"] else 1
            case = ti.pfb_case(w["P"], w["M"], w["F"], real=w["real"], streams=w["S"],
                               seed=ti.SEED_BASE + idx + 100 * seed_offset)
        return case
    if w["call"] == "dft":
        return ti.config2(w["B"], w["N"])
    return ti.config3(w["C"], w["L"], w["K"])   # fir and fir_multi


def cpu_oracle_rate(w, budget_s: float = 15.0):
    """Time the float64 oracle, as it stands, on a bounded sample of the workload.
    Returns (GSamples/s, cores, sample description, seconds)."""
    import oracle
    oracle.build()
    cores = oracle.num_threads()
    if w["call"] in ("pfb", "pfb_fir", "pfb_fft"):
        P, M = w["P"], w["M"]
        probe = max(cores, 8)
        case = ti.pfb_case(P, M, probe, real=w["real"], seed=1)
        t0 = time.perf_counter(); oracle.pfb(case.x[0], P, M, case.window); dt = time.perf_counter() - t0
        n = int(min(max(probe, budget_s / max(dt / probe, 1e-9)), 4096))
        n = max(cores, n - n % cores)
        case = ti.pfb_case(P, M, n, real=w["real"], seed=2)
        t0 = time.perf_counter(); oracle.pfb(case.x[0], P, M, case.window); dt = time.perf_counter() - t0
        return n * P / dt / 1e9, cores, f"{n} frames of one stream (P={P}, M={M}), float64 direct sums", dt
    if w["call"] == "dft":
        N = w["N"]; n = 4096
        x = ti.config2(n, N)
        t0 = time.perf_counter(); oracle.dft(x); dt = time.perf_counter() - t0
        return n * N / dt / 1e9, cores, f"{n} signals of N={N}", dt
    C, L, K = 8, 1 << 20, w["K"]
    x, taps, _ = ti.config3(C, L, K)
    if w["call"] == "fir_multi":
        tm = np.ascontiguousarray(np.tile(taps, (C, 1)))
        t0 = time.perf_counter(); oracle.fir_multi(x, tm); dt = time.perf_counter() - t0
        return C * L / dt / 1e9, cores, f"{C} channels of L={L}, K={K}, per-channel taps", dt
    t0 = time.perf_counter(); oracle.fir(x, taps); dt = time.perf_counter() - t0
    return C * L / dt / 1e9, cores, f"{C} channels of L={L}, K={K}", dt


def cpu_numpy_rate(w, repeats: int = 5, budget_s: float = 25.0):
    """The NumPy-style vectorised CPU PFB of oracle/numpy_pfb.py (the stand-in for the paper's "naive
    implementation written in NumPy (on CPU)"; protocol PAPER.md:208, :214: data resident,
    best of `repeats`), complex64 / float32, numpy.fft for the Fourier stage.  c4 is timed as ONE stream
    (the eight streams are independent and identical in cost; the rate is per sample, so no scaling is
    needed).  Returns a dict, or None for workloads it does not define (FIR)."""
    from oracle import numpy_pfb
    if w["call"] == "dft":
        x = ti.config2(min(w["B"], 16384), w["N"])
        fn, n_samp, sample = (lambda: np.fft.ifft(np.fft.fft(x, axis=1), axis=1).astype(np.complex64)), x.size, \
            f"{x.shape[0]} signals of N={w['N']}, numpy.fft forward + inverse"
    elif w["call"] in ("pfb", "pfb_fft", "pfb_fir"):
        P, M, F = w["P"], w["M"], w["F"]
        case = ti.pfb_case(P, M, F, real=w["real"], streams=1, seed=3)
        x, win = case.x[0], case.window
        if w["call"] == "pfb_fir":
            fn = lambda: numpy_pfb.pfb_subfilter(x, P, M, win)
        else:
            fn = lambda: numpy_pfb.pfb(x, P, M, win)
        n_samp, sample = x.size, f"one stream of {F} frames (P={P}, M={M}), complex64/float32, numpy.fft"
    else:
        return None
    best, t_all = None, time.perf_counter()
    for i in range(repeats):
        t0 = time.perf_counter(); fn(); dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
        if time.perf_counter() - t_all > budget_s:
            break
    try:
        from threadpoolctl import threadpool_info
        blas_threads = max([d.get("num_threads", 1) for d in threadpool_info()] or [1])
    except Exception:
        blas_threads = None
    return {"value": n_samp / best / 1e9, "unit": UNIT, "kind": "numpy", "cores": 1,
            "host_cores": len(os.sched_getaffinity(0)), "blas_threads": blas_threads,
            "numpy": np.__version__, "best_of": i + 1, "seconds": best, "sample": sample,
            "note": "numpy.fft (pocketfft) and the slice multiply-accumulates run on one thread"}


def tina_env():
    """Every TINA_* variable set in the environment (recorded in the JSON line)."""
    return {k: v for k, v in sorted(os.environ.items()) if k.startswith("TINA_")}


REFUSED_ENV = ("TINA_DEBUG_SKIP", "TINA_KSPLIT", "TINA_A_SLOTS", "TINA_B_ENTRIES", "TINA_CL4", "TINA_PROF", "TINA_BUILD_DEV")


def run_peaks(args):
    """--workload peaks: bare-loop ceilings of this device (burst = ~20 ms region, sustained = ~2 s)."""
    import torch
    import paper_2408_16551_b200 as tina
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    names = {0: "ffma_fp32", 1: "ffma2_fp32", 2: "tcgen05_tf32", 3: "tcgen05_bf16", 4: "tcgen05_bf16_n128", 5: "tcgen05_bf16_n64"}
    out = {}
    for which, name in names.items():
        base = 4096 if which < 2 else 2048
        tf, ms = tina.probe_peak(which, base)
        per_ms = base / ms
        burst = max(tina.probe_peak(which, int(per_ms * 20))[0] for _ in range(5))
        sampler = ClockSampler(0); sampler.start(); time.sleep(0.1); t0 = time.time()
        sus, sus_ms = tina.probe_peak(which, int(per_ms * 2000))
        clocks = sampler.stop(t0, time.time())
        out[name] = {"burst_tflops": burst, "sustained_tflops": sus, "sustained_ms": sus_ms, "clocks": clocks}
    print(json.dumps({"metric": "measured_peaks", "peaks": out, "measured_peaks_json": load_peaks()}), flush=True)


def run_reference(args, w):
    """--impl reference: the oracle (oracle/, as it stands) on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    flops, byts, samples, frames = useful_flops_and_bytes(w)
    rates, secs = [], []
    budget = max(0.3, min(15.0, 100.0 / max(args.steps + args.warmup, 1)))   # whole run: about two minutes
    for i in range(args.warmup + args.steps):
        r, cores, sample, dt = cpu_oracle_rate(w, budget_s=budget)
        if i >= args.warmup:
            rates.append(r); secs.append(dt)
    value = float(np.mean(rates))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(secs)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "gpu_launches": 0,
        "config": config_of(args.workload, w),
        "run": {"note": "each step = a bounded sample of the workload run through the float64 oracle (host cores, no GPU)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


L2_BYTES = 126e6


def l2_plan(w):
    """(set_bytes, rotate, n_sets): working sets below ~1 GB are timed cold by rotating over distinct buffer sets."""
    _, byts, _, _ = useful_flops_and_bytes(w)
    set_bytes = 3 * 8.0 * w["B"] * w["N"] if w["call"] == "dft" else byts      # dft: x, out and back buffers
    rotate = set_bytes < 8 * L2_BYTES
    n_sets = int(min(512, max(4, np.ceil(2.5 * L2_BYTES / set_bytes)))) if rotate else 1
    return set_bytes, rotate, n_sets


def config_of(workload, w):
    """The `config` object of the JSON line: the workload and how consecutive steps are kept out of L2.  Identical for
    both arms (`--impl ours|reference`); everything that describes the RUN rather than the workload goes to `run`."""
    set_bytes, rotate, n_sets = l2_plan(w)
    return {"workload": workload, **{k: v for k, v in w.items() if k != "call"},
            "l2": (f"cold: rotating over {n_sets} distinct buffer sets ({n_sets * set_bytes / 1e6:.0f} MB > 2x L2); the hot "
                   "(same buffers) timing is in `hot`") if rotate else
                  "inputs and outputs each exceed the 126 MB L2; no explicit flush"}


def run_ours(args, w):
    import torch
    import torch.distributed as dist
    import paper_2408_16551_b200 as tina
    from paper_2408_16551_b200 import shard

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- libtina has no CPU fallback")
    env = tina_env()
    refused = [k for k in REFUSED_ENV if k in os.environ]
    tina.lib()
    if refused or tina.build_is_dev():
        # knobs that skip work or change the accuracy contract: a number measured with them is not a measurement
        print(f"bench.py: refusing to run with {refused or 'a -DTINA_DEV build of libtina.so'}", file=sys.stderr)
        raise SystemExit(2)
    torch.cuda.set_device(local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    flops, byts, samples, frames = useful_flops_and_bytes(w)
    peaks = load_peaks()
    stream = torch.cuda.current_stream()

    # ---- inputs resident in HBM (each rank its own seeded batch: frames are independent, so
    #      ranks shard the units with no data-path collective -> weak scaling) --------------
    data = make_inputs(w, seed_offset=rank)
    x_host = w_host = None
    NK = None

    def make_set():
        """One set of device buffers + the step that runs on them."""
        nonlocal x_host, w_host, NK
        if w["call"] == "pfb":
            x_host, w_host = torch.from_numpy(data.x), torch.from_numpy(data.window)
            xd, wd = x_host.cuda(), w_host.cuda()
            NK = w["P"] // 2 + 1 if w["real"] else w["P"]
            out = torch.empty((w["S"], w["F"], NK), dtype=torch.complex64, device="cuda")
            return lambda: tina.pfb(xd, w["P"], w["M"], wd, prec=w["prec"], out=out)
        if w["call"] == "pfb_fft":
            xd, wd = torch.from_numpy(data.x).cuda(), torch.from_numpy(data.window).cuda()
            out = torch.empty((w["S"], w["F"], w["P"] // 2 + 1 if w["real"] else w["P"]), dtype=torch.complex64, device="cuda")
            return lambda: tina.pfb_fft(xd, w["P"], w["M"], wd, out=out)
        if w["call"] == "pfb_fir":
            xd, wd = torch.from_numpy(data.x).cuda(), torch.from_numpy(data.window).cuda()
            out = torch.empty((w["S"], w["F"], w["P"]), dtype=xd.dtype, device="cuda")
            return lambda: tina.pfb_fir(xd, w["P"], w["M"], wd, out=out)
        if w["call"] == "dft":
            xd = torch.from_numpy(data).cuda()
            out = torch.empty_like(xd); back = torch.empty_like(xd)
            def step():
                tina.dft(xd, out=out); tina.dft(out, inverse=True, out=back)
            return step
        xh, taps, _ = data
        xd = torch.from_numpy(xh).cuda()
        out = torch.empty((w["C"], w["L"] - w["K"] + 1), dtype=torch.float32, device="cuda")
        if w["call"] == "fir_multi":
            td = torch.from_numpy(np.ascontiguousarray(np.tile(taps, (w["C"], 1)))).cuda()
            return lambda: tina.fir_multi(xd, td, out=out)
        td = torch.from_numpy(taps).cuda()
        return lambda: tina.fir(xd, td, out=out)

    if w["call"] == "dft":
        flops *= 2; byts *= 2
    # Working sets smaller than ~8x L2 are timed twice: HOT (the same buffers every step) and COLD (rotating
    # over >= 4 distinct buffer sets totalling > 2x L2, so no step finds its data in L2).  HBM fractions and
    # `value` are quoted from the cold run.
    set_bytes, rotate, n_sets = l2_plan(w)
    steps_of = [make_set() for _ in range(n_sets)]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(n_steps, pick):
        """CUDA events on the launching stream: whole region + every step."""
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_steps)]
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.time()
        e0.record(stream)
        for i, (a, b) in enumerate(evs):
            a.record(stream); pick(i)(); b.record(stream)
        e1.record(stream)
        barrier()
        t1 = time.time()
        per = [a.elapsed_time(b) for a, b in evs]
        return e0.elapsed_time(e1), per, t0, t1

    n_warm = max(args.warmup, 3)
    for i in range(max(n_warm, n_sets)):
        steps_of[i % n_sets]()
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.15)
    launches0 = tina.launch_count()
    total_ms, per_step, t_wall0, t_wall1 = timed(args.steps, lambda i: steps_of[i % n_sets])
    launches = tina.launch_count() - launches0
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    kern_ms, kern_min = float(np.mean(per_step)), float(np.min(per_step))
    total_ms = shard.max_over_ranks(total_ms, device="cuda")
    ms_per_step = total_ms / args.steps
    value = world * samples / (ms_per_step * 1e-3) / 1e9
    hot = None
    if rotate:
        h_total, h_per, _, _ = timed(args.steps, lambda i: steps_of[0])
        hot = {"ms_per_step": h_total / args.steps, "ms_mean": float(np.mean(h_per)), "ms_min": float(np.min(h_per)),
               "value": world * samples / (h_total / args.steps * 1e-3) / 1e9}
    # launch-latency-bound workloads (c1: a 1 MB problem): microseconds per call of a back-to-back burst of calls on the
    # same buffers, host clock around the burst including the final synchronise (no per-step events in between)
    call_us = None
    if set_bytes < 16e6:
        n_b2b = 2000
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_b2b):
            steps_of[0]()
        torch.cuda.synchronize()
        call_us = (time.perf_counter() - t0) / n_b2b * 1e6
    issued_ratio = tina.last_issued_ratio() if hasattr(tina, "last_issued_ratio") else None
    variant = tina.last_kernel() if hasattr(tina, "last_kernel") else None

    # ---- e2e: host buffers through the C ABI (H2D + kernel + D2H inside the timed region) --
    e2e = None
    if w["call"] == "pfb" and not args.profile:
        xp, wp = x_host.pin_memory(), w_host.pin_memory()
        outp = torch.empty((w["S"], w["F"], NK), dtype=torch.complex64, pin_memory=True)
        n_e2e = max(2, min(args.steps, 5))
        tina.pfb_host(xp, w["P"], w["M"], wp, prec=w["prec"], out=outp)      # warm-up (allocates staging)
        barrier()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            tina.pfb_host(xp, w["P"], w["M"], wp, prec=w["prec"], out=outp)  # synchronous call
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) / n_e2e
        dt = shard.max_over_ranks(dt, device="cuda")
        e2e = {"value": world * samples / dt / 1e9, "unit": UNIT,
               "h2d_bytes_per_step": int(xp.numel() * xp.element_size() + wp.numel() * 4),
               "d2h_bytes_per_step": int(outp.numel() * 8), "ms_per_step": dt * 1e3, "steps": n_e2e}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    tensor_bound = w["call"] in ("pfb", "dft") and tina.last_path() == 2
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath):
        with open(tpath) as fh:
            traffic = json.load(fh).get(args.workload)
    # Which measured peak applies: the burst figure for a short, unthrottled region; the sustained one when the
    # region is long or the power cap was active during it.  BOTH fractions are printed every time.
    throttled = bool(clocks) and ("sw_power_cap" in clocks.get("reasons", []) or
                                  (clocks.get("sm_mhz") and clocks.get("sm_max_mhz") and clocks["sm_mhz"] < 0.85 * clocks["sm_max_mhz"]))
    sustained = total_ms > 1500.0 or throttled
    if tensor_bound:
        pk_b, pk_s = peaks["bf16_tflops"], peaks["bf16_tflops_sustained"]
        peak = pk_s if sustained else pk_b
        achieved = flops / (kern_ms * 1e-3) / 1e12
        passes = 3 if w.get("prec", 0) == 0 else 1
        # issued tensor flops per useful flop: `passes` bf16 products per useful one (error-compensated bf16x3),
        # times the fraction of the Fourier matrix the kernel contracts against (0.5 when every distinct column
        # pair k / P-k is contracted once; reported by the library for the kernel that ran)
        ratio = passes * (issued_ratio if issued_ratio else 1.0)
        roof = {"bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": traffic, "peak_source": f"{peaks['_source']} bf16 {'sustained' if sustained else 'burst'}",
                "useful_flops": flops, "issued_flops": flops * ratio, "issued_passes": passes,
                "issued_per_useful": ratio, "frac_useful_ceiling": 1.0 / ratio,
                "frac_useful": achieved / peak, "frac_issued": ratio * achieved / peak, "issued_frac": ratio * achieved / peak,
                "peak_burst": pk_b, "peak_sustained": pk_s,
                "frac_useful_burst": achieved / pk_b, "frac_useful_sustained": achieved / pk_s,
                "frac_issued_burst": ratio * achieved / pk_b, "frac_issued_sustained": ratio * achieved / pk_s,
                "hbm_gbs_achieved": byts / (kern_ms * 1e-3) / 1e9, "hbm_frac": byts / (kern_ms * 1e-3) / 1e9 / peaks["hbm_gbs"]}
        # Which roof binds: the larger of the two time floors (ISSUED tensor flops at the burst peak, algorithmic bytes
        # at the measured copy bandwidth).  A dense contraction whose arithmetic intensity is below the machine balance
        # (c2: N = 256, 8 N^2 flops x 1.5 issued per 16 N bytes = 192 flop/B against 1662 / 6.55 = 254) sits on the
        # memory side of the ridge: its line reports the HBM fraction as `frac` and keeps the tensor figures beside it.
        t_tensor, t_hbm = roof_floors(flops * ratio, byts, pk_b, peaks["hbm_gbs"])
        roof["floor_ms"] = {"tensor_issued_burst": t_tensor * 1e3, "hbm": t_hbm * 1e3}
        if t_hbm > t_tensor:
            tensor_side = {k: roof[k] for k in ("achieved", "peak", "unit", "frac", "peak_source")}
            roof.update({"bound": "hbm", "achieved": roof["hbm_gbs_achieved"], "peak": peaks["hbm_gbs"], "unit": "GB/s",
                         "frac": roof["hbm_frac"], "peak_source": f"{peaks['_source']} copy", "algorithmic_bytes": byts,
                         "tensor": tensor_side})
    else:
        achieved = byts / (kern_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": achieved / peaks["hbm_gbs"], "traffic": traffic, "peak_source": f"{peaks['_source']} copy",
                "algorithmic_bytes": byts, "frac_nominal_8tbs": achieved / 8000.0}
    roof["kernel_ms"] = kern_ms
    roof["kernel_ms_min"] = kern_min
    roof["kernel"] = variant

    cpu_val, cores, sample, _ = cpu_oracle_rate(w) if (world == 1 and not args.profile) else (None, None, None, None)
    cpu_np = cpu_numpy_rate(w) if (world == 1 and not args.profile) else None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": n_warm,
        "ms_per_step": ms_per_step, "ms_mean": kern_ms, "ms_min": kern_min,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": ("bf16x3->f32" if w.get("prec", 0) == 0 else ("bf16" if w.get("prec", 0) == 1 else "f16")) if (tensor_bound or w["call"] == "pfb_fft") else "f32",
        "data": "synthetic", "spectra_per_s": world * frames / (ms_per_step * 1e-3),
        "config": config_of(args.workload, w),
        "run": {"path": {0: "none", 1: "cuda-core", 2: "tcgen05"}[tina.last_path()],
                "parallelism": f"frame-sharded replicas x{world}, no collective"},
        "roofline": roof, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "tina_env": env,
    }
    if args.profile:
        line["profile_run"] = True
    if hot is not None:
        line["hot"] = hot
    if call_us is not None:
        line["hot"]["back_to_back_us_per_call"] = call_us
    if cpu_val is not None:
        line["cpu_baseline"] = {"value": cpu_val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                                "note": "float64 direct sums (the parity oracle): not a performance baseline"}
    if cpu_np is not None:
        line["cpu_baseline_numpy"] = cpu_np
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4")
    ap.add_argument("--profile", action="store_true",
                    help="profiling run (under ncu): skip the CPU baselines and the e2e leg; the line is not a bench value")
    args = ap.parse_args()
    w = workload_spec(args.workload)
    if w["call"] == "peaks":
        return run_peaks(args)
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
