#!/usr/bin/env python
"""bench_probes.py -- measurement helpers used by bench.py and by the recipes under profiles/ (NOT part of the product
library: the kernels live in bench_probes.cu and build into libms_bench_probes.so beside this file).

    python bench_probes.py fp64              # sustained DFMA rate, >= 2 s per form, median and best
    python bench_probes.py issue-model       # 4 DFMA + K other instructions per loop: which pipes issue beside the fp64 pipe
    python bench_probes.py unweight-density  # ms_unweight alone at acceptance rates 1e-4 .. 1
    python bench_probes.py chili             # ms_chili n = 3, 4, 6 at 2^24 events (CUDA events; ncu-able)
    python bench_probes.py vegas-map         # stand-alone ms_vegas_map, forward and inverse, at the cfg-5 shape
    python bench_probes.py entry-points      # the other stand-alone section-8(b) calls at 2^24 events, each against its own bytes
    python bench_probes.py next-rows         # observables, cuts, histograms, grid accumulation, ... (the NEXT rows), likewise

Each prints one JSON line.
"""
from __future__ import annotations

import ctypes as C
import json
import os
import shutil
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(ROOT, "bench_probes.cu")
LIB = os.path.join(ROOT, "libms_bench_probes.so")
_lib = None


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = [nvcc, "-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC",
           "-shared", SRC, "-o", tmp]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    os.replace(tmp, LIB)
    return LIB


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, i64, i = C.c_void_p, C.c_int64, C.c_int
        L.probe_dfma.argtypes = [i, i, vp, vp]
        L.probe_dfma3.argtypes = [i, i, vp, vp]
        L.probe_write.argtypes = [i64, i, vp, i64, vp]
        L.probe_mix.argtypes = [i, i, i, i, i, vp, vp]
        L.probe_dfma_latency.argtypes = [i, i, i, vp, vp]
        _lib = L
    return _lib


def _check(rc: int, what: str) -> None:
    if rc != 0:
        raise RuntimeError("%s: cudaError %d" % (what, rc))


def fp64_rate(torch, seconds: float = 2.0, three_regs: bool = False) -> dict:
    """DFMA instructions/s sustained for `seconds` ("dependent-free DFMA loop sustained for
    seconds"): back-to-back launches of 8 independent chains per thread, one CUDA-event pair per launch; the MEDIAN
    launch is the figure the rooflines use, the best one is reported beside it."""
    import numpy as np
    fn = lib().probe_dfma3 if three_regs else lib().probe_dfma
    s = torch.cuda.current_stream().cuda_stream
    sms = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    blocks, iters = sms * 8, 1 << 14
    sink = torch.empty(blocks * 256, dtype=torch.float64, device="cuda")
    inst = blocks * 256 * iters * 8
    _check(fn(blocks, iters, sink.data_ptr(), s), "probe_dfma")
    torch.cuda.synchronize()
    rates, t_end = [], time.perf_counter() + seconds
    while time.perf_counter() < t_end or len(rates) < 5:
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(9)]
        evs[0].record()
        for k in range(8):                               # 8 launches in flight: no host gap between them
            _check(fn(blocks, iters, sink.data_ptr(), s), "probe_dfma")
            evs[k + 1].record()
        evs[-1].synchronize()
        rates += [inst / (evs[k].elapsed_time(evs[k + 1]) * 1e-3) for k in range(8)]
    return {"median": float(np.median(rates)), "best": float(np.max(rates)), "launches": len(rates),
            "seconds": seconds, "form": "a*b+c, three registers" if three_regs else "a*const+const"}


def write_stream_gbs(torch, N: int, rows: int, out, ld: int, reps: int = 10) -> float:
    """GB/s of the generation kernel's store pattern with no arithmetic (rows x N doubles, streaming stores)."""
    s = torch.cuda.current_stream().cuda_stream
    _check(lib().probe_write(N, rows, out.data_ptr(), ld, s), "probe_write")
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(reps):
        _check(lib().probe_write(N, rows, out.data_ptr(), ld, s), "probe_write")
    ev1.record()
    ev1.synchronize()
    return 8.0 * rows * N * reps / (ev0.elapsed_time(ev1) * 1e-3) / 1e9


def imad_wide_rate(torch, reps: int = 5) -> float:
    """32x32 -> 64-bit multiply-adds (IMAD.WIDE.U32, the multiply of a Philox round) per second, thread-level like the
    DFMA figure: 8 independent chains per thread, all SMs busy with 8 warps per scheduler."""
    s = torch.cuda.current_stream().cuda_stream
    sms = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    blocks, iters = sms * 4, 1 << 13
    sink = torch.empty(blocks * 256, dtype=torch.float64, device="cuda")
    _check(lib().probe_mix(3, 8, 0, blocks, iters, sink.data_ptr(), s), "probe_mix")
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(reps):
        _check(lib().probe_mix(3, 8, 0, blocks, iters, sink.data_ptr(), s), "probe_mix")
    ev1.record()
    ev1.synchronize()
    return blocks * 256 * iters * 8 * reps / (ev0.elapsed_time(ev1) * 1e-3)


MIX_KINDS = {1: "LOP3", 2: "IMAD", 3: "IMAD.WIDE.U32", 4: "FFMA", 5: "MUFU.RCP (fp32)", 6: "F2I.F64 + I2F.F64 (pair)",
             7: "LDS.64", 8: "IADD3", 9: "MUFU.RCP64H"}


def issue_model(torch) -> dict:
    """Cycles per loop iteration and warp scheduler (4 per SM) of [nd DFMA + k x kind], all SMs busy with 8 warps per
    scheduler, at the SM clock nvidia-smi reports under this load."""
    s = torch.cuda.current_stream().cuda_stream
    props = torch.cuda.get_device_properties(torch.cuda.current_device())
    sms = props.multi_processor_count
    blocks, iters = sms * 4, 1 << 13                      # 4 blocks x 8 warps per SM = 8 warps per scheduler
    sink = torch.empty(blocks * 256, dtype=torch.float64, device="cuda")

    def cycles(kind, k, nd):
        _check(lib().probe_mix(kind, k, nd, blocks, iters, sink.data_ptr(), s), "probe_mix")
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for _ in range(5):
            _check(lib().probe_mix(kind, k, nd, blocks, iters, sink.data_ptr(), s), "probe_mix")
        ev1.record()
        ev1.synchronize()
        t = ev0.elapsed_time(ev1) * 1e-3 / 5
        warp_iters_per_sched = blocks * 8 * iters / (sms * 4)
        return t * clock_hz / warp_iters_per_sched

    try:
        q = subprocess.run(["nvidia-smi", "--query-gpu=clocks.max.sm", "--format=csv,noheader,nounits", "-i", "0"],
                           capture_output=True, text=True).stdout.strip().splitlines()[0]
        clock_hz = float(q) * 1e6
    except Exception:
        clock_hz = 1965e6
    out = {"clock_mhz_assumed": clock_hz / 1e6, "unit": "cycles per iteration per scheduler (includes ~2-3 loop instructions)",
           "dfma4_alone": cycles(0, 0, 4), "rows": []}
    for kind, name in MIX_KINDS.items():
        out["rows"].append({"kind": name, "k4_alone": cycles(kind, 4, 0), "k8_alone": cycles(kind, 8, 0),
                            "dfma4_plus_k2": cycles(kind, 2, 4), "dfma4_plus_k4": cycles(kind, 4, 4),
                            "dfma4_plus_k8": cycles(kind, 8, 4)})
    return out


def dfma_latency(torch) -> dict:
    """Cycles per DFMA of ONE warp per SM with 1, 2, 4, 8 independent chains per thread (dependent-issue latency and the
    parallelism needed to hide it), at the maximum SM clock."""
    s = torch.cuda.current_stream().cuda_stream
    sms = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    iters = 1 << 16
    sink = torch.empty(sms * 32, dtype=torch.float64, device="cuda")
    try:
        q = subprocess.run(["nvidia-smi", "--query-gpu=clocks.max.sm", "--format=csv,noheader,nounits", "-i", "0"],
                           capture_output=True, text=True).stdout.strip().splitlines()[0]
        clock_hz = float(q) * 1e6
    except Exception:
        clock_hz = 1965e6
    out = {"clock_mhz_assumed": clock_hz / 1e6}
    for ch in (1, 2, 4, 8):
        _check(lib().probe_dfma_latency(ch, sms, iters, sink.data_ptr(), s), "probe_dfma_latency")
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for _ in range(5):
            _check(lib().probe_dfma_latency(ch, sms, iters, sink.data_ptr(), s), "probe_dfma_latency")
        ev1.record()
        ev1.synchronize()
        out["cycles_per_dfma_%d_chains" % ch] = ev0.elapsed_time(ev1) * 1e-3 / 5 * clock_hz / (iters * ch)
    return out


def unweight_density(torch, steps: int = 20, warmup: int = 3) -> dict:
    """ms_unweight alone on 2^24 synthetic weights x 24 momentum rows at several acceptance rates -- the unweighting
    efficiencies a production run sees after grid adaptation rather than the 1e-4 of the seeded-grid
    workloads.  Weights w = u^(1/f - 1) with w_max = 1 have <w>/w_max = f."""
    sys.path.insert(0, ROOT)
    import ms_inputs
    import paper_2602_06895_b200 as ms
    ms.lib()
    dev = torch.device("cuda", torch.cuda.current_device())
    N, rows = 1 << 24, 24
    f64 = dict(dtype=torch.float64, device=dev)
    gen = torch.Generator(device=dev)
    gen.manual_seed(5)
    p = torch.rand((rows, N), generator=gen, **f64)
    idx = torch.empty(N, dtype=torch.int64, device=dev)
    w_out, rows_out = torch.empty(N, **f64), torch.empty((rows, N), **f64)
    n_acc = torch.zeros(1, dtype=torch.int64, device=dev)
    sb = ms.ms_unweight_scratch_bytes(N)
    scratch = torch.empty(sb, dtype=torch.uint8, device=dev)
    wmax = torch.ones(1, **f64)
    out = []
    for frac in (1e-4, 1e-3, 1e-2, 0.1, 0.5, 1.0):
        w = torch.rand(N, generator=gen, **f64) ** (1.0 / frac - 1.0)

        def call():
            ms.ms_unweight(N, w, wmax, ms.rng(ms_inputs.SEED_UNWEIGHT, 1, 0), rows, p, N, idx, w_out, rows_out, n_acc, scratch,
                           sb, N, None)
        for _ in range(max(warmup, 3)):
            call()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        ev[0].record()
        for _ in range(steps):
            call()
        ev[1].record()
        torch.cuda.synchronize()
        us = ev[0].elapsed_time(ev[1]) * 1e3 / steps
        k = int(n_acc.item())
        moved = 8 * N + k * 16 * (rows + 2)                    # weights read + (idx, w_out, rows) read and written
        out.append({"efficiency": frac, "accepted": k, "us_per_call": us, "algorithmic_gb_per_s": moved / us / 1e3})
    return {"probe": "unweight-density", "events": N, "rows": rows, "steps": steps, "results": out}


def chili(torch, steps: int = 20, warmup: int = 3, hbm_gbs: float = 0.0) -> dict:
    """ms_chili at 2^24 events, Philox in-kernel, pT_min = 20 GeV on every particle, sqrt(s) = 13 TeV."""
    sys.path.insert(0, ROOT)
    import paper_2602_06895_b200 as ms
    ms.lib()
    dev = torch.device("cuda", torch.cuda.current_device())
    N = 1 << 24
    out = []
    for n in (3, 4, 6):
        p = torch.empty((4 * (n + 2), N), dtype=torch.float64, device=dev)
        w = torch.empty(N, dtype=torch.float64, device=dev)

        def call():
            ms.ms_chili(N, n, 13000.0 ** 2, None, [20.0] * n, None, None, ms.rng(1, 0, 0), p, w, None, N)
        for _ in range(warmup):
            call()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        ev[0].record()
        for _ in range(steps):
            call()
        ev[1].record()
        torch.cuda.synchronize()
        ms_call = ev[0].elapsed_time(ev[1]) / steps
        nbytes = 8 * (4 * (n + 2) + 1) * N
        row = {"n": n, "ms": ms_call, "alg_bytes": nbytes, "achieved_gbs": nbytes / ms_call / 1e6}
        if hbm_gbs > 0:
            row["frac_of_hbm"] = row["achieved_gbs"] / hbm_gbs
        out.append(row)
        del p, w
    return {"probe": "chili", "events": N, "steps": steps, "results": out}


def vegas_map(torch, steps: int = 20, warmup: int = 3, hbm_gbs: float = 0.0) -> dict:
    """The stand-alone ms_vegas_map at the cfg-5 shape -- 20 dimensions x 2^24 events, 128 seeded bins: forward
    from uniform rows (16 B per value), forward from in-kernel Philox (8 B per value), inverse (16 B per value)."""
    sys.path.insert(0, ROOT)
    import ms_inputs
    import paper_2602_06895_b200 as ms
    ms.lib()
    dev = torch.device("cuda", torch.cuda.current_device())
    N, d, nb = 1 << 24, 20, 128
    edges = torch.from_numpy(ms_inputs.seeded_grid(d, nb)).to(dev)
    r = torch.empty((d, N), dtype=torch.float64, device=dev)
    x = torch.empty((d, N), dtype=torch.float64, device=dev)
    jac = torch.empty(N, dtype=torch.float64, device=dev)
    ms.ms_fill_uniforms(N, d, ms.rng(1, 0, 0), r, N)
    cases = {
        "forward_rows": (lambda: ms.ms_vegas_map(N, d, nb, edges, 0, r, ms.rng(0), x, jac, N), 8 * (2 * d + 1) * N),
        "forward_philox": (lambda: ms.ms_vegas_map(N, d, nb, edges, 0, None, ms.rng(1, 0, 0), x, jac, N), 8 * (d + 1) * N),
        "inverse": (lambda: ms.ms_vegas_map(N, d, nb, edges, 1, x, ms.rng(0), r, None, N), 8 * 2 * d * N),
        "inverse_jac": (lambda: ms.ms_vegas_map(N, d, nb, edges, 1, x, ms.rng(0), r, jac, N), 8 * (2 * d + 1) * N),
    }
    out = []
    for name, (call, nbytes) in cases.items():
        for _ in range(warmup):
            call()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        ev[0].record()
        for _ in range(steps):
            call()
        ev[1].record()
        torch.cuda.synchronize()
        ms_call = ev[0].elapsed_time(ev[1]) / steps
        row = {"case": name, "ms": ms_call, "alg_bytes": nbytes, "achieved_gbs": nbytes / ms_call / 1e6}
        if hbm_gbs > 0:
            row["frac_of_hbm"] = row["achieved_gbs"] / hbm_gbs
        out.append(row)
    return {"probe": "vegas-map", "events": N, "dims": d, "bins": nb, "steps": steps, "results": out}


def entry_points(torch, steps: int = 20, warmup: int = 3, hbm_gbs: float = 0.0) -> dict:
    """Every stand-alone entry point of SURVEY.md section 8(b) that bench.py does not time as a stage of its own, at 2^24
    events, against ITS algorithmic bytes (rows read + rows written, 8 B each): the fused path never calls these, a
    stage-by-stage user does."""
    sys.path.insert(0, ROOT)
    import paper_2602_06895_b200 as ms
    ms.lib()
    dev = torch.device("cuda", torch.cuda.current_device())
    N = 1 << 24

    def buf(rows):
        return torch.empty((rows, N), dtype=torch.float64, device=dev)
    cases = []
    # S0
    r8 = buf(8)
    cases.append(("ms_fill_uniforms d=8", lambda: ms.ms_fill_uniforms(N, 8, ms.rng(1, 0, 0), r8, N), 8 * 8))
    # S2/S3/S4 stand-alone: n = 4 FastRambo (8 uniforms) and n = 5 exact Rambo (11 uniforms), rows and Philox
    p4, w = buf(24), torch.empty(N, dtype=torch.float64, device=dev)
    ms.ms_fill_uniforms(N, 8, ms.rng(1, 0, 0), r8, N)
    cases.append(("ms_fastrambo n=4 rows", lambda: ms.ms_fastrambo(N, 4, 1000.0, None, r8, ms.rng(0), p4, w, N), 8 * (8 + 24 + 1)))
    cases.append(("ms_fastrambo n=4 philox", lambda: ms.ms_fastrambo(N, 4, 1000.0, None, None, ms.rng(1, 0, 0), p4, w, N), 8 * (24 + 1)))
    r11, p5 = buf(11), buf(28)
    ms.ms_fill_uniforms(N, 11, ms.rng(1, 0, 0), r11, N)
    cases.append(("ms_rambo_massless n=5 rows", lambda: ms.ms_rambo_massless(N, 5, 1000.0, None, r11, ms.rng(0), p5, w, N), 8 * (11 + 28 + 1)))
    cases.append(("ms_rambo_massless n=5 philox", lambda: ms.ms_rambo_massless(N, 5, 1000.0, None, None, ms.rng(1, 0, 0), p5, w, N), 8 * (28 + 1)))
    # S5: rescale of the n = 4 event in place (16 outgoing rows + w read and written); the input is regenerated each call
    # outside the timed loop's accounting would hide nothing: the call is timed alone on an already massive event, whose
    # Newton iteration converges at once -- so time it on fresh massless input by alternating with ms_fastrambo and
    # subtracting that call's own time (reported as "ms_massive_rescale n=4 (net)")
    cases.append(("ms_fastrambo n=4 philox, sqrt_s=2000 (feeds the rescale)",
                  lambda: ms.ms_fastrambo(N, 4, 2000.0, None, None, ms.rng(1, 0, 0), p4, w, N), 8 * (24 + 1)))
    cases.append(("ms_fastrambo + ms_massive_rescale n=4",
                  lambda: (ms.ms_fastrambo(N, 4, 2000.0, None, None, ms.rng(1, 0, 0), p4, w, N),
                           ms.ms_massive_rescale(N, 4, 2000.0, [173.0, 173.0, 0.0, 0.0], 1e-14, 20, p4, w, N)), 8 * (24 + 1) + 8 * 2 * (16 + 1)))
    # S6: Bjorken x, both phases (n = 5)
    x1x2, shat, jac = buf(2), torch.empty(N, dtype=torch.float64, device=dev), torch.empty(N, dtype=torch.float64, device=dev)
    tau_min = (200.0 / 13600.0) ** 2
    cases.append(("ms_pdf_x_boost sample (philox)", lambda: ms.ms_pdf_x_boost(N, 5, 13600.0 ** 2, tau_min, 0, None, ms.rng(1, 0, 0), x1x2, shat, jac, None, N), 8 * 4))
    cases.append(("ms_pdf_x_boost boost n=5", lambda: ms.ms_pdf_x_boost(N, 5, 13600.0 ** 2, tau_min, 1, None, ms.rng(0), x1x2, None, None, p5, N), 8 * (2 + 2 * 2 * 5 + 8)))   # reads x1, x2 and (E, pz) of five momenta, writes those back and the two incoming momenta
    # S7, S8 helpers
    f = torch.empty(N, dtype=torch.float64, device=dev)
    cases.append(("ms_toy_integrand n=4", lambda: ms.ms_toy_integrand(N, 4, 100.0, p4, f, False, N), 8 * (16 + 1)))
    wmax = torch.zeros(1, dtype=torch.float64, device=dev)
    cases.append(("ms_reduce_max", lambda: ms.ms_reduce_max(N, w, wmax), 8))
    out = []
    for name, call, bytes_per_event in cases:
        for _ in range(warmup):
            call()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        ev[0].record()
        for _ in range(steps):
            call()
        ev[1].record()
        torch.cuda.synchronize()
        ms_call = ev[0].elapsed_time(ev[1]) / steps
        row = {"case": name, "ms": ms_call, "alg_bytes_per_event": bytes_per_event,
               "achieved_gbs": bytes_per_event * N / ms_call / 1e6}
        if hbm_gbs > 0:
            row["frac_of_hbm"] = row["achieved_gbs"] / hbm_gbs
        out.append(row)
    return {"probe": "entry-points", "events": N, "steps": steps, "results": out}


def next_rows(torch, steps: int = 20, warmup: int = 3, hbm_gbs: float = 0.0) -> dict:
    """The calls built beyond section 8(a) (NEXT-2 .. NEXT-4: observables, cuts, histograms, grid accumulation, weight
    histogram, running maximum, Chili from uniform rows) at 2^24 events, each against its own algorithmic bytes."""
    sys.path.insert(0, ROOT)
    import paper_2602_06895_b200 as ms
    ms.lib()
    dev = torch.device("cuda", torch.cuda.current_device())
    N, n = 1 << 24, 4

    def buf(*shape):
        return torch.empty(shape, dtype=torch.float64, device=dev)
    p, w, obs = buf(4 * (n + 2), N), buf(N), buf(N)
    ms.ms_fastrambo(N, n, 1000.0, None, None, ms.rng(1, 0, 0), p, w, N)
    w2 = w.clone()
    cases = []
    for kind, rows in (("PT", 2), ("Y", 2), ("ETA", 3), ("PHI", 2), ("DR", 6), ("MASS", 8)):
        cases.append(("ms_observable %s" % kind, (lambda k=kind: ms.ms_observable(N, k, 2, 3, n, p, obs, N)), 8 * (rows + 1)))
    cases.append(("ms_observable HT (n_out = 4)", lambda: ms.ms_observable(N, "HT", 0, 0, n, p, obs, N), 8 * (4 * n + 1)))
    ms.ms_observable(N, "PT", 2, 3, n, p, obs, N)
    cases.append(("ms_cut", lambda: ms.ms_cut(N, obs, 20.0, float("inf"), w2), 8 * 3))
    sw, sw2 = torch.zeros(102, dtype=torch.float64, device=dev), torch.zeros(102, dtype=torch.float64, device=dev)
    cases.append(("ms_histogram_fill 100 bins", lambda: ms.ms_histogram_fill(N, obs, w, 0.0, 500.0, 100, sw, sw2), 8 * 2))
    hist = torch.zeros((8, 128), dtype=torch.float64, device=dev)
    cases.append(("ms_vegas_accumulate 128 x 8", lambda: ms.ms_vegas_accumulate(N, 8, 128, w, ms.rng(1, 0, 0), hist), 8))
    counts = torch.zeros(32768, dtype=torch.int64, device=dev)      # MS_HIST_BINS
    cases.append(("ms_weight_histogram", lambda: ms.ms_weight_histogram(N, w, counts), 8))
    cases.append(("ms_elementwise_max", lambda: ms.ms_elementwise_max(N, w, w2, obs), 8 * 3))
    xr = buf(3 * n - 2, N)
    ms.ms_fill_uniforms(N, 3 * n - 2, ms.rng(1, 0, 0), xr, N)
    cases.append(("ms_chili n=4 rows", lambda: ms.ms_chili(N, n, 13000.0 ** 2, None, [20.0] * n, None, xr, ms.rng(0), p, w, None, N),
                  8 * (3 * n - 2 + 4 * (n + 2) + 1)))
    out = []
    for name, call, bytes_per_event in cases:
        for _ in range(warmup):
            call()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        ev[0].record()
        for _ in range(steps):
            call()
        ev[1].record()
        torch.cuda.synchronize()
        ms_call = ev[0].elapsed_time(ev[1]) / steps
        row = {"case": name, "ms": ms_call, "alg_bytes_per_event": bytes_per_event,
               "achieved_gbs": bytes_per_event * N / ms_call / 1e6}
        if hbm_gbs > 0:
            row["frac_of_hbm"] = row["achieved_gbs"] / hbm_gbs
        out.append(row)
    return {"probe": "next-rows", "events": N, "steps": steps, "results": out}


def _hbm_peak() -> float:
    pk = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pk):
        with open(pk) as f:
            return float(json.load(f)["hbm_gbs"])
    return 0.0


def main() -> int:
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench_probes.py needs a CUDA device")
    what = sys.argv[1] if len(sys.argv) > 1 else "fp64"
    if what == "fp64":
        res = {"probe": "fp64", "const_operand": fp64_rate(torch, 2.0), "three_registers": fp64_rate(torch, 2.0, True)}
    elif what == "issue-model":
        res = {"probe": "issue-model", **issue_model(torch), "dfma_latency": dfma_latency(torch)}
    elif what == "unweight-density":
        res = unweight_density(torch)
    elif what == "chili":
        res = chili(torch, hbm_gbs=_hbm_peak())
    elif what == "vegas-map":
        res = vegas_map(torch, hbm_gbs=_hbm_peak())
    elif what == "entry-points":
        res = entry_points(torch, hbm_gbs=_hbm_peak())
    elif what == "next-rows":
        res = next_rows(torch, hbm_gbs=_hbm_peak())
    else:
        raise SystemExit("unknown probe: " + what)
    print(json.dumps(res))
    return 0


if __name__ == "__main__":
    sys.exit(main())
