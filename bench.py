#!/usr/bin/env python
"""bench.py -- phase-space events/s of the MadSpace hot path on B200 (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2] [--impl ours|reference]

A step = one pass of the whole hot path over one batch of synthetic (Philox-seeded) events: for the default
workload (BASELINE.json configs[1], "cfg2": massless 2->4 FastRambo, 2^24 events, seeded 128x8 VEGAS grid, toy
integrand, unweighting) that is ms_generate -> ms_reduce_max (pre-run w_max) -> ms_unweight.
N > 1 (torchrun): one process per GPU, every rank generates its own 2^24-event batch at event offset rank*2^24
(weak scaling, no data-path collective); value = events of all ranks / max-over-ranks time.
--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import ms_inputs  # noqa: E402

METRIC = "phase-space events/s (fp64, weighted events through the whole hot path)"
UNIT = "events/s"
FP64_LANES_PER_SM = 64            # B200 (GB100): 64 FP64 FMA lanes per SM (datasheet 37 TFLOP/s = 148*64*2*1.965 GHz)

# Hand-counted fp64-pipe instructions (DADD/DMUL/DFMA/DSETP) of the final formulas, per stage (DESIGN.md §5
# "algorithmic op count"; MUFU seeds and int<->fp conversions run on the XU pipe and are not counted here).
RCP, SQRT, SQRT_H = 3, 5, 7   # third-order correction after the MUFU seed: rcp_fast, sqrt_fast, sqrt_fast with 1/(2 sqrt)
RQF_INVERSE = 16 + SQRT + RCP  # s, beta, a, discriminant (3), sqrt, d1 (2), a2, product, rcp, y (3), z (3)
EXP = 18                   # magic-number reduction (4), r^2, degree-11 Horner, 2 fma
SINCOS = 21                # quarter-turn reduction (4), r^2, two degree-7 Horners, 2


def _pow_cost(r):          # multiplications of u^r by squaring
    return max(r.bit_length() - 1 + bin(r).count("1") - 1, 0)


def _mass_ratio(k):        # v = y^(1/k), u = sqrt(v), 1 - v = z / (1 + v + ... + v^(k-1))
    if k == 1:
        return SQRT
    if k == 2:
        return 2 * (SQRT) + 1 + RCP + 1
    return _pow_cost(2 * k) + 4 + RCP + 2 + 1 + (k - 1) + RCP + 1      # Halley root of order 2k, v, S, rcp, 1-v


def fast_mass_step(k):     # RQF inverse, ratio, weight factor (k+1) D^2 / ((2y + c z) S), q, M, weight products
    return RQF_INVERSE + _mass_ratio(k) + (3 if k == 1 else 7) + 5


def exact_mass_step(k):
    """k = 1: closed form.  k >= 2: the start value and four Newton steps run in fp32 (not fp64-pipe work); what is
    counted is the one fp64 Halley step (three Horners of degree k-1, 16 more), 1 - w, sqrt, and the chain updates."""
    if k == 1:
        return 1 + SQRT + 1 + RCP + 1 + SQRT + 3
    return 1 + 3 * k + 16 + 1 + SQRT + 3


ALG_FP64 = {"uniform": 1, "vegas_dim": 5, "decay_first": 3 + SQRT + 1 + SINCOS + 4 + 1,
            "decay": 3 + SQRT + 1 + SINCOS + 4 + 2 + RCP + 4 + 4 + 3 + 4,
            "toy_pair": 13, "weight": 5 + RCP + 3 + 3, "pdf": 2 * EXP + 4 + RCP + 2 + 4 + 3 + 4, "boost_particle": 4,
            "rescale_start": 1 + RCP + 1 + 1 + SQRT, "rescale_eval_massive": 2 + SQRT_H + 4, "rescale_eval_massless": 2,
            "rescale_eval_fixed": 2 + RCP + 1, "rescale_final_massive": 2 + SQRT_H + 4 + 3, "rescale_final_massless": 5,
            "rescale_weight": 3 + 3 + RCP}
RESCALE_EVALUATIONS = 4    # cfg4 converges in <= 3 Newton steps: 4 evaluations of F


def alg_fp64_per_event(wl: ms_inputs.Workload) -> int:
    n = wl.n
    c = ALG_FP64["uniform"] * wl.d + ALG_FP64["vegas_dim"] * wl.grid_dims
    for i in range(2, n):
        c += fast_mass_step(n - i) if wl.mapping == "fastrambo" else exact_mass_step(n - i)
    c += ALG_FP64["decay_first"] + ALG_FP64["decay"] * (n - 2)
    if wl.toy:
        c += ALG_FP64["toy_pair"] * (n - 1)
    if wl.pdf:
        c += ALG_FP64["pdf"] + ALG_FP64["boost_particle"] * n
    if wl.masses and wl.massive_mode == "reweight":
        # per decay: 1-u via rcp (2 + RCP), factorised Kallen (7) + sqrt, 1/(2M) (RCP + 1), q, e_rest (4), weight (5), M_i (1)
        c += (n - 1) * (2 + RCP + 7 + SQRT + RCP + 1 + 1 + 4 + 5 + 1) + 2
    elif wl.masses:
        nm = sum(1 for m in wl.masses if m > 0)
        c += ALG_FP64["rescale_start"] + ALG_FP64["rescale_weight"]
        c += RESCALE_EVALUATIONS * (ALG_FP64["rescale_eval_massive"] * nm + ALG_FP64["rescale_eval_massless"] * (n - nm)
                                    + ALG_FP64["rescale_eval_fixed"])
        c += ALG_FP64["rescale_final_massive"] * nm + ALG_FP64["rescale_final_massless"] * (n - nm)
    return c + ALG_FP64["weight"]


# dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch, from the committed ncu captures
# (recorded, not measured by this script; --traffic overrides).
NCU_TRAFFIC = {"cfg2": (3.295350e9 + 513.28e3, "profiles/r01e_final.md"), "cfg3": (16.583720e9 + 112.1e3, "profiles/r01e_final.md"),
               "cfg5": (5.443808e9 + 91e3, "profiles/r01e_final.md"), "cfg4": (6.651895e9 + 172.5e3, "profiles/r01e_final.md")}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi sampled DURING the timed region (profiling recipe's clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "20"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for nm, v in zip(names, c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


# ------------------------------------------------------------------------------------------------ CPU oracle arm

def oracle_step(orc, wl, n_events, offset=0):
    """One pass of the same hot path over `n_events` events with the oracle as it stands (tests/helpers.py chain +
    w_max of the pre-run + sequential hit-or-miss unweighting [+ inverse round trip])."""
    from oracle.chain import oracle_chain
    ref = oracle_chain(orc, wl, np.arange(offset, offset + n_events))
    n_acc = None
    if wl.unweight:
        w = np.ascontiguousarray(ref["w"])
        wmax = orc.wmax(np.ascontiguousarray(w[:min(ms_inputs.PRERUN, n_events)]))
        _, _, n_acc = orc.unweight(w, wmax, ms_inputs.SEED_UNWEIGHT, ms_inputs.STREAM_UNWEIGHT, offset, n_events)
    if wl.inverse:
        xi, _ = orc.fastrambo_inverse(wl.n, ref["p"])
        edges = wl.grid()
        if edges is not None:
            orc.vegas_inverse(np.ascontiguousarray(edges[:3 * wl.n - 4]), xi)
    return n_acc


def time_oracle(wl, target_seconds=12.0, steps=1, warmup=0):
    import oracle as orc
    orc.lib()
    probe = 1 << 16
    t0 = time.perf_counter()
    oracle_step(orc, wl, probe)
    t_probe = max(time.perf_counter() - t0, 1e-4)
    per_step = target_seconds / max(steps + warmup, 1)
    n = int(min(wl.N, max(probe, probe * per_step / t_probe)))
    n = 1 << (n.bit_length() - 1)
    for _ in range(warmup):
        oracle_step(orc, wl, n)
    times = []
    for _ in range(steps):
        t0 = time.perf_counter()
        oracle_step(orc, wl, n)
        times.append(time.perf_counter() - t0)
    t = float(np.mean(times))
    out = {"value": n / t, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
           "sample": "first %d events (2^%d) of %s per step, %d step(s); OpenMP over event ranges, sequential unweighting"
                     % (n, n.bit_length() - 1, wl.name, steps)}
    # the same oracle on ONE thread (a per-core figure), on at most 2^20 events
    try:
        from threadpoolctl import threadpool_limits
        n1 = min(n, 1 << 20)
        with threadpool_limits(limits=1, user_api="openmp"):
            if orc.num_threads() == 1:
                t0 = time.perf_counter()
                oracle_step(orc, wl, n1)
                out["per_core_value"] = n1 / (time.perf_counter() - t0)
                out["per_core_sample"] = "first %d events on 1 thread" % n1
    except Exception as ex:                                   # a reported extra, never a reason to fail the bench
        out["per_core_value"] = None
        out["per_core_sample"] = "unavailable: %s" % type(ex).__name__
    return out, t


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = ms_inputs.WORKLOADS[args.workload]
    cb, t = time_oracle(wl, target_seconds=60.0, steps=args.steps, warmup=args.warmup)
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(wl, args.gpus), "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def workload_config(wl, n_gpus):
    return {"workload": "%s: %s" % (wl.name, wl.note), "events_per_gpu_per_step": wl.N, "n": wl.n,
            "grid": "%dx%d %s" % (wl.grid_bins, wl.grid_dims, wl.grid_kind), "parallelism": "events sharded x%d" % n_gpus,
            "l2": "no flush needed: each step streams %.2f GB of fresh output (> 126 MB L2)" % (wl.N * wl.out_bytes_per_event / 1e9)}


# ------------------------------------------------------------------------------------------------ GPU arm

def spec_from_workload(wl):
    from paper_2602_06895_b200.pipeline import PathSpec
    return PathSpec(n=wl.n, sqrt_s=wl.sqrt_s, mapping=wl.mapping, edges=wl.grid(), pdf=wl.pdf, tau_min=wl.tau_min,
                    masses=tuple(wl.masses), massive_mode=wl.massive_mode, toy=wl.toy, toy_reg=ms_inputs.TOY_REG,
                    unweight=wl.unweight,
                    inverse=wl.inverse, prerun=ms_inputs.PRERUN, seed_events=ms_inputs.SEED_EVENTS,
                    seed_unweight=ms_inputs.SEED_UNWEIGHT)


def probe_fp64_rate(ms, torch, seconds=0.25, three_regs=False):
    """Sustained DFMA issue rate (instructions/s) measured with ms_probe_dfma (register * constant + constant) or
    ms_probe_dfma3 (three distinct register operands): 8 independent chains per thread."""
    probe = ms.ms_probe_dfma3 if three_regs else ms.ms_probe_dfma
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    blocks, iters = sms * 8, 1 << 14
    sink = torch.empty(blocks * 256, dtype=torch.float64, device="cuda")
    probe(blocks, iters, sink)
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps, best, t_end = 0, 0.0, time.perf_counter() + seconds
    while time.perf_counter() < t_end or reps < 3:
        ev0.record()
        probe(blocks, iters, sink)
        ev1.record()
        ev1.synchronize()
        best = max(best, blocks * 256 * iters * 8 / (ev0.elapsed_time(ev1) * 1e-3))
        reps += 1
    return best


def probe_write_stream(ms, torch, hp, wl, reps=10):
    """GB/s of the generation kernel's store pattern with no arithmetic (ms_probe_write into the momentum buffer)."""
    rows = hp.spec.rows_p
    ms.ms_probe_write(hp.N, rows, hp.p, hp.ld)
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(reps):
        ms.ms_probe_write(hp.N, rows, hp.p, hp.ld)
    ev1.record()
    ev1.synchronize()
    return 8.0 * rows * hp.N * reps / (ev0.elapsed_time(ev1) * 1e-3) / 1e9


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2602_06895_b200 as ms
    from paper_2602_06895_b200.pipeline import HotPath
    from paper_2602_06895_b200.sharding import gather_counts, output_offsets, weak_range

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the hot path has no CPU fallback (use --impl reference for the oracle)")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    ms.lib()
    wl = ms_inputs.WORKLOADS[args.workload]
    N = wl.N if args.events <= 0 else args.events
    offset, _ = weak_range(N, rank)
    dev = torch.device("cuda", local)
    hp = HotPath(spec_from_workload(wl), N, dev, cap=max(1 << 16, N // 256))
    stream = torch.cuda.current_stream()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-up steps, then exactly K steps between barriers + synchronize
    for _ in range(args.warmup):
        hp.step(offset)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    stages = [("generate", lambda: hp.generate(offset))]
    if wl.unweight:
        stages.append(("unweight", lambda: hp.unweight(offset)))
    if wl.inverse:
        stages.append(("fastrambo_inverse", hp.invert_phase_space))
        stages.append(("vegas_inverse", hp.invert_grid))
    marks = [[torch.cuda.Event(enable_timing=True) for _ in range(len(stages) + 1)] for _ in range(args.steps)]
    ev[0].record(stream)
    for k in range(args.steps):
        marks[k][0].record(stream)
        for j, (_, fn) in enumerate(stages):
            fn()
            marks[k][j + 1].record(stream)
    ev[1].record(stream)
    barrier()
    t_total = ev[0].elapsed_time(ev[1]) * 1e-3
    stage_ms = {name: float(np.mean([m[j].elapsed_time(m[j + 1]) for m in marks])) for j, (name, _) in enumerate(stages)}
    t_gen = stage_ms["generate"] * 1e-3
    per_step = [m[0].elapsed_time(m[-1]) for m in marks]      # median and best beside the mean
    step_stats = {"median": float(np.median(per_step)), "best": float(np.min(per_step)), "worst": float(np.max(per_step))}
    n_acc_local = int(hp.n_acc.item()) if wl.unweight else 0
    if world > 1:
        tt = torch.tensor([t_total, t_gen], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_total, t_gen = float(tt[0]), float(tt[1])
    counts = gather_counts(n_acc_local)
    offsets = output_offsets(counts)
    launches_all = sum(gather_counts(hp.launches(offset) * args.steps))   # ranks > 0 replay the pre-run: one more launch

    # ---- end to end through the public API with HOST buffers: every step copies its input (the grid table) from pinned
    # host memory and the host reads the step's result.  For a generator the result is the unweighted sample: the
    # accepted count and that many entries of idx, w_out and every momentum row.  The read-back is pipelined the way a
    # production driver would do it ("CPU work overlapped"): two sets of buffers, an upload and a download
    # stream, and the host consumes step k-1 while the device runs step k.
    h_edges = torch.from_numpy(wl.grid()).pin_memory() if wl.grid() is not None else None
    h2d_bytes = h_edges.numel() * 8 if h_edges is not None else 0
    d2h_counter = [0]
    if wl.unweight:
        # output capacity of the e2e buffers: next power of two above twice the count seen in the device-resident run
        cap_e2e = min(hp.cap, max(1024, 1 << (2 * max(n_acc_local, 1) - 1).bit_length()))
        hps = [HotPath(spec_from_workload(wl), N, dev, cap=cap_e2e) for _ in range(2)]
        up_stream, down_stream = torch.cuda.Stream(device=dev), torch.cuda.Stream(device=dev)
        rows_p = hp.spec.rows_p
        hb = [dict(nacc=torch.empty(1, dtype=torch.int64).pin_memory(),
                   idx=torch.empty(cap_e2e, dtype=torch.int64).pin_memory(),
                   wout=torch.empty(cap_e2e, dtype=torch.float64).pin_memory(),
                   rows=torch.empty((rows_p, cap_e2e), dtype=torch.float64).pin_memory()) for _ in range(2)]
        ev_grid = [torch.cuda.Event() for _ in range(2)]
        ev_done = [torch.cuda.Event() for _ in range(2)]
        ev_copied = [torch.cuda.Event() for _ in range(2)]

        def launch(k):
            s, h = k % 2, hps[k % 2]
            if h_edges is not None:                        # this step's input, uploaded while the previous step runs
                with torch.cuda.stream(up_stream):
                    h.d_edges.copy_(h_edges, non_blocking=True)
                    ev_grid[s].record(up_stream)
                stream.wait_event(ev_grid[s])
            h.step(offset)
            ev_done[s].record(stream)
            with torch.cuda.stream(down_stream):           # whole contiguous buffers: plain async memcpys into pinned memory
                down_stream.wait_event(ev_done[s])
                hb[s]["nacc"].copy_(h.n_acc, non_blocking=True)
                hb[s]["idx"].copy_(h.idx, non_blocking=True)
                hb[s]["wout"].copy_(h.w_out, non_blocking=True)
                hb[s]["rows"].copy_(h.rows_out, non_blocking=True)
                ev_copied[s].record(down_stream)

        def consume(k):
            s = k % 2
            ev_copied[s].synchronize()                     # the host has this step's sample
            n = int(hb[s]["nacc"][0])
            if n > cap_e2e:
                raise SystemExit("bench.py: %d accepted events exceed the e2e capacity %d" % (n, cap_e2e))
            d2h_counter[0] = 8 + cap_e2e * 8 * (2 + rows_p)
            return n

        def e2e_run(steps):
            launch(0)
            for k in range(1, steps):
                launch(k)
                consume(k - 1)
            consume(steps - 1)
            stream.wait_event(ev_copied[(steps - 1) % 2])  # the timed region ends when the last sample is on the host
        e2e_what = ("every step: grid table H2D from pinned memory, the whole step, D2H of the accepted count and of the "
                    "compacted unweighted sample buffers (idx, w_out, %d momentum rows; capacity %d entries); transfers "
                    "on their own streams with two buffer sets, the host consumes step k-1 while step k runs"
                    % (rows_p, cap_e2e))
    else:
        d2h = [(hp.w, torch.empty(hp.ld, dtype=torch.float64).pin_memory()),
               (hp.p, torch.empty((hp.spec.rows_p, hp.ld), dtype=torch.float64).pin_memory())]

        def e2e_run(steps):
            for _ in range(steps):
                if h_edges is not None:
                    hp.d_edges.copy_(h_edges, non_blocking=True)
                hp.step(offset)
                for d_t, h_t in d2h:
                    h_t.copy_(d_t, non_blocking=True)
                d2h_counter[0] = sum(h_t.numel() * h_t.element_size() for _, h_t in d2h)
                torch.cuda.current_stream().synchronize()  # the host consumes the step's result
        e2e_what = "grid table H2D from pinned memory + whole step + D2H of all momenta and weights, host waits every step"

    e2e_run(2)
    barrier()
    t0 = time.perf_counter()
    ev[0].record(stream)
    e2e_run(args.steps)
    ev[1].record(stream)
    barrier()
    t_e2e_wall = time.perf_counter() - t0
    clocks = sampler.stop() if sampler else None          # sampled over both timed regions (device-resident and e2e)
    t_e2e = max(ev[0].elapsed_time(ev[1]) * 1e-3, 0.0)
    if world > 1:
        tt = torch.tensor([t_e2e], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        t_e2e = float(tt[0])

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (the fused generation kernel)
    hbm_gbs, sm_max_mhz, peak_src = measured_peaks()
    sms = torch.cuda.get_device_properties(local).multi_processor_count
    bytes_per_launch = N * wl.out_bytes_per_event + (h2d_bytes if h_edges is not None else 0)
    inst_per_event = alg_fp64_per_event(wl)
    fp64_peak = sms * FP64_LANES_PER_SM * sm_max_mhz * 1e6            # fp64-pipe instructions / s at max clock
    fp64_probe = probe_fp64_rate(ms, torch)
    fp64_probe3 = probe_fp64_rate(ms, torch, three_regs=True)
    write_probe = probe_write_stream(ms, torch, hp, wl)
    t_hbm = bytes_per_launch / (hbm_gbs * 1e9)
    t_alu = N * inst_per_event / fp64_peak
    if t_hbm >= t_alu:
        roof = {"bound": "hbm", "achieved": bytes_per_launch / t_gen / 1e9, "peak": hbm_gbs, "unit": "GB/s"}
    else:
        roof = {"bound": "alu", "achieved": N * inst_per_event / t_gen / 1e9, "peak": fp64_peak / 1e9, "unit": "Ginst/s (fp64 pipe)"}
    roof["frac"] = roof["achieved"] / roof["peak"]
    traffic, traffic_src = (args.traffic, "--traffic") if args.traffic > 0 else NCU_TRAFFIC.get(wl.name, (None, None))
    if N != wl.N:
        traffic, traffic_src = None, None
    roof.update(traffic=traffic, traffic_source=traffic_src, kernel="ms::gen_kernel<%d,%s,%s>" % (
        wl.n, "exact" if wl.mapping == "rambo" else "fast", "massive" if wl.masses else "massless"),
        kernel_ms=1e3 * t_gen, kernel_share_of_step=t_gen * args.steps / t_total, peak_source=peak_src,
        alg_bytes_per_event=wl.out_bytes_per_event, alg_fp64_inst_per_event=inst_per_event,
        hbm_time_ms=1e3 * t_hbm, alu_time_ms=1e3 * t_alu, frac_of_max_side=max(t_hbm, t_alu) / t_gen,
        fp64_peak_ginst_nominal=fp64_peak / 1e9, fp64_ginst_probe_measured=fp64_probe / 1e9, fp64_ginst_probe_3reg_operands=fp64_probe3 / 1e9, write_stream_probe_gbs=write_probe,
        kernel_events_per_s=N / t_gen)

    cb = None if args.skip_cpu_baseline else time_oracle(wl, target_seconds=12.0)[0]
    total_events = float(N) * world * args.steps
    line = {"metric": METRIC, "value": total_events / t_total, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t_total / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic (Philox-seeded uniforms; seeded VEGAS grid stands in for an adapted one)",
            "config": workload_config(wl, world), "clocks": clocks,
            "e2e": {"value": total_events / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d_bytes, "d2h_bytes_per_step": d2h_counter[0],
                    "wall_value": total_events / t_e2e_wall,
                    "what": e2e_what},
            "gpu_launches": launches_all, "roofline": roof, "stage_ms": stage_ms, "ms_per_step_stats": step_stats, "cpu_baseline": cb,
            "unweighted": ({"accepted_per_step_per_rank": counts, "global_offsets": offsets,
                            "unweighted_events_per_s": sum(counts) * args.steps / t_total} if wl.unweight else None),
            "fail_count": int(hp.fail.item()),
            "paper_context": "PAPER.md:766-770: full LO chain incl. matrix elements ~30M weighted evt/s on A100 (DY+1g), up to 10M on 24 Xeon-4214 cores; not this path in isolation"}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_unweight_density(args):
    """Side measurement (not the bench line): ms_unweight alone on 2^24 synthetic weights x 24 momentum rows at several
    acceptance rates -- the unweighting efficiencies a production run sees after grid adaptation
    rather than the 1e-4 of the seeded-grid workloads.  Weights w = u^(1/f - 1) with w_max = 1 have <w>/w_max = f."""
    import torch
    import paper_2602_06895_b200 as ms
    ms.lib()
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
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
        for _ in range(max(args.warmup, 3)):
            call()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        torch.cuda.synchronize()
        ev[0].record()
        for _ in range(args.steps):
            call()
        ev[1].record()
        torch.cuda.synchronize()
        us = ev[0].elapsed_time(ev[1]) * 1e3 / args.steps
        k = int(n_acc.item())
        moved = 8 * N + k * 16 * (rows + 2)                    # weights read + (idx, w_out, rows) read and written
        out.append({"efficiency": frac, "accepted": k, "us_per_call": us, "algorithmic_gb_per_s": moved / us / 1e3})
    print(json.dumps({"probe": "unweight-density", "events": N, "rows": rows, "steps": args.steps, "results": out}))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg2", choices=sorted(ms_inputs.WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--events", type=int, default=0, help="override events per GPU per step (0 = the workload's)")
    ap.add_argument("--skip-cpu-baseline", action="store_true", help="profiling runs only: do not time the oracle")
    ap.add_argument("--traffic", type=float, default=0.0, help="dram bytes per launch of the dominant kernel from ncu (recorded, not measured here)")
    ap.add_argument("--probe", default="", choices=["", "unweight-density"],
                    help="side measurements for DESIGN.md / profiles (not the bench line)")
    args = ap.parse_args()
    if args.probe == "unweight-density":
        args.steps = min(args.steps, 20)
        return run_unweight_density(args)
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
