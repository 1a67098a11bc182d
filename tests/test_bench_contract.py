"""bench.py's contract, the reference arm (the oracle timed on the host cores)
prints ONE JSON line with the keys the driver reads, non-zero ranks of a multi-process launch print nothing, and the
hand-counted roofline inputs (algorithmic bytes and fp64 instructions per event) follow the workload definitions."""
import json
import os
import subprocess
import sys

import ms_inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run_bench(*args, env=None):
    e = dict(os.environ)
    e.update(env or {})
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), *args], capture_output=True, text=True, env=e,
                       cwd=ROOT, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    return r.stdout


def test_reference_arm_prints_one_contract_line():
    out = run_bench("--impl", "reference", "--steps", "2", "--warmup", "1").strip().splitlines()
    assert len(out) == 1
    d = json.loads(out[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 1 and d["steps"] == 2 and d["warmup"] == 1
    assert d["unit"] == "events/s" and d["higher_is_better"] is True and d["dtype"] == "f64"
    assert d["value"] > 0 and d["ms_per_step"] > 0 and d["vs_baseline"] is None
    assert d["config"]["workload"].startswith("cfg2") and "model" not in d["config"]
    cb = d["cpu_baseline"]
    assert cb["kind"] == "oracle" and cb["cores"] >= 1 and cb["value"] == d["value"] and cb["sample"]
    e2e = d["e2e"]
    assert e2e["value"] == d["value"] and e2e["unit"] == d["unit"]
    assert e2e["h2d_bytes_per_step"] == 0 and e2e["d2h_bytes_per_step"] == 0


def test_reference_arm_other_ranks_stay_silent():
    out = run_bench("--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0",
                    env={"RANK": "1", "LOCAL_RANK": "1", "WORLD_SIZE": "2"})
    assert out.strip() == ""


def test_roofline_inputs_follow_the_workloads():
    sys.path.insert(0, ROOT)
    import bench
    for name, rows in (("cfg1", 21), ("cfg2", 25), ("cfg3", 29), ("cfg4", 25), ("cfg5", 41)):
        wl = ms_inputs.WORKLOADS[name]
        assert wl.out_rows == rows and wl.out_bytes_per_event == 8 * rows
        assert bench.alg_fp64_per_event(wl) > 0
        # the x1, x2 rows the kernel stores where Bjorken x are sampled count as algorithmic bytes
        assert bench.alg_bytes_per_event(wl) == 8 * rows + (16 if wl.pdf else 0)
    assert bench.alg_fp64_inverse(8) > bench.alg_fp64_inverse(4) > 0
    assert set(bench.CLOSED_FORM) == set(ms_inputs.WORKLOADS)
    # the hand count grows with the multiplicity and with every optional stage
    c = {k: bench.alg_fp64_per_event(ms_inputs.WORKLOADS[k]) for k in ms_inputs.WORKLOADS}
    assert c["cfg1"] < c["cfg2"] < c["cfg5"] and c["cfg4rw"] < c["cfg4"]


def test_design_roofline_table_is_the_bench_functions():
    """DESIGN.md section 5 quotes bytes and fp64 instructions per event for every config; they are bench.py's functions, not a
    copy that can drift (the two disagreed)."""
    import re
    sys.path.insert(0, ROOT)
    import bench
    text = open(os.path.join(ROOT, "DESIGN.md")).read()
    rows = re.findall(r"^\| (cfg\w+) \([^|]*\|[^|]*\| (\d+) \| (\d+) \|", text, flags=re.M)
    seen = {}
    for name, nbytes, ninst in rows:
        seen[name] = (int(nbytes), int(ninst))
    assert set(seen) == set(ms_inputs.WORKLOADS), seen
    for name, (nbytes, ninst) in seen.items():
        wl = ms_inputs.WORKLOADS[name]
        assert nbytes == bench.alg_bytes_per_event(wl), name
        assert ninst == bench.alg_fp64_per_event(wl), name


import pytest


@pytest.mark.gpu
def test_our_arm_prints_one_contract_line_on_the_gpu():
    """The product arm on a reduced event count (the full-size line is the driver's to take): every key of the contract
    is there, the launch count is the library's own kernels, and the e2e leg really moved bytes both ways."""
    out = run_bench("--steps", "3", "--warmup", "3", "--events", str(1 << 20), "--skip-cpu-baseline").strip().splitlines()
    assert len(out) == 1
    d = json.loads(out[0])
    assert "impl" not in d or d["impl"] != "reference"
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
              "vs_baseline", "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline", "cpu_baseline"):
        assert k in d, k
    assert d["steps"] == 3 and d["warmup"] == 3 and d["n_gpus"] == 1 and d["scaling"] == "weak" and d["dtype"] == "f64"
    assert d["gpu_launches"] == 3 * 3                      # per step in steady state: generate, decide, scatter
    r = d["roofline"]
    assert r["bound"] in ("hbm", "alu") and r["unit"].split()[0] in ("GB/s", "Ginst/s") and r["peak"] > 0
    assert abs(r["frac"] - r["achieved"] / r["peak"]) < 1e-12 and 0 < r["frac"] < 1.0
    e = d["e2e"]
    assert e["value"] > 0 and e["h2d_bytes_per_step"] > 0 and e["d2h_bytes_per_step"] > 0
    assert d["fail_count"] == 0 and d["unweighted"]["accepted_per_step_per_rank"][0] > 0
    assert "sm_mhz" in d["clocks"] and "reasons" in d["clocks"]


PER_CONFIG_KEYS = ("kernel", "kernel_ms", "alg_bytes_per_event", "alg_fp64_inst_per_event", "hbm_time_ms", "alu_time_ms", "bound",
                   "frac", "traffic", "stages", "parity", "ms_per_step", "events_per_s")
STAGE_KEYS = ("ms", "bound", "roofline_ms", "frac", "traffic", "kernel")


@pytest.mark.gpu
def test_per_config_block_covers_every_config_and_stage():
    """one bench command measures all BASELINE.json configs -- every stage with its own roofline against
    the MEASURED fp64 rate, sampled parity against the oracle, the round-trip exceedance count and the Monte Carlo mean
    against the closed forms."""
    out = run_bench("--steps", "3", "--warmup", "3", "--per-config-steps", "2", "--skip-cpu-baseline").strip().splitlines()
    assert len(out) == 1
    d = json.loads(out[0])
    pc = d["per_config"]
    assert set(pc) == {"cfg1", "cfg2", "cfg3", "cfg4", "cfg4rw", "cfg5"}
    assert d["roofline"]["fp64_ginst_probe_measured"] > 0.5 * d["roofline"]["fp64_peak_ginst_nominal"]
    for name, c in pc.items():
        for k in PER_CONFIG_KEYS:
            assert k in c, (name, k)
        assert c["bound"] in ("hbm", "alu") and 0 < c["frac"] < 1.1
        want = {"generate"} | ({"unweight"} if name in ("cfg2", "cfg5") else set()) \
            | ({"inverse_fused", "fastrambo_inverse", "vegas_inverse"} if name == "cfg5" else set())
        assert set(c["stages"]) == want, (name, set(c["stages"]))
        for sname, st in c["stages"].items():
            for k in STAGE_KEYS:
                assert k in st
            assert st["bound"] in (("latency",) if sname == "unweight" else ("hbm", "alu"))
        if "unweight" in c["stages"]:
            ut = c["unweighting_total"]
            assert ut["total_ms"] > 0 and 0 < ut["frac_of_larger_side"] < 1.5 and ut["generate_with_decision_ms"] > 0
        par = c["parity"]
        assert par["max_dp_over_sqrt_s"] <= 1e-12 and par["fail_count"] == 0
        mc = par["mc_mean_over_closed_form"]
        if name == "cfg5":      # d = 20 on a random grid: heavy-tailed, a weak pin
            assert 0.5 < mc["ratio"] < 2.0, mc
        else:
            assert abs(mc["ratio"] - 1.0) <= 5.0 * mc["mc_error"] + 1e-13, (name, mc)
    assert pc["cfg3"]["alg_bytes_per_event"] == 248
    assert pc["cfg2"]["parity"]["unweighting_bit_exact_vs_oracle_on_all_weights"] is True
    assert pc["cfg5"]["parity"]["unweighting_bit_exact_vs_oracle_on_all_weights"] is True
    assert pc["cfg5"]["parity"]["round_trip"]["events_with_dr_above_1e-10"] <= 1024
    assert "cuda_graph_replay_ms_per_step" in pc["cfg1"]
