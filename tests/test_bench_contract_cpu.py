"""bench.py's contract, as far as it can be checked without a GPU: the reference arm (the oracle timed on the host cores)
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
    # the hand count grows with the multiplicity and with every optional stage
    c = {k: bench.alg_fp64_per_event(ms_inputs.WORKLOADS[k]) for k in ms_inputs.WORKLOADS}
    assert c["cfg1"] < c["cfg2"] < c["cfg5"] and c["cfg4rw"] < c["cfg4"]
