"""SURVEY.md section 5 ("Race detection / sanitizers"): the oracle built with -fsanitize=address,undefined and run over one
small chain per BASELINE.json config (plus unweighting and the inverse round trip) in a subprocess -- an out-of-bounds
access, a use of uninitialised stack through UB, a signed overflow or a misaligned access aborts the child.

The child imports only ``oracle`` and ``ms_inputs``; libasan has to be preloaded because the interpreter itself is not
instrumented.  Leak checking is off (CPython's own allocations)."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r"""
import numpy as np
import ms_inputs
import oracle
from oracle.chain import oracle_chain
oracle.lib()
assert oracle._SO.endswith("libms_oracle_san.so")
N = 777
for name, wl in ms_inputs.WORKLOADS.items():
    ref = oracle_chain(oracle, wl, np.arange(5, 5 + N))
    assert np.all(np.isfinite(ref["w"])) and np.all(ref["w"] > 0), name
    if wl.unweight:
        w = np.ascontiguousarray(ref["w"])
        idx, wout, nacc = oracle.unweight(w, oracle.wmax(np.ascontiguousarray(w[:100])), ms_inputs.SEED_UNWEIGHT, 1, 5, N)
        assert 0 < nacc <= N
    if wl.inverse:
        xi, wi = oracle.fastrambo_inverse(wl.n, ref["p"])
        r, _ = oracle.vegas_inverse(np.ascontiguousarray(wl.grid()[:3 * wl.n - 4]), xi)
        assert np.max(np.abs(r - ref["r"][:3 * wl.n - 4])) < 1e-6
# the ragged ends: one event, and the literal __float128 evaluator
one = oracle_chain(oracle, ms_inputs.WORKLOADS["cfg5"], np.arange(1))
x = oracle.fill_uniforms(33, 8, 1, 0, 0)
oracle.lit_rambo(4, x, 1000.0)
oracle.lit_rambo(4, x, 1000.0, exact=True)
print("sanitized oracle ok")
"""


def test_oracle_under_address_and_undefined_behaviour_sanitizers():
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("gcc has no libasan on this box")
    env = dict(os.environ, MS_ORACLE_SANITIZE="1", LD_PRELOAD=asan, PYTHONPATH=ROOT,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1:halt_on_error=1", UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1",
               OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-c", CHILD], capture_output=True, text=True, env=env, cwd=ROOT, timeout=600)
    assert r.returncode == 0, "sanitized oracle failed:\n%s\n%s" % (r.stdout[-2000:], r.stderr[-6000:])
    assert "sanitized oracle ok" in r.stdout
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr
