"""oracle -- TEST INFRASTRUCTURE (not product code).

ctypes binding of the plain-C fp64 oracle in ``ms_oracle.c`` / ``ms_oracle_lit.c``.
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package; nothing under
``paper_2602_06895_b200/`` does, and this package imports nothing from there.

Arrays are numpy float64, structure of arrays ``a[row, event]`` (C-contiguous).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# MS_ORACLE_SANITIZE=1 (tests/test_oracle_sanitizers.py, in a subprocess with libasan preloaded): the same sources built
# with -fsanitize=address,undefined into a second library; the arithmetic flags are unchanged.
_SANITIZE = os.environ.get("MS_ORACLE_SANITIZE", "") == "1"
_SO = os.path.join(_HERE, "libms_oracle_san.so" if _SANITIZE else "libms_oracle.so")
_SRCS = [os.path.join(_HERE, "ms_oracle.c"), os.path.join(_HERE, "ms_oracle_lit.c")]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2 -ffp-contract=off: no FMA contraction)."""
    srcs = [s for s in _SRCS if os.path.exists(s)]
    if not force and os.path.exists(_SO) and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in srcs):
        return _SO
    tmp = _SO + ".tmp.%d" % os.getpid()
    opt = ["-O1", "-g", "-fno-omit-frame-pointer", "-fsanitize=address,undefined", "-fno-sanitize-recover=all"] if _SANITIZE \
        else ["-O2"]
    cmd = ["gcc", "-std=gnu11"] + opt + ["-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
                                         "-Wall", "-o", tmp] + srcs + ["-lquadmath", "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _SO)
    return _SO


_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int64)


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        L.orc_uniform.restype = C.c_double
        L.orc_uniform.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64, C.c_uint32]
        L.orc_phi_n.restype = C.c_double
        L.orc_phi_n.argtypes = [C.c_int, C.c_double]
        L.orc_ck.restype = C.c_double
        L.orc_ck.argtypes = [C.c_int]
        for name in ("orc_rqf_forward", "orc_rqf_density", "orc_rqf_inverse"):
            getattr(L, name).restype = C.c_double
            getattr(L, name).argtypes = [C.c_double, C.c_double]
        L.orc_rambo_mass_step.restype = C.c_int
        L.orc_rambo_mass_step.argtypes = [C.c_double, C.c_int, _dp, _dp]
        L.orc_massive_rescale.restype = C.c_int64
        L.orc_unweight.restype = C.c_int64
        L.orc_max.restype = C.c_double
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a):
    return a.ctypes.data_as(_dp) if a is not None else None


def _chk(a, rows=None):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    if rows is not None:
        assert a.shape[0] == rows, (a.shape, rows)
    return a


def num_threads() -> int:
    return int(lib().orc_num_threads())


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def uniform(seed, stream, event, j) -> float:
    return float(lib().orc_uniform(seed, stream, event, j))


def fill_uniforms(N, d, seed, stream=0, event_offset=0):
    r = np.empty((d, N), dtype=np.float64)
    lib().orc_fill_uniforms(C.c_int64(N), C.c_int(d), C.c_uint64(seed), C.c_uint32(stream),
                            C.c_uint64(event_offset), _p(r), C.c_int64(N))
    return r


def vegas_forward(edges, r):
    d, N = r.shape
    nb = edges.shape[1] - 1
    _chk(edges, d), _chk(r)
    x = np.empty_like(r)
    jac = np.empty(N)
    lib().orc_vegas_forward(C.c_int64(N), C.c_int(d), C.c_int(nb), _p(edges), _p(r), _p(x), _p(jac), C.c_int64(N))
    return x, jac


def vegas_inverse(edges, x):
    d, N = x.shape
    nb = edges.shape[1] - 1
    _chk(edges, d), _chk(x)
    r = np.empty_like(x)
    jac = np.empty(N)
    lib().orc_vegas_inverse(C.c_int64(N), C.c_int(d), C.c_int(nb), _p(edges), _p(x), _p(r), _p(jac), C.c_int64(N))
    return r, jac


def phi_n(n, E):
    return float(lib().orc_phi_n(n, E))


def ck(k):
    return float(lib().orc_ck(k))


def rqf_forward(y, c):
    return float(lib().orc_rqf_forward(y, c))


def rqf_density(y, c):
    return float(lib().orc_rqf_density(y, c))


def rqf_inverse(x, c):
    return float(lib().orc_rqf_inverse(x, c))


def rambo_mass_step(r, k):
    u, t = C.c_double(), C.c_double()
    it = lib().orc_rambo_mass_step(C.c_double(r), C.c_int(k), C.byref(u), C.byref(t))
    return u.value, t.value, int(it)


def _rambo(fn, n, x, sqrt_s):
    N = x.shape[1]
    _chk(x, 3 * n - 4)
    p = np.empty((4 * (n + 2), N))
    w = np.empty(N)
    if np.isscalar(sqrt_s):
        fn(C.c_int64(N), C.c_int(n), C.c_double(float(sqrt_s)), None, _p(x), _p(p), _p(w), C.c_int64(N))
    else:
        _chk(sqrt_s)
        fn(C.c_int64(N), C.c_int(n), C.c_double(-1.0), _p(sqrt_s), _p(x), _p(p), _p(w), C.c_int64(N))
    return p, w


def fastrambo(n, x, sqrt_s):
    return _rambo(lib().orc_fastrambo, n, x, sqrt_s)


def rambo_massless(n, x, sqrt_s):
    return _rambo(lib().orc_rambo_massless, n, x, sqrt_s)


def fastrambo_inverse(n, p):
    N = p.shape[1]
    _chk(p, 4 * (n + 2))
    x = np.empty((3 * n - 4, N))
    w = np.empty(N)
    lib().orc_fastrambo_inverse(C.c_int64(N), C.c_int(n), _p(p), _p(x), _p(w), C.c_int64(N))
    return x, w


def massive_rescale(n, sqrt_s, masses, p, w, rel_tol=1e-14, max_iter=10):
    """Returns (k, w*w_m, n_fail); inputs are not modified."""
    N = p.shape[1]
    _chk(p, 4 * (n + 2))
    p2, w2 = p.copy(), w.copy()
    m = np.ascontiguousarray(masses, dtype=np.float64)
    nf = lib().orc_massive_rescale(C.c_int64(N), C.c_int(n), C.c_double(sqrt_s), _p(m), C.c_double(rel_tol),
                                   C.c_int(max_iter), _p(p2), _p(w2), C.c_int64(N))
    return p2, w2, int(nf)


def rambo_massive_reweight(n, x, sqrt_s, masses, exact=False):
    """Massive phase space by reweighting (strategy (ii), Eq. 68-69).  Returns (p, w, n_bad)."""
    N = x.shape[1]
    _chk(x, 3 * n - 4)
    m = np.ascontiguousarray(masses, dtype=np.float64)
    assert m.shape[0] == n
    p = np.empty((4 * (n + 2), N))
    w = np.empty(N)
    lib().orc_rambo_massive_reweight.restype = C.c_int64
    nb = lib().orc_rambo_massive_reweight(C.c_int(int(exact)), C.c_int64(N), C.c_int(n), C.c_double(sqrt_s), _p(m),
                                          _p(x), _p(p), _p(w), C.c_int64(N))
    return p, w, int(nb)


def vegas_accumulate(d, n_bins, w, seed, stream=0, event_offset=0, hist=None):
    """hist[dim][bin of the event's uniform r_dim] += w^2 (VEGAS adaptation, accumulation pass; reading V-4)."""
    _chk(w)
    if hist is None:
        hist = np.zeros((d, n_bins))
    assert hist.shape == (d, n_bins) and hist.flags["C_CONTIGUOUS"]
    lib().orc_vegas_accumulate(C.c_int64(w.shape[0]), C.c_int(d), C.c_int(n_bins), _p(w), C.c_uint64(seed),
                               C.c_uint32(stream), C.c_uint64(event_offset), _p(hist))
    return hist


def rambo_massive_reweight_inverse(n, p, masses):
    """Inverse of rambo_massive_reweight (FastRambo u_i): returns (x, w)."""
    N = p.shape[1]
    _chk(p, 4 * (n + 2))
    m = np.ascontiguousarray(masses, dtype=np.float64)
    x = np.empty((3 * n - 4, N))
    w = np.empty(N)
    lib().orc_rambo_massive_reweight_inverse(C.c_int64(N), C.c_int(n), _p(m), _p(p), _p(x), _p(w), C.c_int64(N))
    return x, w


def pdf_x_sample(s_had, tau_min, r):
    N = r.shape[1]
    _chk(r)
    assert r.shape[0] >= 2
    x1x2 = np.empty((2, N))
    rs = np.empty(N)
    jac = np.empty(N)
    lib().orc_pdf_x_sample(C.c_int64(N), C.c_double(s_had), C.c_double(tau_min), _p(r), _p(x1x2), _p(rs), _p(jac),
                           C.c_int64(N))
    return x1x2, rs, jac


def pdf_boost(n, s_had, x1x2, p):
    N = p.shape[1]
    _chk(p, 4 * (n + 2)), _chk(x1x2, 2)
    p2 = p.copy()
    lib().orc_pdf_boost(C.c_int64(N), C.c_int(n), C.c_double(s_had), _p(x1x2), _p(p2), C.c_int64(N))
    return p2


def toy_integrand(n, p, reg=100.0):
    N = p.shape[1]
    _chk(p, 4 * (n + 2))
    f = np.empty(N)
    lib().orc_toy_integrand(C.c_int64(N), C.c_int(n), C.c_double(reg), _p(p), _p(f), C.c_int64(N))
    return f


def unweight(w, w_max, seed, stream=1, event_offset=0, cap=None):
    N = w.shape[0]
    _chk(w)
    cap = N if cap is None else cap
    idx = np.empty(cap, dtype=np.int64)
    wout = np.empty(cap)
    n_acc = lib().orc_unweight(C.c_int64(N), _p(w), C.c_double(w_max), C.c_uint64(seed), C.c_uint32(stream),
                               C.c_uint64(event_offset), C.c_int64(cap), idx.ctypes.data_as(_ip), _p(wout))
    m = min(int(n_acc), cap)
    return idx[:m].copy(), wout[:m].copy(), int(n_acc)


def wmax(w):
    _chk(w)
    return float(lib().orc_max(C.c_int64(w.shape[0]), _p(w)))


# ---- literal __float128 evaluator (ms_oracle_lit.c) -------------------------------------------

def lit_rambo(n, x, sqrt_s, exact=False):
    N = x.shape[1]
    _chk(x, 3 * n - 4)
    p = np.empty((4 * (n + 2), N))
    w = np.empty(N)
    if np.isscalar(sqrt_s):
        lib().lit_rambo(C.c_int(int(exact)), C.c_int64(N), C.c_int(n), C.c_double(float(sqrt_s)), None, _p(x),
                        _p(p), _p(w), C.c_int64(N))
    else:
        _chk(sqrt_s)
        lib().lit_rambo(C.c_int(int(exact)), C.c_int64(N), C.c_int(n), C.c_double(-1.0), _p(sqrt_s), _p(x),
                        _p(p), _p(w), C.c_int64(N))
    return p, w


def lit_pdf_x_sample(s_had, tau_min, r):
    N = r.shape[1]
    _chk(r)
    x1x2 = np.empty((2, N))
    rs = np.empty(N)
    jac = np.empty(N)
    lib().lit_pdf_x_sample(C.c_int64(N), C.c_double(s_had), C.c_double(tau_min), _p(r), _p(x1x2), _p(rs), _p(jac),
                           C.c_int64(N))
    return x1x2, rs, jac


def lit_massive_rescale(n, sqrt_s, masses, p, w):
    N = p.shape[1]
    p2, w2 = p.copy(), w.copy()
    m = np.ascontiguousarray(masses, dtype=np.float64)
    lib().lit_massive_rescale(C.c_int64(N), C.c_int(n), C.c_double(sqrt_s), _p(m), _p(p2), _p(w2), C.c_int64(N))
    return p2, w2
