"""paper_2602_06895_b200 -- B200-native (sm_100a) hot path of MadSpace (arXiv 2602.06895).

Thin ctypes binding of ``libmadspace_b200.so`` (C ABI: ``include/madspace_b200.h``).  The functions here carry
the SAME names as the C entry points and do argument marshalling only: every step of the path runs in the
library's CUDA kernels.  PyTorch is used for device memory and streams, nothing else.  There is NO CPU
fallback: if the library cannot be built/loaded the import of a function raises, and every call raises
``MadSpaceError`` on a non-zero return code.

Layout: structure of arrays, fp64, ``a[row, event]`` (C-contiguous torch tensors on the device); momentum
row = 4*particle + mu with mu = (E, px, py, pz), particles 0,1 incoming, 2..n+1 outgoing.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass, field
from typing import Optional, Sequence

from . import _build

MS_MAX_N = 9
MS_OK, MS_EINVAL, MS_EGRID, MS_EKIN, MS_ECUDA, MS_ELIMIT = 0, -1, -2, -3, -4, -5
_ERR = {MS_EINVAL: "MS_EINVAL", MS_EGRID: "MS_EGRID", MS_EKIN: "MS_EKIN", MS_ECUDA: "MS_ECUDA", MS_ELIMIT: "MS_ELIMIT"}
MS_UNWEIGHT_STATIC_MAX_EVENTS = 1 << 24

EXPORTS = ("ms_version", "ms_last_cuda_error", "ms_check_grid", "ms_vegas_map", "ms_vegas_accumulate", "ms_vegas_refine", "ms_rambo_massless", "ms_fastrambo",
           "ms_fastrambo_inverse", "ms_massive_rescale", "ms_rambo_massive_reweight", "ms_rambo_massive_reweight_inverse", "ms_chili", "ms_pdf_x_boost", "ms_toy_integrand", "ms_reduce_max",
           "ms_unweight_scratch_bytes", "ms_unweight", "ms_unweight_static", "ms_fastrambo_inverse_vegas", "ms_weight_histogram", "ms_wmax_from_histogram", "ms_elementwise_max", "ms_gather", "ms_observable", "ms_cut", "ms_histogram_fill", "ms_invariant_map", "ms_generate", "ms_generate_unweight", "ms_unweight_compact", "ms_accept_bits_words", "ms_fill_uniforms")


class MadSpaceError(RuntimeError):
    def __init__(self, fn: str, code: int, cuda: int = 0):
        self.code, self.cuda = code, cuda
        super().__init__("%s failed: %s%s" % (fn, _ERR.get(code, str(code)),
                                              " (cudaError %d)" % cuda if code == MS_ECUDA else ""))


class ms_rng(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("stream", C.c_uint32), ("reserved", C.c_uint32), ("event_offset", C.c_uint64)]


class ms_gen_config(C.Structure):
    _fields_ = [("n", C.c_int32), ("mapping", C.c_int32), ("grid_dims", C.c_int32), ("grid_bins", C.c_int32),
                ("pdf", C.c_int32), ("massive", C.c_int32), ("toy", C.c_int32), ("max_iter", C.c_int32),
                ("tail_unit_jacobian", C.c_int32), ("reserved", C.c_int32),
                ("sqrt_s", C.c_double), ("tau_min", C.c_double), ("rel_tol", C.c_double), ("toy_reg", C.c_double),
                ("masses", C.c_double * MS_MAX_N)]


_lib = None
_vp, _i64, _int, _dbl = C.c_void_p, C.c_int64, C.c_int, C.c_double


def lib_path() -> str:
    return _build.LIB


def lib() -> C.CDLL:
    """Load (building first if the sources are newer) the CUDA library.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        L.ms_version.restype = C.c_char_p
        L.ms_unweight_scratch_bytes.restype = C.c_size_t
        L.ms_unweight_scratch_bytes.argtypes = [_i64]
        L.ms_check_grid.argtypes = [_int, _int, _vp]
        L.ms_fill_uniforms.argtypes = [_i64, _int, ms_rng, _vp, _i64, _vp]
        L.ms_invariant_map.argtypes = [_i64, _int, _int, _dbl, _dbl, _vp, _vp, _dbl, _dbl, _vp, _vp, _vp, _vp]
        L.ms_observable.argtypes = [_i64, _int, _int, _int, _int, _vp, _vp, _i64, _vp]
        L.ms_cut.argtypes = [_i64, _vp, _dbl, _dbl, _vp, _vp]
        L.ms_histogram_fill.argtypes = [_i64, _vp, _vp, _dbl, _dbl, _int, _vp, _vp, _vp]
        L.ms_weight_histogram.argtypes = [_i64, _vp, _vp, _vp]
        L.ms_wmax_from_histogram.argtypes = [_vp, _dbl, _vp]
        L.ms_elementwise_max.argtypes = [_i64, _vp, _vp, _vp, _vp]
        L.ms_gather.argtypes = [_i64, _vp, _int, _vp, _i64, _vp, _i64, _i64, _vp, _vp]
        L.ms_vegas_accumulate.argtypes = [_i64, _int, _int, _vp, ms_rng, _vp, _vp]
        L.ms_vegas_refine.argtypes = [_int, _int, _vp, _dbl, _vp, _vp]
        L.ms_vegas_map.argtypes = [_i64, _int, _int, _vp, _int, _vp, ms_rng, _vp, _vp, _i64, _vp]
        for name in ("ms_rambo_massless", "ms_fastrambo"):
            getattr(L, name).argtypes = [_i64, _int, _dbl, _vp, _vp, ms_rng, _vp, _vp, _i64, _vp, _vp]
        L.ms_fastrambo_inverse.argtypes = [_i64, _int, _vp, _vp, _vp, _i64, _vp]
        L.ms_chili.argtypes = [_i64, _int, _dbl, _vp, _vp, _vp, _vp, ms_rng, _vp, _vp, _vp, _i64, _vp]
        L.ms_rambo_massive_reweight_inverse.argtypes = [_i64, _int, _vp, _vp, _vp, _vp, _i64, _vp]
        L.ms_rambo_massive_reweight.argtypes = [_i64, _int, _int, _dbl, _vp, _vp, ms_rng, _vp, _vp, _i64, _vp, _vp]
        L.ms_massive_rescale.argtypes = [_i64, _int, _dbl, _vp, _dbl, _int, _vp, _vp, _i64, _vp, _vp]
        L.ms_pdf_x_boost.argtypes = [_i64, _int, _dbl, _dbl, _int, _vp, ms_rng, _vp, _vp, _vp, _vp, _i64, _vp]
        L.ms_toy_integrand.argtypes = [_i64, _int, _dbl, _vp, _vp, _int, _i64, _vp]
        L.ms_reduce_max.argtypes = [_i64, _vp, _vp, _vp]
        L.ms_unweight.argtypes = [_i64, _vp, _vp, ms_rng, _int, _vp, _i64, _vp, _vp, _vp, _vp, _vp, C.c_size_t, _i64, _vp]
        L.ms_fastrambo_inverse_vegas.argtypes = [_i64, _int, _vp, _vp, _int, _int, _vp, _vp, _i64, _vp]
        L.ms_unweight_static.argtypes = [_i64, _vp, _vp, ms_rng, _int, _vp, _i64, _vp, _vp, _vp, _vp, _i64, _vp]
        L.ms_generate.argtypes = [C.POINTER(ms_gen_config), _i64, ms_rng, _vp, _vp, _vp, _vp, _i64, _vp, _vp]
        L.ms_generate_unweight.argtypes = [C.POINTER(ms_gen_config), _i64, ms_rng, _vp, _vp, _vp, _vp, _i64, _vp, _vp, ms_rng, _vp, _vp]
        L.ms_unweight_compact.argtypes = [_i64, _vp, _vp, _vp, _int, _vp, _i64, _vp, _vp, _vp, _vp, _vp, C.c_size_t, _i64, _vp]
        L.ms_accept_bits_words.restype = C.c_size_t
        L.ms_accept_bits_words.argtypes = [_i64]
        _lib = L
    return _lib


def _ptr(t) -> Optional[int]:
    """Device (or host) address of a torch tensor / numpy array / raw int; None stays NULL."""
    if t is None:
        return None
    if isinstance(t, int):
        return t
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def _stream(stream) -> Optional[int]:
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def _check(fn: str, rc: int) -> None:
    if rc != MS_OK:
        raise MadSpaceError(fn, rc, lib().ms_last_cuda_error() if rc == MS_ECUDA else 0)


def rng(seed: int, stream: int = 0, event_offset: int = 0) -> ms_rng:
    return ms_rng(seed, stream, 0, event_offset)


# ----------------------------------------------------------------------------------------------- C ABI mirrors

def ms_version() -> str:
    return lib().ms_version().decode()


def ms_last_cuda_error() -> int:
    return int(lib().ms_last_cuda_error())


def ms_check_grid(h_edges) -> int:
    """h_edges: numpy float64 [d][n_bins+1] on the host.  Returns the code (does not raise on MS_EGRID)."""
    d, nb1 = h_edges.shape
    return int(lib().ms_check_grid(d, nb1 - 1, h_edges.ctypes.data))


def ms_fill_uniforms(N, d, r: ms_rng, d_r, ld, stream=None) -> None:
    _check("ms_fill_uniforms", lib().ms_fill_uniforms(N, d, r, _ptr(d_r), ld, _stream(stream)))


def ms_vegas_map(N, d, n_bins, d_edges, direction, d_in, r: ms_rng, d_out, d_jac, ld, stream=None) -> None:
    _check("ms_vegas_map", lib().ms_vegas_map(N, d, n_bins, _ptr(d_edges), direction, _ptr(d_in), r, _ptr(d_out),
                                              _ptr(d_jac), ld, _stream(stream)))


def ms_rambo_massless(N, n, sqrt_s, d_sqrt_s, d_x, r: ms_rng, d_p, d_w, ld, d_fail=None, stream=None) -> None:
    _check("ms_rambo_massless", lib().ms_rambo_massless(N, n, sqrt_s, _ptr(d_sqrt_s), _ptr(d_x), r, _ptr(d_p), _ptr(d_w),
                                                        ld, _ptr(d_fail), _stream(stream)))


def ms_fastrambo(N, n, sqrt_s, d_sqrt_s, d_x, r: ms_rng, d_p, d_w, ld, d_fail=None, stream=None) -> None:
    _check("ms_fastrambo", lib().ms_fastrambo(N, n, sqrt_s, _ptr(d_sqrt_s), _ptr(d_x), r, _ptr(d_p), _ptr(d_w), ld,
                                              _ptr(d_fail), _stream(stream)))


def ms_fastrambo_inverse(N, n, d_p, d_x, d_w, ld, stream=None) -> None:
    _check("ms_fastrambo_inverse", lib().ms_fastrambo_inverse(N, n, _ptr(d_p), _ptr(d_x), _ptr(d_w), ld, _stream(stream)))


def ms_fastrambo_inverse_vegas(N, n, d_p, d_edges, grid_dims, grid_bins, d_r, d_w, ld, stream=None) -> None:
    _check("ms_fastrambo_inverse_vegas", lib().ms_fastrambo_inverse_vegas(N, n, _ptr(d_p), _ptr(d_edges), grid_dims, grid_bins,
                                                                          _ptr(d_r), _ptr(d_w), ld, _stream(stream)))


def ms_massive_rescale(N, n, sqrt_s, masses: Sequence[float], rel_tol, max_iter, d_p, d_w, ld, d_fail=None,
                       stream=None) -> None:
    h = (C.c_double * len(masses))(*[float(m) for m in masses])
    if len(masses) != n:
        raise MadSpaceError("ms_massive_rescale", MS_EINVAL)
    _check("ms_massive_rescale", lib().ms_massive_rescale(N, n, sqrt_s, C.addressof(h), rel_tol, max_iter, _ptr(d_p),
                                                          _ptr(d_w), ld, _ptr(d_fail), _stream(stream)))


def ms_pdf_x_boost(N, n, s_had, tau_min, phase, d_r, r: ms_rng, d_x1x2, d_sqrt_shat, d_jac, d_p, ld, stream=None) -> None:
    _check("ms_pdf_x_boost", lib().ms_pdf_x_boost(N, n, s_had, tau_min, phase, _ptr(d_r), r, _ptr(d_x1x2),
                                                  _ptr(d_sqrt_shat), _ptr(d_jac), _ptr(d_p), ld, _stream(stream)))


def ms_toy_integrand(N, n, reg, d_p, d_f, accumulate, ld, stream=None) -> None:
    _check("ms_toy_integrand", lib().ms_toy_integrand(N, n, reg, _ptr(d_p), _ptr(d_f), int(accumulate), ld, _stream(stream)))


def ms_reduce_max(N, d_w, d_out, stream=None) -> None:
    _check("ms_reduce_max", lib().ms_reduce_max(N, _ptr(d_w), _ptr(d_out), _stream(stream)))


def ms_unweight_scratch_bytes(N) -> int:
    return int(lib().ms_unweight_scratch_bytes(N))


def ms_unweight(N, d_w, d_wmax, r: ms_rng, n_rows, d_rows_in, cap, d_idx, d_w_out, d_rows_out, d_n_accepted, d_scratch,
                scratch_bytes, ld, stream=None) -> None:
    _check("ms_unweight", lib().ms_unweight(N, _ptr(d_w), _ptr(d_wmax), r, n_rows, _ptr(d_rows_in), cap, _ptr(d_idx),
                                            _ptr(d_w_out), _ptr(d_rows_out), _ptr(d_n_accepted), _ptr(d_scratch),
                                            scratch_bytes, ld, _stream(stream)))


def ms_unweight_static(N, d_w, d_wmax, r: ms_rng, n_rows, d_rows_in, cap, d_idx, d_w_out, d_rows_out, d_n_accepted, ld,
                       stream=None) -> None:
    _check("ms_unweight_static", lib().ms_unweight_static(N, _ptr(d_w), _ptr(d_wmax), r, n_rows, _ptr(d_rows_in), cap,
                                                          _ptr(d_idx), _ptr(d_w_out), _ptr(d_rows_out), _ptr(d_n_accepted),
                                                          ld, _stream(stream)))


def gen_config(n, mapping="fastrambo", sqrt_s=0.0, grid_dims=0, grid_bins=0, pdf=False, tau_min=0.0, masses=(),
               rel_tol=1e-14, max_iter=10, toy=False, toy_reg=100.0, tail_unit_jacobian=False,
               massive_mode="rescale") -> ms_gen_config:
    cfg = ms_gen_config()
    cfg.n, cfg.mapping = n, {"fastrambo": 0, "rambo": 1}[mapping]
    cfg.grid_dims, cfg.grid_bins = grid_dims, grid_bins
    cfg.pdf, cfg.toy, cfg.max_iter = int(pdf), int(toy), max_iter
    cfg.massive = {"rescale": 1, "reweight": 2}[massive_mode] if len(masses) > 0 else 0
    cfg.sqrt_s, cfg.tau_min, cfg.rel_tol, cfg.toy_reg = sqrt_s, tau_min, rel_tol, toy_reg
    cfg.tail_unit_jacobian, cfg.reserved = int(tail_unit_jacobian), 0
    for i, m in enumerate(masses):
        cfg.masses[i] = float(m)
    return cfg


def ms_generate(cfg: ms_gen_config, N, r: ms_rng, d_edges, d_p, d_w, d_x1x2, ld, d_fail=None, stream=None) -> None:
    _check("ms_generate", lib().ms_generate(C.byref(cfg), N, r, _ptr(d_edges), _ptr(d_p), _ptr(d_w), _ptr(d_x1x2), ld,
                                            _ptr(d_fail), _stream(stream)))


def ms_accept_bits_words(N) -> int:
    return int(lib().ms_accept_bits_words(N))


def ms_generate_unweight(cfg: ms_gen_config, N, r: ms_rng, d_edges, d_p, d_w, d_x1x2, ld, d_fail, d_wmax, r_unweight: ms_rng,
                         d_accept_bits, stream=None) -> None:
    _check("ms_generate_unweight", lib().ms_generate_unweight(C.byref(cfg), N, r, _ptr(d_edges), _ptr(d_p), _ptr(d_w),
                                                              _ptr(d_x1x2), ld, _ptr(d_fail), _ptr(d_wmax), r_unweight,
                                                              _ptr(d_accept_bits), _stream(stream)))


def ms_unweight_compact(N, d_w, d_wmax, d_accept_bits, n_rows, d_rows_in, cap, d_idx, d_w_out, d_rows_out, d_n_accepted,
                        d_scratch, scratch_bytes, ld, stream=None) -> None:
    _check("ms_unweight_compact", lib().ms_unweight_compact(N, _ptr(d_w), _ptr(d_wmax), _ptr(d_accept_bits), n_rows,
                                                            _ptr(d_rows_in), cap, _ptr(d_idx), _ptr(d_w_out), _ptr(d_rows_out),
                                                            _ptr(d_n_accepted), _ptr(d_scratch), scratch_bytes, ld,
                                                            _stream(stream)))


def ms_rambo_massive_reweight(N, n, mapping, sqrt_s, masses: Sequence[float], d_x, r: ms_rng, d_p, d_w, ld,
                              d_fail=None, stream=None) -> None:
    if len(masses) != n:
        raise MadSpaceError("ms_rambo_massive_reweight", MS_EINVAL)
    h = (C.c_double * len(masses))(*[float(m) for m in masses])
    _check("ms_rambo_massive_reweight",
           lib().ms_rambo_massive_reweight(N, n, {"fastrambo": 0, "rambo": 1}[mapping], sqrt_s, C.addressof(h), _ptr(d_x),
                                           r, _ptr(d_p), _ptr(d_w), ld, _ptr(d_fail), _stream(stream)))


def ms_rambo_massive_reweight_inverse(N, n, masses: Sequence[float], d_p, d_x, d_w, ld, stream=None) -> None:
    if len(masses) != n:
        raise MadSpaceError("ms_rambo_massive_reweight_inverse", MS_EINVAL)
    h = (C.c_double * len(masses))(*[float(m) for m in masses])
    _check("ms_rambo_massive_reweight_inverse",
           lib().ms_rambo_massive_reweight_inverse(N, n, C.addressof(h), _ptr(d_p), _ptr(d_x), _ptr(d_w), ld,
                                                   _stream(stream)))


def ms_vegas_accumulate(N, d, n_bins, d_w, r: ms_rng, d_hist, stream=None) -> None:
    _check("ms_vegas_accumulate", lib().ms_vegas_accumulate(N, d, n_bins, _ptr(d_w), r, _ptr(d_hist), _stream(stream)))


def ms_vegas_refine(h_hist, h_edges, alpha=0.5):
    """Host arrays in, refined host edges out (numpy, C-contiguous float64)."""
    import numpy as np
    h_hist = np.ascontiguousarray(h_hist, dtype=np.float64)
    h_edges = np.ascontiguousarray(h_edges, dtype=np.float64)
    d, nb = h_hist.shape
    if h_edges.shape != (d, nb + 1):
        raise MadSpaceError("ms_vegas_refine", MS_EINVAL)
    out = np.empty_like(h_edges)
    _check("ms_vegas_refine", lib().ms_vegas_refine(d, nb, h_hist.ctypes.data, float(alpha), h_edges.ctypes.data,
                                                    out.ctypes.data))
    return out


MS_HIST_BINS = 1 << 15


def ms_weight_histogram(N, d_w, d_counts, stream=None) -> None:
    _check("ms_weight_histogram", lib().ms_weight_histogram(N, _ptr(d_w), _ptr(d_counts), _stream(stream)))


def ms_wmax_from_histogram(h_counts, fraction) -> float:
    """h_counts: numpy uint64/int64 [MS_HIST_BINS] on the host."""
    import numpy as np
    h = np.ascontiguousarray(h_counts).view(np.uint64)
    if h.shape != (MS_HIST_BINS,):
        raise MadSpaceError("ms_wmax_from_histogram", MS_EINVAL)
    out = C.c_double(0.0)
    _check("ms_wmax_from_histogram", lib().ms_wmax_from_histogram(h.ctypes.data, float(fraction), C.addressof(out)))
    return float(out.value)


def ms_elementwise_max(N, d_a, d_b, d_out, stream=None) -> None:
    _check("ms_elementwise_max", lib().ms_elementwise_max(N, _ptr(d_a), _ptr(d_b), _ptr(d_out), _stream(stream)))


def ms_gather(K, d_idx, n_rows, d_in, ld_in, d_out, ld_out, idx_add=0, d_idx_out=None, stream=None) -> None:
    _check("ms_gather", lib().ms_gather(K, _ptr(d_idx), n_rows, _ptr(d_in), ld_in, _ptr(d_out), ld_out, idx_add,
                                        _ptr(d_idx_out), _stream(stream)))


def ms_chili(N, n, s_lab, masses, pt_min, y_cut, d_x, r: ms_rng, d_p, d_w, d_x1x2, ld, stream=None) -> None:
    def harr(v):
        if v is None:
            return None, None
        if len(v) != n:
            raise MadSpaceError("ms_chili", MS_EINVAL)
        a = (C.c_double * n)(*[float(t) for t in v])
        return a, C.addressof(a)
    keep = [harr(masses), harr(pt_min), harr(y_cut)]
    _check("ms_chili", lib().ms_chili(N, n, s_lab, keep[0][1], keep[1][1], keep[2][1], _ptr(d_x), r, _ptr(d_p), _ptr(d_w),
                                      _ptr(d_x1x2), ld, _stream(stream)))


OBS_KINDS = ("E", "PX", "PY", "PZ", "PT", "PABS", "PHI", "THETA", "Y", "ABSY", "ETA", "ABSETA", "DPHI", "DETA", "DR", "MASS",
             "SQRT_SHAT", "ET_TOT", "HT")


def ms_observable(N, kind: str, a, b, n_out, d_p, d_obs, ld, stream=None) -> None:
    _check("ms_observable", lib().ms_observable(N, OBS_KINDS.index(kind), a, b, n_out, _ptr(d_p), _ptr(d_obs), ld,
                                                _stream(stream)))


def ms_cut(N, d_obs, lo, hi, d_w, stream=None) -> None:
    _check("ms_cut", lib().ms_cut(N, _ptr(d_obs), float(lo), float(hi), _ptr(d_w), _stream(stream)))


def ms_histogram_fill(N, d_obs, d_w, lo, hi, n_bins, d_sum_w, d_sum_w2, stream=None) -> None:
    _check("ms_histogram_fill", lib().ms_histogram_fill(N, _ptr(d_obs), _ptr(d_w), float(lo), float(hi), n_bins,
                                                        _ptr(d_sum_w), _ptr(d_sum_w2), _stream(stream)))


MAP_KINDS = ("FLAT", "POWER", "BW")


def ms_invariant_map(N, kind: str, direction, x_min, x_max, m2, par, d_in, d_out, d_g=None, d_x_min=None, d_x_max=None,
                     stream=None) -> None:
    _check("ms_invariant_map", lib().ms_invariant_map(N, MAP_KINDS.index(kind), direction, float(x_min), float(x_max),
                                                      _ptr(d_x_min), _ptr(d_x_max), float(m2), float(par), _ptr(d_in),
                                                      _ptr(d_out), _ptr(d_g), _stream(stream)))
