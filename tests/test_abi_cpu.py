"""CPU-side checks of the C-ABI library: it loads without a GPU, exports every symbol include/madspace_b200.h
declares, and rejects bad arguments on the host before any launch (no compute calls here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import ms_inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
FAKE = 0x1000          # aligned, non-NULL, never dereferenced: validation failures return before any launch


@pytest.fixture(scope="module")
def ms():
    import paper_2602_06895_b200 as m
    m.lib()
    return m


def test_library_exports_every_declared_symbol(ms):
    header = open(os.path.join(ROOT, "include", "madspace_b200.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(ms_[a-z0-9_]+)\s*\(", header))
    assert {"ms_vegas_map", "ms_rambo_massless", "ms_fastrambo", "ms_fastrambo_inverse", "ms_massive_rescale",
            "ms_pdf_x_boost", "ms_unweight"} <= declared
    L = ms.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(ms.EXPORTS)
    assert "sm_100a" in ms.ms_version()


def test_struct_layouts_match_the_header(ms):
    assert C.sizeof(ms.ms_rng) == 24
    assert C.sizeof(ms.ms_gen_config) == 10 * 4 + 4 * 8 + 9 * 8


def test_check_grid(ms):
    assert ms.ms_check_grid(ms_inputs.uniform_grid(5, 64)) == ms.MS_OK
    assert ms.ms_check_grid(ms_inputs.seeded_grid(20, 128)) == ms.MS_OK
    bad = ms_inputs.seeded_grid(3, 16)
    bad[1, 5] = bad[1, 4]
    assert ms.ms_check_grid(bad) == ms.MS_EGRID
    bad = ms_inputs.uniform_grid(2, 8)
    bad[0, 0] = 1e-9
    assert ms.ms_check_grid(bad) == ms.MS_EGRID
    bad = ms_inputs.uniform_grid(2, 8)
    bad[1, -1] = 0.999
    assert ms.ms_check_grid(bad) == ms.MS_EGRID
    assert ms.ms_check_grid(np.zeros((40, 9))) == ms.MS_EINVAL          # d > MS_MAX_DIMS


def _code(ms, fn, *args):
    with pytest.raises(ms.MadSpaceError) as ei:
        fn(*args)
    return ei.value.code


def test_host_side_argument_errors(ms):
    r0 = ms.rng(1)
    # n out of range, NULL / misaligned pointers, ld < N
    assert _code(ms, ms.ms_fastrambo, 8, 10, 1000.0, None, None, r0, FAKE, FAKE, 8, None, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_fastrambo, 8, 1, 1000.0, None, None, r0, FAKE, FAKE, 8, None, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_fastrambo, 8, 4, 1000.0, None, None, r0, None, FAKE, 8, None, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_fastrambo, 8, 4, 1000.0, None, None, r0, FAKE + 8, FAKE, 8, None, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_fastrambo, 8, 4, 1000.0, None, None, r0, FAKE, FAKE, 7, None, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_rambo_massless, -1, 4, 1000.0, None, None, r0, FAKE, FAKE, 8, None, 0) == ms.MS_EINVAL
    # no energy at all
    assert _code(ms, ms.ms_rambo_massless, 8, 4, 0.0, None, None, r0, FAKE, FAKE, 8, None, 0) == ms.MS_EKIN
    # masses
    assert _code(ms, ms.ms_massive_rescale, 8, 4, 300.0, (173.0, 173.0, 0.0, 0.0), 1e-14, 10, FAKE, FAKE, 8, None, 0) == ms.MS_EKIN
    assert _code(ms, ms.ms_massive_rescale, 8, 4, 2000.0, (173.0, -1.0, 0.0, 0.0), 1e-14, 10, FAKE, FAKE, 8, None, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_rambo_massive_reweight, 8, 4, "fastrambo", 300.0, (173.0, 173.0, 0.0, 0.0), None, r0, FAKE, FAKE, 8, None, 0) == ms.MS_EKIN
    assert _code(ms, ms.ms_rambo_massive_reweight, 8, 4, "rambo", 2000.0, (173.0, 173.0, 0.0, 0.0), None, r0, None, FAKE, 8, None, 0) == ms.MS_EINVAL
    # tau_min
    assert _code(ms, ms.ms_pdf_x_boost, 8, 5, 1e8, 1.5, 0, None, r0, FAKE, FAKE, FAKE, None, 8, 0) == ms.MS_EKIN
    assert _code(ms, ms.ms_pdf_x_boost, 8, 5, 1e8, 0.1, 2, None, r0, FAKE, FAKE, FAKE, None, 8, 0) == ms.MS_EINVAL
    # VEGAS
    assert _code(ms, ms.ms_vegas_map, 8, 5, 64, FAKE, 1, None, r0, FAKE, None, 8, 0) == ms.MS_EINVAL   # inverse needs x
    assert _code(ms, ms.ms_vegas_map, 8, 5, 64, FAKE, 3, FAKE, r0, FAKE, None, 8, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_vegas_map, 8, 32, 1024, FAKE, 0, FAKE, r0, FAKE, None, 8, 0) == ms.MS_EINVAL  # table > smem
    # fused call: grid smaller than the uniforms the map consumes
    cfg = ms.gen_config(5, "rambo", 13600.0, 12, 64, pdf=True, tau_min=1e-3)
    assert _code(ms, ms.ms_generate, cfg, 8, r0, FAKE, FAKE, FAKE, None, 8, None, 0) == ms.MS_EINVAL
    cfg = ms.gen_config(4, "fastrambo", 300.0, masses=(173.0, 173.0, 0.0, 0.0))
    assert _code(ms, ms.ms_generate, cfg, 8, r0, None, FAKE, FAKE, None, 8, None, 0) == ms.MS_EKIN
    # unweighting: scratch too small
    assert _code(ms, ms.ms_unweight, 1 << 20, FAKE, FAKE, ms.rng(3, 1), 0, None, 16, FAKE, FAKE, None, FAKE, FAKE, 64,
                 1 << 20, 0) == ms.MS_EINVAL
    # a non-zero reserved field is rejected
    bad = ms.ms_rng(1, 0, 5, 0)
    assert _code(ms, ms.ms_fastrambo, 8, 4, 1000.0, None, None, bad, FAKE, FAKE, 8, None, 0) == ms.MS_EINVAL


def test_round_2_entry_points_validate_on_the_host(ms):
    """ms_fastrambo_inverse_vegas and ms_unweight_static reject bad sizes before any CUDA call (no GPU needed)."""
    r1 = ms.rng(3, 1)
    # the grid must have exactly 3n-4 dimensions and 64 or 128 bins
    for gd, gb in ((7, 128), (9, 128), (8, 100), (8, 256), (8, 32)):
        assert _code(ms, ms.ms_fastrambo_inverse_vegas, 8, 4, FAKE, FAKE, gd, gb, FAKE, None, 8, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_fastrambo_inverse_vegas, 8, 4, FAKE, None, 8, 128, FAKE, None, 8, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_fastrambo_inverse_vegas, 8, 4, FAKE, FAKE, 8, 128, FAKE, None, 7, 0) == ms.MS_EINVAL     # ld < N
    assert _code(ms, ms.ms_fastrambo_inverse_vegas, (1 << 31) + 1, 4, FAKE, FAKE, 8, 128, FAKE, None, (1 << 31) + 2, 0) == ms.MS_EINVAL
    # beyond the static scratch: MS_ELIMIT, a code of its own
    big = ms.MS_UNWEIGHT_STATIC_MAX_EVENTS + 1
    assert _code(ms, ms.ms_unweight_static, big, FAKE, FAKE, r1, 0, None, 16, FAKE, FAKE, None, FAKE, big, 0) == ms.MS_ELIMIT
    assert ms.MS_ELIMIT == -5 and _code(ms, ms.ms_unweight_static, -1, FAKE, FAKE, r1, 0, None, 16, FAKE, FAKE, None, FAKE, 8, 0) == ms.MS_EINVAL
    header = open(os.path.join(ROOT, "include", "madspace_b200.h")).read()
    assert "#define MS_UNWEIGHT_STATIC_MAX_EVENTS ((int64_t)1 << 24)" in header and ms.MS_UNWEIGHT_STATIC_MAX_EVENTS == 1 << 24
    # the scratch the static array provides is what ms_unweight asks for at the maximum size
    assert ms.ms_unweight_scratch_bytes(1 << 24) == int(re.search(r"#define MS_UNWEIGHT_STATIC_SCRATCH_BYTES (\d+)", header).group(1))


def test_batches_beyond_the_32_bit_event_index_are_rejected(ms):
    """The per-multiplicity kernels index events with 32 bits; N > MS_MAX_EVENTS = 2^31 returns MS_EINVAL before any
    launch instead of silently processing N mod 2^32 events."""
    r0, big = ms.rng(1), (1 << 31) + 1
    assert _code(ms, ms.ms_fastrambo, big, 4, 1000.0, None, None, r0, FAKE, FAKE, big + 1, None, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_rambo_massless, 1 << 32, 4, 1000.0, None, None, r0, FAKE, FAKE, 1 << 32, None, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_rambo_massive_reweight, big, 4, "fastrambo", 2000.0, (173.0, 173.0, 0.0, 0.0), None, r0, FAKE, FAKE,
                 big + 1, None, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_fastrambo_inverse, big, 4, FAKE, FAKE, None, big + 1, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_rambo_massive_reweight_inverse, big, 4, (173.0, 173.0, 0.0, 0.0), FAKE, FAKE, None, big + 1, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_chili, big, 3, 1e8, None, None, None, None, r0, FAKE, FAKE, None, big + 1, 0) == ms.MS_EINVAL
    cfg = ms.gen_config(4, "fastrambo", 1000.0)
    assert _code(ms, ms.ms_generate, cfg, big, r0, None, FAKE, FAKE, None, big + 1, None, 0) == ms.MS_EINVAL


def test_fused_unweighting_entry_points_validate_on_the_host(ms):
    r0, ru = ms.rng(1), ms.rng(3, 1)
    cfg = ms.gen_config(4, "fastrambo", 1000.0, toy=True)
    # the decision needs w_max and a bit array; a non-zero reserved field of either rng is rejected
    assert _code(ms, ms.ms_generate_unweight, cfg, 8, r0, None, FAKE, FAKE, None, 8, None, FAKE, ru, None, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_generate_unweight, cfg, 8, r0, None, FAKE, FAKE, None, 8, None, None, ru, FAKE, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_generate_unweight, cfg, 8, r0, None, FAKE, FAKE, None, 8, None, FAKE, ms.ms_rng(3, 1, 7, 0), FAKE, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_generate_unweight, cfg, 8, r0, None, FAKE, FAKE, None, 1 << 33, None, FAKE, ru, FAKE, 0) == ms.MS_EINVAL   # ld >= 2^32
    # one ballot word per 32 events, in whole 256-event tiles
    assert [ms.ms_accept_bits_words(n) for n in (0, 1, 256, 257, 1 << 24)] == [0, 8, 8, 16, 1 << 19]
    # compaction: bits required, scratch as for ms_unweight
    assert _code(ms, ms.ms_unweight_compact, 1 << 20, FAKE, FAKE, None, 0, None, 16, FAKE, FAKE, None, FAKE, FAKE,
                 ms.ms_unweight_scratch_bytes(1 << 20), 1 << 20, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_unweight_compact, 1 << 20, FAKE, FAKE, FAKE, 0, None, 16, FAKE, FAKE, None, FAKE, FAKE, 64,
                 1 << 20, 0) == ms.MS_EINVAL
    # gather: row stride of the output must hold K entries; NULL index list
    assert _code(ms, ms.ms_gather, 10, FAKE, 2, FAKE, 100, FAKE, 5, 0, None, 0) == ms.MS_EINVAL
    assert _code(ms, ms.ms_gather, 10, None, 2, FAKE, 100, FAKE, 10, 0, None, 0) == ms.MS_EINVAL
    ms.ms_gather(0, None, 2, None, 0, None, 0, 0, None, 0)
    # the VEGAS inverse runs in place or on disjoint buffers, never on partially overlapping ones
    assert _code(ms, ms.ms_vegas_map, 1000, 5, 64, FAKE, 1, 0x100000, r0, 0x100000 + 4096, None, 1000, 0) == ms.MS_EINVAL


def test_empty_batches_are_no_ops(ms):
    r0 = ms.rng(1)
    ms.ms_fastrambo(0, 4, 1000.0, None, None, r0, FAKE, FAKE, 0, None, 0)
    ms.ms_fastrambo_inverse(0, 4, FAKE, FAKE, None, 0, 0)
    ms.ms_vegas_map(0, 5, 64, FAKE, 0, None, r0, FAKE, None, 0, 0)
    ms.ms_generate(ms.gen_config(3, "fastrambo", 1000.0), 0, r0, None, FAKE, FAKE, None, 0, None, 0)


def test_scratch_size(ms):
    """The query is the contract (cub style): positive, 256-byte granular, monotone, linear in N (the header
    states 68 B per 512 events plus 64 KB)."""
    sizes = [ms.ms_unweight_scratch_bytes(n) for n in (0, 1, 511, 512, 513, 1 << 16, 1 << 24, 1 << 26)]
    assert sizes[0] == 256 and all(b > 0 and b % 256 == 0 for b in sizes)
    assert sizes == sorted(sizes)
    assert 68 * ((1 << 24) // 512) <= sizes[6] <= 68 * ((1 << 24) // 512) + 65536 + 4096
    assert ms.ms_unweight_scratch_bytes(-1) == 0
