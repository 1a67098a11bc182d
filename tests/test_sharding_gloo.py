"""N > 1 host logic on CPU (gloo, world_size 2): event ranges, accepted-count exchange, global output offsets.

The generation path has no data-path collective: each rank owns a contiguous range of GLOBAL event
indices and the counter-based RNG makes its events identical to the single-process ones.  What is exchanged is one
int64 per rank.  Here two gloo processes each run the ORACLE on their shard and the test checks that
(1) the shards tile the batch, (2) concatenating the per-rank results reproduces the single-process result bit for
bit (weights, accepted indices, w_out), and (3) gather_counts / output_offsets place each rank's accepted events
where the single-process compaction puts them.
"""
from __future__ import annotations

import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

from paper_2602_06895_b200.sharding import output_offsets, shard_range, weak_range  # noqa: E402


def test_shard_ranges_tile_the_batch():
    for n in (0, 1, 7, 1 << 16, (1 << 16) + 3):
        for world in (1, 2, 3, 8):
            spans = [shard_range(n, r, world) for r in range(world)]
            assert spans[0][0] == 0
            assert sum(c for _, c in spans) == n
            for (o0, c0), (o1, _) in zip(spans, spans[1:]):
                assert o0 + c0 == o1
            assert max(c for _, c in spans) - min(c for _, c in spans) <= 1
    assert weak_range(100, 3) == (300, 100)
    assert output_offsets([3, 0, 5]) == [0, 3, 3]
    with pytest.raises(ValueError):
        shard_range(10, 2, 2)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, n_total: int, q) -> None:
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      OMP_NUM_THREADS="2")
    import torch.distributed as dist

    import ms_inputs
    import oracle
    from oracle.chain import oracle_chain
    from paper_2602_06895_b200.sharding import gather_counts, output_offsets, shard_range

    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = ms_inputs.WORKLOADS["cfg2"]
        prerun = 1024
        offset, count = shard_range(n_total, rank, world)
        w = np.ascontiguousarray(oracle_chain(oracle, wl, np.arange(offset, offset + count))["w"])
        # every rank replays the same pre-run events for w_max: deterministic, no communication
        w_pre = np.ascontiguousarray(oracle_chain(oracle, wl, np.arange(prerun))["w"])
        wmax = oracle.wmax(w_pre)
        idx, w_out, n_acc = oracle.unweight(w, wmax, ms_inputs.SEED_UNWEIGHT, ms_inputs.STREAM_UNWEIGHT, offset, count)
        counts = gather_counts(n_acc)
        offs = output_offsets(counts)
        q.put((rank, offset, count, w, np.asarray(idx) + offset, np.asarray(w_out), counts, offs))
    finally:
        dist.destroy_process_group()


def test_two_ranks_reproduce_the_single_process_result(orc):
    import torch.multiprocessing as mp

    import ms_inputs
    from oracle.chain import oracle_chain

    n_total, world, prerun = 6000 + 7, 2, 1024
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_total, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted((q.get(timeout=300) for _ in range(world)), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0

    wl = ms_inputs.WORKLOADS["cfg2"]
    w_ref = np.ascontiguousarray(oracle_chain(orc, wl, np.arange(n_total))["w"])
    wmax = orc.wmax(np.ascontiguousarray(w_ref[:prerun]))
    idx_ref, wout_ref, nacc_ref = orc.unweight(w_ref, wmax, ms_inputs.SEED_UNWEIGHT, ms_inputs.STREAM_UNWEIGHT, 0, n_total)

    assert np.array_equal(np.concatenate([g[3] for g in got]), w_ref)          # events independent of the sharding
    counts = got[0][6]
    assert counts == got[1][6] == [len(g[4]) for g in got]                      # all_gather of the accepted counts
    assert got[0][7] == got[1][7] == output_offsets(counts)
    assert sum(counts) == nacc_ref
    glob_idx, glob_w = np.empty(nacc_ref, dtype=np.int64), np.empty(nacc_ref)
    for (_, _, _, _, idx, w_out, _, offs), r in zip(got, range(world)):
        glob_idx[offs[r]:offs[r] + len(idx)] = idx
        glob_w[offs[r]:offs[r] + len(idx)] = w_out
    assert np.array_equal(glob_idx, np.asarray(idx_ref)) and np.array_equal(glob_w, np.asarray(wout_ref))
