"""N > 1 host logic on CPU (gloo, world_size 2): the path shards by independent batches with no data-path collective
(DESIGN.md section 8), so what there is to test is (a) every rank draws its OWN seeded batch, (b) a batch's result does
not depend on which rank computes it (checked with the oracle standing in for the device), (c) bench.py's
max-over-ranks timing reduction and whole-job aggregation."""
import os
import socket
import sys
from types import SimpleNamespace

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    import bench
    import datagen
    import oracle
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    args = SimpleNamespace(workload="tiny", duration=0.03)
    w = bench.get_workload(args, rank)
    x = datagen.generate(w, chans=[0, 1], n_threads=1)
    cfg = oracle.OracleConfig(2, w.chan_width_hz * 2, w.f_center_hz - 0.5 * w.bw_hz + w.chan_width_hz,
                              w.dm_trials, w.n_fft, w.n_int)
    out = oracle.dedisp(cfg, x)
    # fake per-rank step times: rank r took (r + 1) ms
    t_max = bench.reduce_max_over_ranks(float(rank + 1), world, "cpu")
    # gather the input digests so rank 0 can check the batches differ
    digest = torch.tensor([float(np.abs(x.astype(np.int64)).sum()), float(out.sum())], dtype=torch.float64)
    got = [torch.zeros(2, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(got, digest)
    dist.barrier()
    if rank == 0:
        q.put({"seed": [w.seed], "t_max": t_max, "digests": [g.tolist() for g in got], "shape": list(out.shape)})
    dist.destroy_process_group()


def test_two_ranks_draw_independent_batches_and_reduce_max():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res["t_max"] == 2.0                       # MAX over ranks, not rank 0's own time
    d0, d1 = res["digests"]
    assert d0 != d1                                  # rank-local seeds: different batches
    assert res["shape"][2] > 0


def test_rank_batch_is_reproducible_anywhere():
    """A rank's batch depends on (workload, rank) only: recomputing rank 1's batch in this process gives the same
    input, hence the same output, as any other process would get."""
    sys.path.insert(0, ROOT)
    import bench
    import datagen
    args = SimpleNamespace(workload="tiny", duration=0.03)
    a = datagen.generate(bench.get_workload(args, 1), chans=[0, 1], n_threads=1)
    b = datagen.generate(bench.get_workload(args, 1), chans=[1], n_threads=1)
    c = datagen.generate(bench.get_workload(args, 0), chans=[1], n_threads=1)
    assert np.array_equal(a[:, 1], b[:, 0])
    assert not np.array_equal(b, c)


def test_whole_job_value_is_the_sum_over_ranks():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.whole_job_value(1_000_000, 1, 1e-3) == pytest.approx(1000.0)
    assert bench.whole_job_value(1_000_000, 8, 1e-3) == pytest.approx(8000.0)
