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


# ----------------------------------------------------------------------------------------------------------------
# Channel-range shards (bench.py --shard channels, dedisp_plan_shard): every rank
# dedisperses its own contiguous channel range with the WHOLE band's framing -- the oracle stands in for the device --
# the ranges are gathered into the whole band's output, and the band sum is one all-reduce of the ranks' partial sums
# ----------------------------------------------------------------------------------------------------------------
def _shard_worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist
    import bench
    import datagen
    import oracle
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    args = SimpleNamespace(workload="tiny", duration=0.02, shard="channels")
    wb = replace_chans(bench.get_workload(args, rank), 6)               # 6 channels: ranges of 3 + 3
    c0, n = bench.channel_shard(wb.n_chan, rank, world)
    cfg = oracle.OracleConfig(wb.n_chan, wb.bw_hz, wb.f_center_hz, (10.0, -4.0), wb.n_fft, wb.n_int)
    head, tail, L = oracle.framing(cfg)
    x_loc = datagen.generate(wb, chans=range(c0, c0 + n), n_threads=1)   # the rank's own columns only
    # the oracle on a channel range with the band's framing: units (c, b) of the whole configuration
    x_full = np.zeros((x_loc.shape[0], wb.n_chan, 2), dtype=np.int8)
    x_full[:, c0:c0 + n] = x_loc                                         # the other columns are never read
    nb = oracle.n_blocks(cfg, x_loc.shape[0])
    per = L // cfg.n_int
    chans = np.repeat(np.arange(c0, c0 + n), nb)
    blocks = np.tile(np.arange(nb), n)
    units = oracle.dedisp_units(cfg, x_full, chans, blocks)             # [n*nb][n_dm][per]
    out_loc = units.reshape(n, nb, cfg.n_dm, per).transpose(2, 0, 1, 3).reshape(cfg.n_dm, n, nb * per)
    # band sum of the rank's channels on the band's common time axis, then the one exchange of the path
    n_ser = nb * per - max(int(oracle.band_shifts(cfg, d).max()) for d in range(cfg.n_dm))
    part = np.zeros((cfg.n_dm, n_ser))
    for d in range(cfg.n_dm):
        sh = oracle.band_shifts(cfg, d)
        for c in range(c0, c0 + n):
            part[d] += out_loc[d, c - c0, sh[c]: sh[c] + n_ser]
    t_part = torch.from_numpy(part.copy())
    dist.all_reduce(t_part)
    gathered = [torch.zeros(cfg.n_dm, n, nb * per, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(gathered, torch.from_numpy(np.ascontiguousarray(out_loc)))
    samples = torch.tensor([float(n * nb * L)], dtype=torch.float64)
    dist.all_reduce(samples)
    dist.barrier()
    if rank == 0:
        x_all = datagen.generate(wb, n_threads=1)
        whole = oracle.dedisp(cfg, x_all)
        q.put({"concat_equal": bool(np.array_equal(torch.cat(gathered, dim=1).numpy(), whole)),
               "band_equal": bool(np.allclose(t_part.numpy(), oracle.band_sum(cfg, whole), rtol=1e-12, atol=0)),
               "slice_equal": bool(np.array_equal(x_all[:, c0:c0 + n], x_loc)),
               "samples": float(samples.item()), "expect_samples": float(wb.n_chan * nb * L), "n_ser": int(n_ser)})
    dist.destroy_process_group()


def replace_chans(w, n_chan):
    from dataclasses import replace
    return replace(w, n_chan=n_chan, bw_hz=n_chan * w.chan_width_hz)


def test_channel_shards_concatenate_and_band_sum_is_one_allreduce():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res["slice_equal"] and res["concat_equal"] and res["band_equal"], res
    assert res["samples"] == res["expect_samples"] and res["n_ser"] > 0


def test_channel_shard_ranges_tile_the_band_and_share_the_framing():
    sys.path.insert(0, ROOT)
    import bench
    import datagen
    for n_chan, world in ((512, 8), (64, 3), (7, 2)):
        r = [bench.channel_shard(n_chan, k, world) for k in range(world)]
        assert r[0][0] == 0 and all(r[k][0] + r[k][1] == r[k + 1][0] for k in range(world - 1))
        assert r[-1][0] + r[-1][1] == n_chan and max(n for _, n in r) - min(n for _, n in r) <= 1
    w = datagen.WORKLOADS["gmrt32"]
    s = bench.sub_band(w, 128, 64)
    assert s.chan_width_hz == w.chan_width_hz
    lo = w.f_center_hz - 0.5 * w.bw_hz
    assert s.f_center_hz - 0.5 * s.bw_hz == pytest.approx(lo + 128 * w.chan_width_hz, rel=1e-15)
