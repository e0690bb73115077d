"""GPU: channel-range shards and per-channel-group framing (NEXT-2; P:L121, P:L139-141;
DESIGN R18) through dedisp_plan_shard.  A shard with the band's framing must reproduce the matching rows of the whole
plan BIT FOR BIT (same chirp factors, same per-unit arithmetic); a group with its own framing is checked against the
oracle run on that sub-band and against the whole plan on the common time axis."""
import os
from dataclasses import replace

import numpy as np
import pytest

import datagen
import oracle
from test_gpu_parity import assert_parity, dd, make_plan, ocfg, run_gpu, torch  # noqa: F401  (fixtures)

pytestmark = pytest.mark.gpu
NT = os.cpu_count() or 1


def wide_case():
    """A band wide enough for the smear to fall by 2.6x across it: 64 channels x 500 kHz, 84-116 MHz, 3 trial DMs."""
    return replace(datagen.WORKLOADS["wideband"], name="wide64", n_chan=64, bw_hz=32e6, f_center_hz=100e6,
                   dm_trials=(0.25, 0.275, 0.3), pulse_dm=0.275, n_fft=4096, n_int=16, duration_s=0.12, seed=77)


def shard_plan(dd, w, c0, n, **kw):
    return dd.dedisp_plan_shard(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int, c0, n, **kw)


@pytest.mark.parametrize("name,n_shards", [("tiny", 2), ("tiny", 4), ("gmrt16", 2)])
def test_shards_concatenate_to_the_whole_plan_bitwise(dd, torch, name, n_shards):
    w = datagen.WORKLOADS[name].scaled(0.1 if name == "tiny" else 0.2)
    x = datagen.generate(w, n_threads=NT)
    with make_plan(dd, w) as plan:
        whole = run_gpu(torch, plan, x)
        fr = (plan.head, plan.tail, plan.L)
    per = w.n_chan // n_shards
    parts = []
    for r in range(n_shards):
        with shard_plan(dd, w, r * per, per) as sp:
            assert (sp.head, sp.tail, sp.L) == fr and sp.time_offset == 0 and sp.n_chan == per
            parts.append(run_gpu(torch, sp, np.ascontiguousarray(x[:, r * per:(r + 1) * per])))
    assert np.array_equal(np.concatenate(parts, axis=1), whole)


def test_full_input_shard_reads_its_own_columns(dd, torch):
    w = datagen.WORKLOADS["tiny"].scaled(0.08)
    x = datagen.generate(w, n_threads=NT)
    c0, n = 24, 16
    with shard_plan(dd, w, c0, n) as a, shard_plan(dd, w, c0, n, full_input=True) as b:
        ga = run_gpu(torch, a, np.ascontiguousarray(x[:, c0:c0 + n]))
        gb = run_gpu(torch, b, x)
        assert np.array_equal(ga, gb)
        with pytest.raises(dd.DedispError):
            b.stream_begin(1024)


def test_shard_band_shifts_are_the_whole_plans_rows(dd):
    w = wide_case()
    with make_plan(dd, w) as plan, shard_plan(dd, w, 16, 32) as sp:
        for d in range(plan.n_dm):
            assert np.array_equal(sp.band_shifts(d), plan.band_shifts(d)[16:48])
        assert sp.debug_chirp(1, 5).tobytes() == plan.debug_chirp(1, 21).tobytes()


def test_shard_argument_checks(dd):
    w = datagen.WORKLOADS["tiny"]
    for c0, n in ((-1, 8), (0, 0), (60, 8), (0, 65)):
        with pytest.raises(dd.DedispError):
            shard_plan(dd, w, c0, n)


def test_group_framing_against_oracle_and_common_time_axis(dd, torch):
    """NEXT-2 / R18: four groups of 16 channels, each framed for its own smear; outputs match the oracle run on the
    group's sub-band, and after the integer re-timing they match the whole-band plan."""
    w = wide_case()
    x = datagen.generate(w, n_threads=NT)
    with make_plan(dd, w) as plan:
        whole = run_gpu(torch, plan, x)
        head_w, L_w = plan.head, plan.L
    kept = []
    for g in range(4):
        c0, n = 16 * g, 16
        dv = w.bw_hz / w.n_chan
        cfg_g = oracle.OracleConfig(n, n * dv, w.f_center_hz - 0.5 * w.bw_hz + (c0 + 0.5 * n) * dv, w.dm_trials,
                                    w.n_fft, w.n_int)
        with shard_plan(dd, w, c0, n, full_input=True, own_framing=True) as gp:
            assert (gp.head, gp.tail, gp.L) == oracle.framing(cfg_g)
            assert gp.head <= head_w and gp.L >= L_w and gp.time_offset == (head_w - gp.head) // w.n_int
            got = run_gpu(torch, gp, x)
            ref = oracle.dedisp(cfg_g, np.ascontiguousarray(x[:, c0:c0 + n]), n_threads=NT)
            assert_parity(got, ref, gp.L // w.n_int)
            # common time axis: out_whole[j] ~ out_group[j + offset].  Not equal: an untapered chirp's impulse response
            # has tails beyond the nominal smear (P5: 99 % inside), and what wraps around differs with the framing
            # (0.5 % here, oracle pin P19); one output sample off would be 40 %.
            off = gp.time_offset
            m = min(whole.shape[2], got.shape[2] - off)
            a, b = whole[:, c0:c0 + n, :m].astype(np.float64), got[:, :, off:off + m].astype(np.float64)
            rel = np.sqrt(((a - b) ** 2).sum() / (a ** 2).sum())
            assert rel < 0.02, rel
            kept.append(gp.L)
    assert kept[-1] > kept[0]                       # the top group keeps more of every transform ...
    assert sum(kept) / 4 > 1.08 * L_w               # ... and on average the groups beat the one-framing plan by 10 %


def test_band_sum_over_groups_equals_band_sum_of_the_whole_plan(dd, torch):
    w = wide_case()
    x = datagen.generate(w, n_threads=NT)
    dx = torch.from_numpy(x).cuda()
    with make_plan(dd, w) as plan:
        out = plan.execute(dx)
        ref = plan.band_sum(out).cpu().numpy().astype(np.float64)
    total = None
    for g in range(4):
        with shard_plan(dd, w, 16 * g, 16, full_input=True, own_framing=True) as gp:
            s = gp.band_sum(gp.execute(dx)).cpu().numpy().astype(np.float64)
            m = s.shape[1] if total is None else min(total.shape[1], s.shape[1])
            total = s[:, :m] if total is None else total[:, :m] + s[:, :m]
    m = min(total.shape[1], ref.shape[1])
    rel = np.sqrt(((total[:, :m] - ref[:, :m]) ** 2).sum() / (ref[:, :m] ** 2).sum())
    assert m > 100 and rel < 0.02, (m, rel)  # (framing-dependent wrap-around, see above)
