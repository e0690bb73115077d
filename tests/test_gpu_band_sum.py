"""GPU parity of the sub-band alignment + band sum against the fp64 oracle.

Inputs never come from the CUDA path: the kernel alone is fed seeded arrays that the oracle receives as float64
copies of the same float32 values; the chain test feeds the same seeded int8 voltages to both chains."""
import os

import numpy as np
import pytest

import datagen
import oracle

pytestmark = pytest.mark.gpu
NT = os.cpu_count() or 1


@pytest.fixture(scope="module")
def dd():
    import paper_1509_00186_b200 as m
    return m


@pytest.fixture(scope="module")
def torch():
    import torch as t
    assert t.cuda.is_available()
    return t


@pytest.mark.parametrize("name", ["tiny", "gmrt16", "gmrt32", "lowfreq", "wideband"])
def test_band_shifts_match_oracle(dd, name):
    w = datagen.WORKLOADS[name]
    cfg = oracle.OracleConfig(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int)
    with dd.dedisp_plan(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int) as plan:
        for d in range(plan.n_dm):
            assert np.array_equal(plan.band_shifts(d), oracle.band_shifts(cfg, d))


@pytest.mark.parametrize("n_chan,dm,n_int,n_out", [
    (64, (10.0,), 16, 3848),            # tiny's geometry
    (37, (25.0, 0.0, -25.0), 4, 5001),  # odd sizes, a ragged tail of outputs, zero and negative DM
    (512, (71.0,), 4, 20011),           # gmrt32's shifts (up to 8606 samples) on a short series
    (3, (1.0,), 1, 7),                  # fewer outputs than one thread's share
])
def test_band_sum_kernel_matches_oracle(dd, torch, n_chan, dm, n_int, n_out):
    bw = 62.5e3 * n_chan if n_chan != 64 else 16e6
    cfg = oracle.OracleConfig(n_chan, bw, 325e6, dm, 1024, n_int)
    rng = np.random.Generator(np.random.Philox(key=n_chan * 1000 + n_out))
    out = (rng.standard_normal((len(dm), n_chan, n_out), dtype=np.float32) * 40.0 + 3200.0).astype(np.float32)
    ref = oracle.band_sum(cfg, out.astype(np.float64))
    with dd.dedisp_plan(n_chan, bw, 325e6, dm, 1024, n_int) as plan:
        assert plan.band_samples(n_out) == ref.shape[1]
        if ref.shape[1] == 0:
            with pytest.raises(dd.DedispError):
                plan.band_sum(torch.from_numpy(out).cuda())
            return
        ser = torch.full((len(dm), ref.shape[1] + 5), -1.0, dtype=torch.float32, device="cuda")
        plan.band_sum(torch.from_numpy(out).cuda(), ser)
        torch.cuda.synchronize()
        got = ser.cpu().numpy()
    assert (got[:, ref.shape[1]:] == -1.0).all()                       # nothing written past the series
    # fp32 accumulation of C terms of ~3e3: |error| <= C * eps * |sum| is a hard bound; typical is sqrt(C) * eps
    assert np.abs(got[:, : ref.shape[1]] / ref - 1.0).max() < 2e-6 * max(1.0, np.sqrt(n_chan))


def test_band_sum_integer_closed_form_on_gpu(dd, torch):
    """One unit impulse per channel at its own arrival sample -> exactly C at one series sample, 0 elsewhere."""
    w = datagen.WORKLOADS["gmrt16"]
    with dd.dedisp_plan(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int) as plan:
        sh = plan.band_shifts(0)
        n_out, j0 = int(sh.max()) + 4000, 777
        out = torch.zeros((1, w.n_chan, n_out), dtype=torch.float32)
        out[0, torch.arange(w.n_chan), torch.from_numpy(j0 + sh)] = 1.0
        got = plan.band_sum(out.cuda()).cpu().numpy()[0]
    assert got[j0] == w.n_chan and got.sum() == w.n_chan


def test_chain_dedisperse_then_band_sum_matches_oracle_chain(dd, torch):
    """int8 voltages -> coherent dedispersion per channel -> alignment -> band sum, both chains from the same input."""
    w = datagen.WORKLOADS["tiny"]
    x = datagen.generate(w)
    cfg = oracle.OracleConfig(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int)
    ref = oracle.band_sum(cfg, oracle.dedisp(cfg, x, n_threads=NT))
    with dd.dedisp_plan(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int) as plan:
        got = plan.band_sum(plan.execute(torch.from_numpy(x).cuda())).cpu().numpy()
    assert got.shape == ref.shape and ref.shape[1] > 3000
    err = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    assert err < 2e-6, err
    assert np.abs(got - ref).max() < 1e-5 * ref.max()


@pytest.mark.parametrize("n,n_bins,period", [(240_394, 39, 1.6e-3 * 1.00013), (5000, 64, 5e-3), (100, 1, 0.7), (70_001, 1024, 33e-3)])
def test_fold_matches_oracle(dd, torch, n, n_bins, period):
    rng = np.random.Generator(np.random.Philox(key=n + n_bins))
    x = (rng.standard_normal(n, dtype=np.float32) * 50.0 + 1600.0).astype(np.float32)
    t0, dt = 0.00317, 64e-6
    ref_s, ref_n = oracle.fold(x.astype(np.float64), t0, dt, period, n_bins)
    s, c = dd.dedisp_fold(torch.from_numpy(x).cuda(), t0, dt, period, n_bins)
    torch.cuda.synchronize()
    assert np.array_equal(c.cpu().numpy().astype(np.int64), ref_n)              # bins decided in fp64 on both sides
    got = s.cpu().numpy().astype(np.float64)
    assert np.abs(got - ref_s).max() <= 1e-5 * max(ref_s.max(), 1.0)


def test_chain_folded_profile_shows_the_injected_pulsar(dd, torch):
    """Whole widened chain on the GPU: dedisperse -> align + band sum -> fold at the injected period, against the same
    chain in the oracle (tiny workload)."""
    w = datagen.WORKLOADS["tiny"]
    x = datagen.generate(w)
    cfg = oracle.OracleConfig(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int)
    head, tail, L = oracle.framing(cfg)
    t0, dt = (head + 0.5 * w.n_int) / w.chan_width_hz, w.n_int / w.chan_width_hz
    ser = oracle.band_sum(cfg, oracle.dedisp(cfg, x, n_threads=NT))[0]
    ref_s, ref_n = oracle.fold(ser, t0, dt, w.pulse_period_s, 39)
    with dd.dedisp_plan(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int) as plan:
        d_ser = plan.band_sum(plan.execute(torch.from_numpy(x).cuda()))
        s, c = dd.dedisp_fold(d_ser[0].contiguous(), t0, dt, w.pulse_period_s, 39)
        torch.cuda.synchronize()
    assert np.array_equal(c.cpu().numpy().astype(np.int64), ref_n)
    prof, ref = s.cpu().numpy() / ref_n, ref_s / ref_n
    assert np.abs(prof / ref - 1.0).max() < 1e-5
    assert prof.max() > 1.15 * np.median(prof)           # the pulse stands out of the noise floor
