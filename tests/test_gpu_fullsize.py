"""GPU parity at BASELINE.json's FULL sizes (all five configs), in the launch configuration bench.py times
(dedisp_execute on the whole device-resident workload).  The oracle cannot redo a whole config in seconds, so it
recomputes SAMPLED (channel, block) units one by one: the first and last block of the lowest, a middle and the highest
channel (the edges of the framing and of the grid) plus seeded random units; every sampled unit is compared element by
element with BASELINE.json's tolerances.  Properties that hold at any size are checked on the whole output: every value
finite and positive, and the mean level: noise floor n_int * (2 sigma^2 + 1/6) (P7) plus the pulsar's duty-cycle power."""
import os

import numpy as np
import pytest

import datagen
import oracle

pytestmark = pytest.mark.gpu

REL_L2_TOL = 2e-5     # north_star, per output block
MAX_ABS_TOL = 1e-3    # x block RMS
NT = os.cpu_count() or 1


def sampled_units(n_chan, nb, n_random, seed):
    rng = np.random.default_rng(seed)
    chans = [0, 0, n_chan // 2, n_chan // 2, n_chan - 1, n_chan - 1]
    blocks = [0, nb - 1, 0, nb - 1, 0, nb - 1]
    # a pair boundary and an odd tail exercise the two-blocks-per-thread kernel
    chans += [1, 1]
    blocks += [min(1, nb - 1), max(nb - 2, 0)]
    chans += list(rng.integers(0, n_chan, n_random))
    blocks += list(rng.integers(0, nb, n_random))
    return np.asarray(chans, dtype=np.int32), np.asarray(blocks, dtype=np.int64)


@pytest.mark.parametrize("name,n_random", [("tiny", 40), ("gmrt16", 56), ("gmrt32", 56), ("lowfreq", 24),
                                           ("wideband", 8)])
def test_full_size_config_sampled_parity(name, n_random):
    import torch
    import paper_1509_00186_b200 as dd
    w = datagen.WORKLOADS[name]
    x = datagen.generate(w)
    assert x.shape == (w.n_samp, w.n_chan, 2)
    cfg = oracle.OracleConfig(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int)
    with dd.dedisp_plan(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int) as plan:
        assert (plan.head, plan.tail, plan.L) == oracle.framing(cfg)
        nb = plan.n_blocks(w.n_samp)
        per = plan.L // plan.n_int
        d_in = torch.from_numpy(x).cuda()
        d_out = plan.execute(d_in)
        torch.cuda.synchronize()
        del d_in
        assert d_out.shape == (plan.n_dm, w.n_chan, nb * per)
        # whole-output properties
        assert bool(torch.isfinite(d_out).all()) and float(d_out.min()) > 0.0
        level = float(d_out.double().mean()) / (w.n_int * (2 * w.sigma ** 2 + 1.0 / 6.0))
        # noise floor + the injected pulsar's mean power (duty cycle x amplitude^2; the chirp filter is unitary)
        expect = 1.0 + (w.pulse_width_s / w.pulse_period_s) * w.pulse_amp_sigma ** 2
        assert abs(level / expect - 1.0) < 0.03, (level, expect)
        # sampled units against the oracle
        chans, blocks = sampled_units(w.n_chan, nb, n_random, seed=w.seed + 100)
        ref = oracle.dedisp_units(cfg, x, chans, blocks, n_threads=NT)          # [n_units][n_dm][per]
        idx = torch.from_numpy(blocks[:, None] * per + np.arange(per)[None, :]).cuda()       # [n_units][per]
        got = d_out[:, torch.from_numpy(chans.astype(np.int64)).cuda()[:, None], idx]        # [n_dm][n_units][per]
        got = got.permute(1, 0, 2).double().cpu().numpy()
    den = (ref ** 2).sum(-1)
    rel = np.sqrt(((got - ref) ** 2).sum(-1) / den)
    mx = np.abs(got - ref).max(-1) / np.sqrt(den / per)
    assert rel.max() <= REL_L2_TOL, (name, float(rel.max()))
    assert mx.max() <= MAX_ABS_TOL, (name, float(mx.max()))
    print(f"{name}: {len(chans)} units x {plan.n_dm} DMs, worst rel-L2 {rel.max():.2e}, worst max/rms {mx.max():.2e}, "
          f"level {level:.4f}")
