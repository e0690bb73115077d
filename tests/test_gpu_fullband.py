"""GPU parity of the full-band mode (dedisp_fullband_*) against
the fp64 oracle oracle/fullband.py on seeded GSB-like spectra.  Tolerances as for the channelised path: per output block
relative L2 <= 2e-5 and max |diff| <= 1e-3 x block RMS; the c2r step is compared at 1e-6 of the series RMS."""
import numpy as np
import pytest

from oracle import fullband as fb
from test_gpu_parity import MAX_ABS_TOL, REL_L2_TOL, dd, torch  # noqa: F401  (fixtures)

pytestmark = pytest.mark.gpu


def gsb_spectra(n_spec, n_chan, seed, sigma=20.0):
    """int8 [n_spec][C][2]: Gaussian(sigma) re/im clipped to +-127, like the voltage-beam spectra of P:L35."""
    rng = np.random.default_rng(seed)
    return np.clip(np.rint(rng.normal(0.0, sigma, size=(n_spec, n_chan, 2))), -127, 127).astype(np.int8)


def check_blocks(got, ref, per):
    assert got.shape == ref.shape and got.shape[1] % per == 0 and got.shape[1] > 0
    g = got.astype(np.float64).reshape(got.shape[0], -1, per)
    r = ref.reshape(g.shape)
    den = (r ** 2).sum(-1)
    rel = np.sqrt(((g - r) ** 2).sum(-1) / den).max()
    mx = (np.abs(g - r).max(-1) / np.sqrt(den / per)).max()
    assert rel <= REL_L2_TOL and mx <= MAX_ABS_TOL, (rel, mx)
    return rel, mx


def test_framing_is_the_oracles(dd):
    for bw, f_lo, dms, N, n_int in ((16e6, 317e6, (1.5,), 2 ** 20, 16), (32e6, 309e6, (0.5, 1.0), 2 ** 21, 64),
                                    (16e6, 602e6, (30.0,), 2 ** 22, 1024)):
        assert dd.dedisp_fullband_framing(bw, f_lo, dms, N, n_int) == fb.framing(bw, f_lo, dms, N, n_int)
    with pytest.raises(dd.DedispError):
        dd.dedisp_fullband_framing(16e6, 317e6, (30.0,), 2 ** 20, 16)        # smear longer than the transform


@pytest.mark.parametrize("n_chan", [512, 1024])
def test_gsb_inverse_matches_oracle(dd, torch, n_chan):
    s = gsb_spectra(300, n_chan, seed=1)
    s[0, :, :] = -128                                                        # extreme byte, incl. the ignored Im of bin 0
    with dd.FullbandPlan(n_chan, 16e6, 317e6, (1.0,), 2 ** 20, 16) as plan:
        got = plan.debug_series(torch.from_numpy(s).cuda()).cpu().numpy().astype(np.float64)
    ref = fb.gsb_inverse(s)
    assert got.shape == ref.shape
    g, r = got.reshape(300, -1), ref.reshape(300, -1)                        # per spectrum: fp32 against fp64
    assert (np.abs(g - r).max(1) <= 1e-6 * np.abs(r).max(1)).all()


@pytest.mark.parametrize("n_chan,bw,f_lo,dms,lg_n,n_int,n_blocks", [
    (512, 16e6, 317e6, (1.5,), 20, 16, 3),            # 1024 x 1024, odd block count: the last pair is half empty
    (512, 16e6, 317e6, (0.5, 2.0), 20, 1024, 2),      # two trial DMs, paper-like integration (15 us ~ 10^3 samples)
    (1024, 32e6, 309e6, (1.0,), 21, 64, 2),           # 1024 x 2048
])
def test_fullband_matches_oracle(dd, torch, n_chan, bw, f_lo, dms, lg_n, n_int, n_blocks):
    N = 2 ** lg_n
    D, L = fb.framing(bw, f_lo, dms, N, n_int)
    n_spec = -(-(n_blocks * L + D) // (2 * n_chan))
    s = gsb_spectra(n_spec, n_chan, seed=lg_n + n_blocks)
    ref = fb.fullband(s, bw, f_lo, dms, N, n_int)
    assert ref.shape[1] == n_blocks * (L // n_int)
    with dd.FullbandPlan(n_chan, bw, f_lo, dms, N, n_int) as plan:
        assert (plan.D, plan.L) == (D, L) and plan.n1 * plan.n2 == N
        assert plan.out_samples(n_spec) == ref.shape[1]
        got = plan.execute(torch.from_numpy(s).cuda())
        torch.cuda.synchronize()
        again = plan.execute(torch.from_numpy(s).cuda())
        torch.cuda.synchronize()
        assert torch.equal(got, again)
    check_blocks(got.cpu().numpy(), ref, L // n_int)


def test_fullband_dispersed_impulse_collapses(dd, torch):
    """North-star identity through the CUDA path: a real impulse dispersed by the ISM term (Eq. 3 as printed) with one
    whole-series FFT comes back as one sample at its own position (R20: first D outputs of a block dropped)."""
    n_chan, bw, f_lo, dm, N, n_int = 512, 16e6, 317e6, 1.5, 2 ** 20, 1
    D, L = fb.framing(bw, f_lo, (dm,), N, n_int)
    n_spec = -(-(2 * L + D) // (2 * n_chan))
    T = n_spec * 2 * n_chan
    v = np.zeros(T)
    spots = [D + L // 3, D + L, D + 2 * L - 1]
    v[spots] = 80.0
    fl = np.arange(T // 2 + 1) * (2.0 * bw / T)
    psi = 4.148808e15 * dm * fl ** 2 / ((fl + f_lo) * f_lo ** 2)
    vd = np.fft.irfft(np.fft.rfft(v) * np.exp(2j * np.pi * (psi - np.floor(psi))), n=T)
    # as GSB spectra: forward real FFT of every 2C-sample frame, bins 0 .. C-1, rounded to int8 (inside a frame the
    # dispersed impulse is nearly monochromatic, so a spectrum concentrates it: amplitude 80 stays inside +-127)
    X = np.fft.rfft(vd.reshape(n_spec, 2 * n_chan), axis=1)[:, :n_chan]
    assert np.abs(X.real).max() < 127 and np.abs(X.imag).max() < 127
    s = np.stack([np.rint(X.real), np.rint(X.imag)], axis=-1).astype(np.int8)
    with dd.FullbandPlan(n_chan, bw, f_lo, (dm,), N, n_int) as plan:
        out = plan.execute(torch.from_numpy(s).cuda()).cpu().numpy()[0]
    assert out.size == 2 * L
    peak = sum(out[p - D] for p in spots)
    assert peak / out.sum() > 0.99                                            # (the oracle gives 0.997 on this input)
    for p in spots:
        assert abs(out[p - D] / 80.0 ** 2 - 1.0) < 0.02
    ref = fb.fullband(s, bw, f_lo, (dm,), N, n_int)[0]
    assert abs(peak / sum(ref[p - D] for p in spots) - 1.0) < 1e-5


def test_fullband_argument_checks(dd):
    for args in ((500, 16e6, 317e6, (1.0,), 2 ** 20, 16), (512, 16e6, 317e6, (1.0,), 2 ** 19, 16),
                 (512, 16e6, 317e6, (1.0,), 3 * 2 ** 19, 16), (512, 16e6, 317e6, (-1.0,), 2 ** 20, 16),
                 (512, 16e6, 317e6, (1.0,), 2 ** 20, 48)):
        with pytest.raises(dd.DedispError):
            dd.FullbandPlan(*args)
