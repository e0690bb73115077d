"""CPU pins of the full-band oracle (oracle/fullband.py):
the paper's own mode -- c2r inverse of the GSB spectra, one long real FFT over the whole band, lower-edge Eq. 3 chirp,
overlap-save, square, integrate.  Every pin is something other than the oracle's own formula retyped."""
import os

import numpy as np
import pytest

import oracle
from oracle import fullband as fb

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")) as _f:
    for _ln in _f:
        _ln = _ln.split("#")[0]
        if "=" in _ln:
            _k, _v = _ln.split("=")
            GOLD[_k.strip()] = float(_v)


# ---------------------------------------------------------------------------------------------------- step 1
def test_f1_gsb_inverse_is_the_written_out_real_inverse_dft():
    """x[n] = (1/2C) [Re X_0 + 2 sum_{k=1}^{C-1} Re(X_k e^{+2 pi i k n / 2C})]: the definition of the inverse of a 2C-point
    real FFT with the Nyquist bin absent (R19), written as a cosine/sine sum."""
    rng = np.random.default_rng(1)
    C, n_spec = 8, 3
    s = rng.integers(-128, 128, size=(n_spec, C, 2)).astype(np.int8)
    got = fb.gsb_inverse(s).reshape(n_spec, 2 * C)
    n = np.arange(2 * C)
    for j in range(n_spec):
        ref = np.full(2 * C, float(s[j, 0, 0]))
        for k in range(1, C):
            ref += 2.0 * (s[j, k, 0] * np.cos(2 * np.pi * k * n / (2 * C)) - s[j, k, 1] * np.sin(2 * np.pi * k * n / (2 * C)))
        assert np.allclose(got[j], ref / (2 * C), rtol=0, atol=1e-12)


def test_f1_gsb_inverse_undoes_a_forward_real_fft():
    """A real series whose 2C-point spectrum happens to be int8-exact comes back sample for sample."""
    C = 16
    n = np.arange(2 * C)
    v = 3.0 + 2.0 * np.cos(2 * np.pi * 5 * n / (2 * C)) - 1.5 * np.sin(2 * np.pi * 11 * n / (2 * C))
    X = np.fft.rfft(v)                                    # X_0 = 96, X_5 = 32, X_11 = 24i: all integers
    s = np.zeros((1, C, 2), np.int8)
    s[0, :, 0], s[0, :, 1] = np.rint(X[:C].real), np.rint(X[:C].imag)
    assert np.abs(X[:C] - (s[0, :, 0] + 1j * s[0, :, 1])).max() < 1e-9 and abs(X[C]) < 1e-9
    assert np.allclose(fb.gsb_inverse(s), v, atol=1e-12)


# ---------------------------------------------------------------------------------------------------- length rule
@pytest.mark.parametrize("fc_mhz,bw_mhz,key", [(610, 16, "MAXDM_610_16"), (610, 32, "MAXDM_610_32"),
                                               (325, 16, "MAXDM_325_16"), (325, 32, "MAXDM_325_32")])
def test_f2_paper_max_dm_figures_need_two_to_the_27(fc_mhz, bw_mhz, key):
    """P:L313 through this module's own smear and N rule (and the C oracle's, an independent implementation)."""
    dm = GOLD[key]
    lo, hi = (fc_mhz - bw_mhz / 2) * 1e6, (fc_mhz + bw_mhz / 2) * 1e6
    assert fb.nfft_rule(fb.smear_seconds(dm, lo, hi) * 2 * bw_mhz * 1e6) == 2 ** 27
    assert fb.smear_seconds(dm, lo, hi) == pytest.approx(oracle.smear_seconds(dm, lo, hi), rel=1e-13)


def test_f2_framing_is_the_smear_in_nyquist_samples():
    D, L = fb.framing(16e6, 317e6, (1.5,), 2 ** 18, 16)
    smear = 4.148808e15 * 1.5 * (1 / 317e6 ** 2 - 1 / 333e6 ** 2) * 32e6
    assert D % 16 == 0 and 0 <= D - smear < 16 and D + L == 2 ** 18
    with pytest.raises(ValueError):
        fb.framing(16e6, 317e6, (3000.0,), 2 ** 18, 16)


# ---------------------------------------------------------------------------------------------------- steps 2-6
def _disperse_whole_series(v, bw, f_lo, dm):
    """The ISM's in-band term (Eq. 3 as printed: exp(+2 pi i psi)) applied by ONE real FFT over the whole series:
    independent of the block framing under test."""
    n = v.size
    fl = np.arange(n // 2 + 1) * (2.0 * bw / n)
    psi = 4.148808e15 * dm * fl ** 2 / ((fl + f_lo) * f_lo ** 2)
    return np.fft.irfft(np.fft.rfft(v) * np.exp(+2j * np.pi * (psi - np.floor(psi))), n=n)


def test_f3_dispersed_impulses_collapse_at_their_own_sample():
    """Delta -> disperse at DM -> dedisperse at DM -> delta (north_star identity), for impulses in mid-block, at the
    FIRST valid sample of a block and at the LAST one: a wrong chirp sign, a wrong discard end (R20) or a wrong block
    stride smears or loses them."""
    bw, f_lo, dm, N, n_int = 4e6, 148e6, 0.01, 4096, 1
    D, L = fb.framing(bw, f_lo, (dm,), N, n_int)
    assert 300 < D < N // 2
    T = 3 * L + D
    v = np.zeros(T)
    spots = [D + L // 2, D + L, D + 2 * L - 1, D + 2 * L + 11]
    v[spots] = 500.0
    vd = _disperse_whole_series(v, bw, f_lo, dm)
    out, volt = fb.dedisp_series(vd, bw, f_lo, (dm,), N, n_int, want_voltage=True)
    assert out.shape == (1, 3 * L)
    peak = sum(out[0, s - D] for s in spots)
    assert peak / out.sum() > 0.995
    for s in spots:
        assert abs(volt[0, s - D] / 500.0 - 1.0) < 0.02          # sign and amplitude of the voltage too
    # the conjugate chirp (DM of the other sign) does not collapse them
    assert D == fb.framing(bw, f_lo, (-dm,), N, n_int)[0]
    wrong = fb.dedisp_series(vd, bw, f_lo, (-dm,), N, n_int)
    assert sum(wrong[0, s - D] for s in spots) / wrong.sum() < 0.05


def test_f3_discarding_at_the_other_end_loses_the_block_edge():
    """R20 against the reading 'drop the LAST D outputs': the impulse that disperses ahead of a block's first sample
    is then rebuilt from a block that does not hold its early part."""
    bw, f_lo, dm, N = 4e6, 148e6, 0.01, 4096
    D, L = fb.framing(bw, f_lo, (dm,), N, 1)
    v = np.zeros(2 * L + D)
    v[D + L] = 500.0                                              # first valid sample of block 1
    vd = _disperse_whole_series(v, bw, f_lo, dm)
    h = fb.chirp(bw, f_lo, dm, N)
    y = np.fft.irfft(np.fft.rfft(vd[L: L + N]) * h, n=N)         # block 1
    assert y[D] ** 2 / 500.0 ** 2 > 0.98                          # R20: valid part starts at D
    y_alt = np.fft.irfft(np.fft.rfft(vd[L + D: L + D + N][:N] if vd.size >= L + D + N else
                                     np.pad(vd[L + D:], (0, N - (vd.size - L - D)))) * h, n=N)
    assert y_alt[0] ** 2 / 500.0 ** 2 < 0.6                       # block starting AT the impulse: its early part is cut


def test_f4_dm_zero_is_the_integer_boxcar_of_the_squared_series():
    rng = np.random.default_rng(4)
    v = rng.integers(-100, 100, size=5000).astype(np.float64)
    N, n_int = 1024, 8
    out = fb.dedisp_series(v, 16e6, 317e6, (0.0,), N, n_int)
    nb = (v.size) // N
    ref = (v[: nb * N] ** 2).reshape(-1, n_int).sum(1)
    assert fb.framing(16e6, 317e6, (0.0,), N, n_int) == (0, N)
    assert np.allclose(out[0], ref, rtol=1e-10)


def test_f5_white_noise_power_is_kept():
    """The chirp has unit modulus: mean(out) = n_int * var(v) (normalisation R7 through both real transforms)."""
    rng = np.random.default_rng(5)
    v = rng.normal(0.0, 20.0, size=2 ** 17)
    out = fb.dedisp_series(v, 16e6, 317e6, (0.1,), 2 ** 15, 16)
    assert abs(out.mean() / (16 * 400.0) - 1.0) < 0.02
    hann = fb.dedisp_series(v, 16e6, 317e6, (0.1,), 2 ** 15, 16, taper="hann")
    assert abs(hann.mean() / (16 * 400.0) - 0.375) < 0.02        # mean of cos^4 over the band


def test_f6_whole_path_from_gsb_spectra_matches_the_series_path():
    rng = np.random.default_rng(6)
    C, n_spec = 64, 256
    s = rng.integers(-60, 60, size=(n_spec, C, 2)).astype(np.int8)
    a = fb.fullband(s, 16e6, 317e6, (0.005, 0.008), 4096, 4)
    b = fb.dedisp_series(fb.gsb_inverse(s), 16e6, 317e6, (0.005, 0.008), 4096, 4)
    assert a.shape[0] == 2 and a.shape[1] > 0 and np.array_equal(a, b)
    assert not np.allclose(a[0], a[1])


def test_f7_single_precision_long_transforms_are_measurably_worse():
    """P:L151 / P:L219 / Fig. 8: the paper needed fp64 for its long transforms.  Measured here at N = 2^20: the fp32 path
    (two fp32 real FFTs + fp32 chirp values) against the fp64 oracle, relative L2 of the dedispersed voltages."""
    rng = np.random.default_rng(7)
    bw, f_lo, N = 16e6, 317e6, 2 ** 20
    dm = 5.0
    D, L = fb.framing(bw, f_lo, (dm,), N, 16)
    v = np.rint(rng.normal(0.0, 20.0, size=N + L))
    _, v64 = fb.dedisp_series(v, bw, f_lo, (dm,), N, 16, want_voltage=True)
    _, v32 = fb.dedisp_series(v, bw, f_lo, (dm,), N, 16, want_voltage=True, fft_dtype=np.float32)
    rel = np.sqrt(((v64 - v32) ** 2).sum() / (v64 ** 2).sum())
    print(f"fp32 long-transform path, N = 2^20: relative L2 of the voltages {rel:.2e}")
    assert 1e-8 < rel < 1e-4
