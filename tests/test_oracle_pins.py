"""Pins of the fp64 oracle to things other than itself (CPU only).

Every test names the pin (P1..P14 of SURVEY.md section 8(c) / DESIGN.md) and the
paper passage that fixes the expected value.  The expected values come from:
the paper's printed numbers (tests/golden/paper_values.txt), closed forms,
mpmath extended precision, numpy's own FFT (a different library routine from
the oracle's radix-2), and brute force on tiny inputs.
"""
import math
import os

import mpmath
import numpy as np
import pytest

import datagen
import oracle

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].strip()
        if "=" in line:
            k, v = line.split("=")
            GOLD[k.strip()] = float(v)

D_HZ = GOLD["D_MHZ2_US"] * 1e12 * 1e-6  # MHz^2 us -> Hz^2 s


def cfg_tiny(**kw):
    base = dict(n_chan=64, bw_hz=16e6, f_center_hz=325e6, dm=(10.0,), n_fft=1024, n_int=16)
    base.update(kw)
    return oracle.OracleConfig(**base)


# ----------------------------------------------------------------------------- P1: transforms
@pytest.mark.parametrize("n", [1, 2, 4, 8, 16, 32, 64])
def test_p1_radix2_equals_bruteforce_dft(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    for sign in (-1, +1):
        a = oracle.fft(x, sign, force_radix2=True)
        b = oracle.dft_naive(x, sign)
        assert np.max(np.abs(a - b)) < 1e-12 * max(1.0, np.max(np.abs(b)))


@pytest.mark.parametrize("n", [3, 5, 12, 64])
def test_p1_naive_dft_is_the_definition(n):
    """Naive DFT against the DFT matrix written out with mpmath (definition, sign convention)."""
    rng = np.random.default_rng(100 + n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    got = oracle.dft_naive(x, -1)
    mpmath.mp.dps = 30
    for k in (0, 1, n - 1):
        acc = mpmath.mpc(0)
        for m in range(n):
            acc += mpmath.mpc(x[m]) * mpmath.e ** (-2j * mpmath.pi * k * m / n)
        assert abs(complex(acc) - got[k]) < 1e-12


@pytest.mark.parametrize("n", [128, 1024, 4096, 16384])
def test_p1_fft_vs_numpy_and_identities(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    X = oracle.fft(x, -1)
    # independent library routine (pocketfft), same sign convention exp(-2 pi i k n / N)
    assert np.max(np.abs(X - np.fft.fft(x))) < 1e-9
    # inverse(forward) = N * identity
    assert np.max(np.abs(oracle.fft(X, +1) / n - x)) < 1e-12
    # Parseval
    assert abs(np.sum(np.abs(X) ** 2) / n - np.sum(np.abs(x) ** 2)) < 1e-8 * n
    # delta -> flat spectrum of ones; delta at n0 -> exp(-2 pi i k n0 / N) (shift theorem)
    d = np.zeros(n, complex); d[0] = 1
    assert np.max(np.abs(oracle.fft(d, -1) - 1)) < 1e-13
    n0 = 7
    d = np.zeros(n, complex); d[n0] = 1
    k = np.arange(n)
    assert np.max(np.abs(oracle.fft(d, -1) - np.exp(-2j * np.pi * k * n0 / n))) < 1e-11
    # linearity / transposed operand check: FFT of a pure tone is a single bin at +k0
    k0 = 5
    tone = np.exp(2j * np.pi * k0 * np.arange(n) / n)
    T = oracle.fft(tone, -1)
    assert abs(T[k0] - n) < 1e-8 and np.max(np.abs(np.delete(T, k0))) < 1e-8


# ----------------------------------------------------------------------------- P2: chirp formula (Eq. 3)
def test_p2_chirp_phase_matches_eq1_expansion_in_extended_precision():
    """Eq. 1 -> Eq. 2 -> Eq. 3: the in-band term equals
    D*DM*[1/(f_c+f) - 1/f_c + f/f_c^2] exactly; evaluated with 50 digits."""
    mpmath.mp.dps = 50
    for (dm, fc, f) in [(10.0, 317.125e6, -125e3), (71.0, 309.03125e6, 31.25e3 * 0.37),
                        (107.5, 200.09765625e6, -97656.25), (150.0, 142.015625e6, 15625.0 * 0.99),
                        (-26.77, 610e6, 1.0e3)]:
        D, DM, FC, F = map(mpmath.mpf, (D_HZ, dm, fc, f))
        ref = D * DM * (1 / (FC + F) - 1 / FC + F / FC ** 2)
        got = oracle.chirp_phase_cycles(dm, fc, f)
        assert abs(got - float(ref)) <= 1e-13 * max(1.0, abs(float(ref)))
    assert oracle.chirp_phase_cycles(10.0, 325e6, 0.0) == 0.0
    # psi >= 0 on both sides of the centre for DM > 0
    assert oracle.chirp_phase_cycles(10.0, 325e6, -1e5) > 0 and oracle.chirp_phase_cycles(10.0, 325e6, 1e5) > 0


def test_p2_chirp_array_unit_modulus_sign_and_bin_order():
    cfg = cfg_tiny()
    H = oracle.chirp(cfg, 0, 0)
    assert abs(H[0] - 1.0) < 1e-15                       # f = 0 -> psi = 0
    assert np.max(np.abs(np.abs(H) - 1.0)) < 1e-14       # no taper -> pure phase
    dv = oracle.chan_width(cfg)
    assert dv == 250e3
    # bin order (R5): k < N/2 positive, N/2 -> -dv/2
    assert oracle.bin_freq(cfg, 1) == dv / 1024 and oracle.bin_freq(cfg, 512) == -dv / 2
    assert oracle.bin_freq(cfg, 1023) == -dv / 1024
    # channel centres (R3): tile the band
    assert oracle.chan_freq(cfg, 0) == 317e6 + 125e3 and oracle.chan_freq(cfg, 63) == 333e6 - 125e3
    # sign (R1): the applied chirp is the INVERSE of Eq. 3, i.e. angle(H[k]) = -2 pi psi for small psi
    k = 3
    psi = float(mpmath.mpf(D_HZ) * 10 * mpmath.mpf(oracle.bin_freq(cfg, k)) ** 2
                / ((oracle.chan_freq(cfg, 0) + oracle.bin_freq(cfg, k)) * oracle.chan_freq(cfg, 0) ** 2))
    assert 0 < psi < 0.25
    assert abs(np.angle(H[k]) + 2 * np.pi * psi) < 1e-12
    # independent full-array evaluation with mpmath at a few bins, including large phases
    mpmath.mp.dps = 40
    fc = mpmath.mpf(oracle.chan_freq(cfg, 0))
    for k in (100, 511, 512, 700, 1023):
        f = mpmath.mpf(oracle.bin_freq(cfg, k))
        ph = 2 * mpmath.pi * mpmath.mpf(D_HZ) * 10 * f ** 2 / ((fc + f) * fc ** 2)
        ref = complex(mpmath.cos(ph), -mpmath.sin(ph))
        assert abs(H[k] - ref) < 1e-11


def test_p2_tapers():
    dv = 62.5e3
    assert oracle.taper("none", 1234.0, dv) == 1.0
    assert abs(oracle.taper("hann", 0.0, dv) - 1.0) < 1e-15 and abs(oracle.taper("hann", dv / 4, dv) - 0.5) < 1e-15
    assert abs(oracle.taper("hann", -dv / 2, dv)) < 1e-30
    assert oracle.taper("welch", 0.0, dv) == 1.0 and abs(oracle.taper("welch", dv / 4, dv) - 0.75) < 1e-15
    assert oracle.taper("welch", -dv / 2, dv) == 0.0
    # mean(w^2) over the band: 3/8 (Hann), 8/15 (Welch)
    f = (np.arange(4096) - 2048) / 4096 * dv
    assert abs(np.mean([oracle.taper("hann", x, dv) ** 2 for x in f]) - 0.375) < 1e-3
    assert abs(np.mean([oracle.taper("welch", x, dv) ** 2 for x in f]) - 8 / 15) < 1e-3


# ----------------------------------------------------------------------------- P3: delay law and constant D
def test_p3_group_delay_is_the_cold_plasma_delay():
    """-dpsi/df must be D*DM*(1/(f_c+f)^2 - 1/f_c^2): the textbook dispersion delay
    4.148808 ms * DM * (f/GHz)^-2 relative to the channel centre."""
    dm, fc = 57.0, 320.0e6
    for f in (-30e3, -1e3, 2e3, 31e3):
        h = 1.0
        dpsi = (oracle.chirp_phase_cycles(dm, fc, f + h) - oracle.chirp_phase_cycles(dm, fc, f - h)) / (2 * h)
        t_ms = lambda fr: 4.148808 * dm * (fr / 1e9) ** -2      # ms
        ref = (t_ms(fc + f) - t_ms(fc)) * 1e-3                   # s, arrival(f_c+f) - arrival(f_c)
        assert abs(-dpsi - ref) < 1e-6 * abs(ref)
    # in-band smear
    lo, hi = 317e6, 317.25e6
    assert abs(oracle.smear_seconds(10.0, lo, hi) - 4.148808e-3 * 10 * ((lo / 1e9) ** -2 - (hi / 1e9) ** -2)) < 1e-15


def test_p3_ism_term_delays_low_edge_and_the_applied_chirp_undoes_it():
    """Sign bookkeeping of R1/R9.  Eq. 3 = exp(+2 pi i psi) is the ISM term: with H = exp(-i phi) its group
    delay is (1/2 pi) dphi/df = -dpsi/df, > 0 (late) below the channel centre and < 0 (early) above it for DM > 0,
    the low side the longer one (1/f^2 law).  The chirp the oracle applies has the opposite phase slope
    (the inverse of the third term), bin by bin."""
    dm, fc, h = 10.0, 317.125e6, 1.0
    tau = lambda f: -(oracle.chirp_phase_cycles(dm, fc, f + h) - oracle.chirp_phase_cycles(dm, fc, f - h)) / (2 * h)
    assert tau(-100e3) > 0 and tau(+100e3) < 0
    assert tau(-100e3) > -tau(+100e3)
    cfg = cfg_tiny()
    H = oracle.chirp(cfg, 0, 0)
    fc0 = oracle.chan_freq(cfg, 0)
    for k in (1, 2, 1022, 1023):                     # small phases: no unwrapping needed
        psi = oracle.chirp_phase_cycles(10.0, fc0, oracle.bin_freq(cfg, k))
        assert 0 < psi < 0.1 and abs(np.angle(H[k]) + 2 * np.pi * psi) < 1e-12


# ----------------------------------------------------------------------------- P4: numbers the paper prints
@pytest.mark.parametrize("fc_mhz,bw_mhz,key", [(610, 16, "MAXDM_610_16"), (610, 32, "MAXDM_610_32"),
                                               (325, 16, "MAXDM_325_16"), (325, 32, "MAXDM_325_32")])
def test_p4_max_dm_figures_map_to_one_transform_length(fc_mhz, bw_mhz, key):
    """the four largest DMs that fit the 6 GB card.  With the smear function and the
    N rule of P:L139-141 (real Nyquist sampling, 2*BW samples/s) all four must give N = 2^27,
    and a DM 20 % larger must need 2^28 (so they really are the maxima)."""
    dm = GOLD[key]
    lo, hi = (fc_mhz - bw_mhz / 2) * 1e6, (fc_mhz + bw_mhz / 2) * 1e6
    fs = 2 * bw_mhz * 1e6
    assert oracle.nfft_rule(oracle.smear_seconds(dm, lo, hi) * fs) == 2 ** 27
    assert oracle.nfft_rule(oracle.smear_seconds(1.2 * dm, lo, hi) * fs) == 2 ** 28


def test_p4_nfft_rule_boundaries():
    assert oracle.nfft_rule(100.0) == 256          # smallest power of 2 GREATER than 200
    assert oracle.nfft_rule(128.0) == 512          # 2*128 = 256 is not greater than 256
    assert oracle.nfft_rule(0.3) == 1


def test_p4_data_rates_and_time_resolution():
    """120 / 240 / 1500 GB/h at 16 / 32 / 200 MHz pins 2 bytes per complex channel sample at a
    total rate of BW complex samples/s; P:L35 / P:L99: 256 channels over 16 MHz -> 62.5 kHz -> 16 us."""
    for bw, key in ((16e6, "RATE_16MHZ_GB_H"), (32e6, "RATE_32MHZ_GB_H"), (200e6, "RATE_200MHZ_GB_H")):
        gb_h = bw * 2 * 3600 / 1e9
        assert abs(gb_h - GOLD[key]) / GOLD[key] < 0.05
    c16 = oracle.OracleConfig(256, 16e6, 325e6, (1.0,), 2048, 8)
    assert oracle.chan_width(c16) == GOLD["CHANW_16MHZ_KHZ"] * 1e3
    assert abs(1e6 / oracle.chan_width(c16) - GOLD["TRES_256CH_US"]) < 1e-9
    c32 = oracle.OracleConfig(256, 32e6, 325e6, (1.0,), 2048, 8)
    assert oracle.chan_width(c32) == GOLD["CHANW_32MHZ_KHZ"] * 1e3
    c512 = oracle.OracleConfig(512, 16e6, 325e6, (1.0,), 2048, 8)
    assert abs(1e6 / oracle.chan_width(c512) - GOLD["TRES_512CH_US"]) < 1e-9


# ----------------------------------------------------------------------------- P5: impulse response support
def test_p5_impulse_response_support_and_scaling():
    """'The length of the response is equal to the dispersion time in the observing band';
    P:L45: length ~ f^-3, ~ DM, ~ BW^2."""
    cfg = cfg_tiny()
    head, tail, L = oracle.framing(cfg)
    H = oracle.chirp(cfg, 0, 0)
    h = np.fft.ifft(H)                       # lag m at index m (m >= 0) or N+m (m < 0)
    e = np.abs(h) ** 2
    inside = e[: head + 1].sum() + e[len(e) - tail:].sum()
    assert inside / e.sum() > 0.99
    # energy really is spread over ~ the smear (not concentrated): 10 % of the support holds < 50 %
    assert e[:8].sum() + e[-8:].sum() < 0.5 * e.sum()

    def smear(fc, dm, dv):
        return oracle.smear_seconds(dm, fc - dv / 2, fc + dv / 2) * dv
    s0 = smear(317.125e6, 10.0, 250e3)
    assert abs(s0 - 162.6) < 0.2                                             # 162.6 samples
    assert abs(smear(317.125e6, 20.0, 250e3) / s0 - 2.0) < 1e-9              # ~ DM^1
    assert abs(smear(317.125e6, 10.0, 500e3) / s0 - 4.0) < 0.01              # ~ BW^2
    assert abs(smear(2 * 317.125e6, 10.0, 250e3) / s0 - 2.0 ** GOLD["SCALE_FREQ_EXP"]) < 0.001   # ~ f^-3


@pytest.mark.parametrize("name,expect", [("tiny", (96, 96, 832, 74)), ("gmrt16", (32, 32, 1984, 251)),
                                         ("gmrt32", (40, 56, 4000, 249)), ("lowfreq", (224, 224, 15936, 31)),
                                         ("wideband", (2176, 2176, 12032, 129))])
def test_p5_framing_of_the_five_workloads(name, expect):
    """R9 framing; BASELINE configs[0]: 'overlap = per-channel smear samples rounded up to a multiple
    of 32' -> 192 / 64 / 96 / 448 for configs 1-4."""
    w = datagen.WORKLOADS[name]
    cfg = oracle.OracleConfig(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int)
    head, tail, L = oracle.framing(cfg)
    assert (head, tail, L, oracle.n_blocks(cfg, w.n_samp)) == expect
    assert head % w.n_int == 0 and L % w.n_int == 0 and head + tail + L == w.n_fft
    dv = w.chan_width_hz
    lo = w.f_center_hz - w.bw_hz / 2
    smear = oracle.smear_seconds(max(w.dm_trials), lo, lo + dv) * dv
    if name != "wideband":
        assert head + tail == 32 * math.ceil(smear / 32) or head + tail == 32 * math.ceil((smear + 2) / 32)
    assert head + tail >= smear


def test_p5_framing_negative_dm_swaps_head_and_tail():
    a = oracle.framing(cfg_tiny(dm=(10.0,), n_int=1))
    b = oracle.framing(cfg_tiny(dm=(-10.0,), n_int=1))
    assert a[0] + a[1] == b[0] + b[1]
    assert a[0] > a[1] - 32 and b[0] <= a[1] and b[1] >= a[0]
    # a case where the two sides differ clearly (2 MHz channel at 60 MHz): DM > 0 puts the SHORTER, high-edge side
    # (375 samples) in head and the longer low-edge side (394) in tail; DM < 0 the other way round.  By hand:
    # D*0.005*2e6*(1/60e6^2 - 1/61e6^2) = 374.7, D*0.005*2e6*(1/59e6^2 - 1/60e6^2) = 393.8
    p = oracle.framing(oracle.OracleConfig(1, 2e6, 60e6, (0.005,), 2048, 1))
    n = oracle.framing(oracle.OracleConfig(1, 2e6, 60e6, (-0.005,), 2048, 1))
    assert p[0] == 375 and n[0] == 394 and p[0] + p[1] == n[0] + n[1] == 800 and p[1] >= 394 and n[1] >= 375
    with pytest.raises(ValueError):
        oracle.framing(cfg_tiny(dm=(100.0,)))       # smear 1626 samples > N = 1024


# ----------------------------------------------------------------------------- helpers for P6-P13
def _to_int8(z):
    """complex array [T][C] -> int8 [T][C][2]; asserts exact representability is NOT required."""
    v = np.stack([np.rint(z.real), np.rint(z.imag)], axis=-1)
    assert np.max(np.abs(v)) <= 127
    return v.astype(np.int8)


def _whole_series_filter(x, dm, fc, dv, sign):
    """ONE long transform over the whole series (numpy FFT): multiply by exp(sign * 2 pi i psi);
    sign = +1 is Eq. 3 as printed, the ISM's dispersing term."""
    n = x.size
    f = np.fft.fftfreq(n, d=1.0 / dv)
    psi = D_HZ * dm * f * f / ((fc + f) * fc * fc)
    return np.fft.ifft(np.fft.fft(x) * np.exp(sign * 2j * np.pi * psi))


# ----------------------------------------------------------------------------- P6: chirp o inverse chirp
def test_p6_chirp_times_inverse_chirp_is_identity():
    """north_star identity: applying chirp then inverse chirp returns the input.  H(DM) * H(-DM) = 1."""
    cp = cfg_tiny(dm=(10.0, -10.0), n_int=1)
    H1, H2 = oracle.chirp(cp, 0, 5), oracle.chirp(cp, 1, 5)
    assert np.max(np.abs(H1 * H2 - 1.0)) < 1e-12
    assert np.max(np.abs(H2 - np.conj(H1))) < 1e-12
    rng = np.random.default_rng(6)
    x = rng.standard_normal(1024) + 1j * rng.standard_normal(1024)
    y = oracle.fft(oracle.fft(x, -1) * H1, +1) / 1024
    z = oracle.fft(oracle.fft(y, -1) * H2, +1) / 1024
    assert np.max(np.abs(z - x)) < 1e-12


# ----------------------------------------------------------------------------- P7: normalisation / noise power
def test_p7_white_noise_power_is_preserved():
    """north_star identity: output intensity for white noise matches the input power.
    int8 Gaussian sigma=20 per component, rounded: E|x|^2 = 2*(sigma^2 + 1/12) = 800.17;
    unitary filter + 1/N inverse (R7) -> mean(out) = n_int * 800.17."""
    cfg = cfg_tiny(n_chan=8, bw_hz=2e6, f_center_hz=318e6)
    x = datagen.noise_only(40000, 8, seed=7)
    out = oracle.dedisp(cfg, x, n_threads=4)
    expect = cfg.n_int * 2 * (20.0 ** 2 + 1 / 12)
    n_indep = out.size * cfg.n_int
    assert abs(out.mean() / expect - 1.0) < 5.0 / math.sqrt(n_indep)
    # and it matches the integer input power over the same rows to sampling error
    assert abs(out.mean() / (cfg.n_int * np.mean(np.sum(x.astype(np.float64) ** 2, axis=-1))) - 1.0) < 1e-2


# ----------------------------------------------------------------------------- P8: DM = 0 closed form
@pytest.mark.parametrize("n_fft,n_int,C,T", [(64, 4, 3, 1000), (128, 8, 2, 1111), (1024, 16, 4, 5000)])
def test_p8_dm_zero_is_integer_boxcar_power(n_fft, n_int, C, T):
    """DM = 0 -> H = 1 -> the whole path is the identity, so out[j] must equal the INTEGER
    sum of re^2 + im^2 over rows head + j*n_int .. (a textbook boxcar), across every block boundary.
    Pins unpack, [t][chan][2] layout, framing, block stitching, 1/N, detection, integration."""
    cfg = oracle.OracleConfig(C, 1e6, 300e6, (0.0,), n_fft, n_int)
    head, tail, L = oracle.framing(cfg)
    assert (head, tail, L) == (0, 0, n_fft)
    x = datagen.uniform_int8(T, C, seed=8)          # includes -128
    out = oracle.dedisp(cfg, x)
    nb = T // n_fft
    assert out.shape == (1, C, nb * n_fft // n_int) and nb >= 2
    p = np.sum(x.astype(np.int64) ** 2, axis=-1)    # [T][C]
    ref = p[: nb * n_fft].reshape(-1, n_int, C).sum(axis=1).T
    assert np.max(np.abs(out[0] - ref)) < 1e-7 * ref.max()


def test_p8_nonzero_head_boxcar_with_dm_pair():
    """Same closed form with head, tail > 0: a plan whose two trial DMs are (+dm, 0): the DM = 0 row
    must be the boxcar of rows head + j*n_int (R12) even though the framing comes from the other DM."""
    cfg = cfg_tiny(n_chan=2, bw_hz=0.5e6, f_center_hz=317.25e6, dm=(10.0, 0.0))
    head, tail, L = oracle.framing(cfg)
    assert head > 0 and tail > 0
    x = datagen.uniform_int8(5000, 2, seed=9)
    out = oracle.dedisp(cfg, x)
    nb = (5000 - head - tail) // L
    p = np.sum(x.astype(np.int64) ** 2, axis=-1)
    ref = p[head: head + nb * L].reshape(-1, cfg.n_int, 2).sum(axis=1).T
    assert out.shape[2] == nb * L // cfg.n_int
    assert np.max(np.abs(out[1] - ref)) < 1e-7 * ref.max()
    assert np.max(np.abs(out[0] - ref)) > 1e-3 * ref.max()      # the DM = 10 row is NOT the boxcar


# ----------------------------------------------------------------------------- P9: delta collapses, discard placement
@pytest.mark.parametrize("dm", [10.0, -10.0])
def test_p9_dispersed_delta_collapses_to_a_delta(dm):
    """north_star identity: a delta pulse dispersed at DM collapses back to a delta when dedispersed at
    the same DM.  The delta is dispersed with Eq. 3 as printed through ONE whole-series numpy FFT (independent of
    the block framing), quantised to int8, then run through the block algorithm with n_int = 1.
    Deltas sit mid-block, at the last valid sample of block 0 and at the first valid sample of block 1:
    a wrong head/tail split or a wrong chirp sign smears or loses them."""
    cfg = cfg_tiny(n_chan=1, bw_hz=250e3, f_center_hz=317.125e6, dm=(dm,), n_int=1)
    head, tail, L = oracle.framing(cfg)
    T = 3 * L + head + tail
    fc, dv = oracle.chan_freq(cfg, 0), oracle.chan_width(cfg)
    A = 700.0
    spots = [head + L // 2, head + L - 1, head + L, head + 2 * L + 7]
    x = np.zeros(T, complex)
    for s in spots:
        x[s] = A
    xd = _whole_series_filter(x, dm, fc, dv, sign=+1)           # disperse = Eq. 3 = conj of the applied chirp
    assert np.max(np.abs(xd)) < 127
    out = oracle.dedisp(cfg, _to_int8(xd[:, None]))[0, 0]
    assert out.size == 3 * L
    tot = out.sum()
    peak = sum(out[s - head] for s in spots)
    assert peak / tot > 0.999
    for s in spots:
        assert abs(out[s - head] / A ** 2 - 1.0) < 0.02
    # negative control: the opposite chirp sign does NOT collapse it
    cfg_wrong = cfg_tiny(n_chan=1, bw_hz=250e3, f_center_hz=317.125e6, dm=(-dm,), n_int=1)
    h2, t2, L2 = oracle.framing(cfg_wrong)
    out_w = oracle.dedisp(cfg_wrong, _to_int8(xd[:, None]))[0, 0]
    assert out_w.max() < 0.05 * A ** 2


def test_p9_misplaced_discard_fails_visibly():
    """If the valid window were taken at the wrong place (all the discard at one end) the collapsed
    delta next to a block edge would lose energy: check with the voltage output of a unit."""
    cfg = cfg_tiny(n_chan=1, bw_hz=250e3, f_center_hz=317.125e6, dm=(10.0,), n_int=1)
    head, tail, L = oracle.framing(cfg)
    fc, dv = oracle.chan_freq(cfg, 0), oracle.chan_width(cfg)
    T = 2 * L + head + tail
    x = np.zeros(T, complex)
    x[head] = 700.0                                           # first valid sample of block 0
    xd = _whole_series_filter(x, 10.0, fc, dv, sign=+1)
    xi = _to_int8(xd[:, None])
    out, volt = oracle.dedisp_units(cfg, xi, [0], [0], want_voltage=True)
    assert abs(volt[0, 0, 0]) ** 2 / 700.0 ** 2 > 0.98
    # emulate "discard everything at the beginning" (textbook wording P:L125): the block would then
    # start head+tail rows later and the sample `head` of the series would fall in the discarded part;
    # emulate "discard everything at the end": sample index 0 of a block needs `head` past samples that
    # the block does not contain -> the same delta placed at block-local index 0 does not collapse.
    x2 = np.zeros(T, complex); x2[0] = 700.0
    xd2 = _whole_series_filter(x2, 10.0, fc, dv, sign=+1)
    blk = np.fft.ifft(np.fft.fft(np.rint(xd2[:1024].real) + 1j * np.rint(xd2[:1024].imag)) * oracle.chirp(cfg, 0, 0))
    assert abs(blk[0]) ** 2 / 700.0 ** 2 < 0.9                # polluted by the circular wrap


# ----------------------------------------------------------------------------- P11: multi-DM rows
def test_p11_multi_dm_rows_equal_single_dm_plans_when_framing_is_shared():
    dms = (8.0, 9.0, 10.0)
    kw = dict(n_chan=3, bw_hz=0.75e6, f_center_hz=317.375e6)
    x = datagen.noise_only(6000, 3, seed=11)
    multi = oracle.dedisp(cfg_tiny(dm=dms, **kw), x)
    # the largest DM fixes the framing; add it as a second trial so single-DM plans share it
    for i, dm in enumerate(dms):
        single = oracle.dedisp(cfg_tiny(dm=(dm, dms[-1]), **kw), x)
        assert np.array_equal(single[0], multi[i])


# ----------------------------------------------------------------------------- P12: brute force on tiny inputs
@pytest.mark.parametrize("n_fft", [64, 128])
def test_p12_bruteforce_time_domain_circular_convolution(n_fft):
    """Tiny case: per block, y[n] = sum_m h[m] x[(n-m) mod N] with h = IDFT(H) written out as loops;
    H from the formula in mpmath; keep [head, N-tail); |.|^2; sums of n_int = 2."""
    C, n_int, T = 2, 2, 5 * n_fft + 3
    cfg = oracle.OracleConfig(C, 0.2e6, 100e6, (0.02,), n_fft, n_int)
    head, tail, L = oracle.framing(cfg)
    assert head > 0 and tail > 0 and L > 0
    x = datagen.uniform_int8(T, C, seed=12)
    out = oracle.dedisp(cfg, x)
    nb = (T - head - tail) // L
    mpmath.mp.dps = 30
    dv = 0.1e6
    for c in range(C):
        fc = 100e6 - 0.1e6 + (c + 0.5) * dv
        H = np.zeros(n_fft, complex)
        for k in range(n_fft):
            f = (k if k < n_fft // 2 else k - n_fft) * dv / n_fft
            ph = 2 * mpmath.pi * mpmath.mpf(D_HZ) * mpmath.mpf("0.02") * mpmath.mpf(f) ** 2 / (
                (mpmath.mpf(fc) + f) * mpmath.mpf(fc) ** 2)
            H[k] = complex(mpmath.cos(ph), -mpmath.sin(ph))     # inverse of Eq. 3 (R1)
        h = np.array([sum(H[k] * np.exp(2j * np.pi * k * m / n_fft) for k in range(n_fft)) / n_fft
                      for m in range(n_fft)])
        ref = []
        for b in range(nb):
            xb = x[b * L: b * L + n_fft, c, 0].astype(float) + 1j * x[b * L: b * L + n_fft, c, 1].astype(float)
            y = np.array([sum(h[m] * xb[(n - m) % n_fft] for m in range(n_fft)) for n in range(n_fft)])
            p = np.abs(y[head: head + L]) ** 2
            ref.append(p.reshape(-1, n_int).sum(axis=1))
        ref = np.concatenate(ref)
        assert out.shape[2] == ref.size
        assert np.max(np.abs(out[0, c] - ref)) < 1e-9 * ref.max()


# ----------------------------------------------------------------------------- P13: tones and tapers
@pytest.mark.parametrize("taper,k_frac,w", [("none", 0.25, 1.0), ("hann", 0.25, 0.5), ("welch", 0.25, 0.75),
                                            ("hann", 0.5, 0.0), ("welch", 0.5, 0.0), ("hann", 0.0, 1.0),
                                            ("welch", 0.75, 0.75)])
def test_p13_exact_int8_tones(taper, k_frac, w):
    """x[n] = A e^{2 pi i k0 n / N}, k0 in {0, N/4, N/2, 3N/4} is exactly representable in int8; a tone
    sits in one FFT bin so out = n_int * A^2 * w(f_k0)^2 for ANY DM (|H| = w)."""
    cfg = cfg_tiny(n_chan=2, bw_hz=0.5e6, f_center_hz=317.25e6, taper=taper)
    head, tail, L = oracle.framing(cfg)
    T, A = 4000, 100
    n = np.arange(T)
    z = A * np.exp(2j * np.pi * k_frac * n)
    x = _to_int8(np.stack([z, z], axis=1))
    out = oracle.dedisp(cfg, x)
    expect = cfg.n_int * A * A * w * w
    assert np.max(np.abs(out - expect)) < 1e-6 * (A * A * cfg.n_int)


# ----------------------------------------------------------------------------- P14: science sanity on the tiny workload
def test_p14_injected_pulsar_is_sharpest_at_its_dm():
    """Statistical, not parity: fold the tiny workload's outputs at the injected period; the profile peak
    is highest at the injected DM (10), lower at 5, lowest at 0; off-pulse level = n_int * 800.17."""
    w = datagen.WORKLOADS["tiny"]
    chans = [0, 31, 63]
    x = datagen.generate(w, chans=chans)
    fcs = datagen.chan_freqs_hz(w)
    peaks = {}
    for dm in (10.0, 5.0, 0.0):
        tops = []
        for i, c in enumerate(chans):
            # single-channel plan centred on channel c with the same channel width
            cfg = oracle.OracleConfig(1, w.chan_width_hz, float(fcs[c]), (dm, 10.0), w.n_fft, w.n_int)
            head, tail, L = oracle.framing(cfg)
            out = oracle.dedisp(cfg, np.ascontiguousarray(x[:, i:i + 1, :]))[0, 0]
            t = (head + np.arange(out.size) * w.n_int + 0.5 * w.n_int) / w.chan_width_hz
            delay = datagen.D_HZ2_S * w.pulse_dm * (1 / fcs[c] ** 2 - 1 / (w.f_center_hz + w.bw_hz / 2) ** 2)
            ph = np.mod(t - delay, w.pulse_period_s) / w.pulse_period_s
            nbin = 39
            b = np.minimum((ph * nbin).astype(int), nbin - 1)
            prof = np.bincount(b, out, nbin) / np.maximum(np.bincount(b, None, nbin), 1)
            tops.append(prof.max())
            if dm == 10.0:
                assert abs(np.median(prof) / (w.n_int * 800.17) - 1.0) < 0.02
                assert prof.argmax() == 0
        peaks[dm] = np.mean(tops)
    assert peaks[10.0] > 1.3 * peaks[5.0] > 1.3 * 1.2 * peaks[0.0]


# ----------------------------------------------------------------------------- P15-P17: band alignment + sum (NEXT-3)
def test_p15_band_shifts_follow_the_printed_delay_law():
    """P:L39-41 / P:L117: the delay between two frequencies is D * DM * (f1^-2 - f2^-2) with D printed in MHz/us
    units (golden file); the oracle's shifts (computed in Hz/s) must be that delay in whole output samples."""
    for name in ("tiny", "gmrt32", "lowfreq"):
        w = datagen.WORKLOADS[name]
        cfg = oracle.OracleConfig(w.n_chan, w.bw_hz, w.f_center_hz, w.dm_trials, w.n_fft, w.n_int)
        sh = oracle.band_shifts(cfg, 0)
        f_mhz = datagen.chan_freqs_hz(w) / 1e6
        delay_us = GOLD["D_MHZ2_US"] * w.dm_trials[0] * (f_mhz ** -2 - f_mhz[-1] ** -2)        # paper's units
        expect = delay_us * 1e-6 * w.chan_width_hz / w.n_int                                 # output samples
        assert sh[-1] == 0 and sh.min() == 0
        assert np.all(np.diff(sh) <= 0)                        # lower channels arrive later
        assert np.abs(sh - expect).max() <= 0.5 + 1e-6         # nearest whole sample
        # adjacent channels differ by the dispersion smear between their centres (an independent oracle helper)
        fc = datagen.chan_freqs_hz(w)
        smear = np.array([oracle.smear_seconds(w.dm_trials[0], fc[c], fc[c + 1]) for c in range(w.n_chan - 1)])
        assert np.abs(-np.diff(sh) - smear * w.chan_width_hz / w.n_int).max() <= 1.0 + 1e-6


def test_p15_negative_dm_mirrors_the_shifts():
    cfg_p = cfg_tiny(dm=(10.0,))
    cfg_n = cfg_tiny(dm=(-10.0,))
    sp, sn = oracle.band_shifts(cfg_p, 0), oracle.band_shifts(cfg_n, 0)
    assert sn.min() == 0 and sn[0] == 0 and np.all(np.diff(sn) >= 0)
    assert np.abs((sp.max() - sp) - sn).max() <= 1


def test_p16_band_sum_integer_closed_form():
    """A unit impulse placed in every channel at its own arrival sample sums to exactly C at one sample and to 0
    elsewhere; DM = 0 reduces the band sum to the plain sum over channels."""
    cfg = cfg_tiny(dm=(10.0, 0.0, -7.0))
    n_out, j0 = 900, 123
    out = np.zeros((3, cfg.n_chan, n_out))
    for d in range(3):
        sh = oracle.band_shifts(cfg, d)
        out[d, np.arange(cfg.n_chan), j0 + sh] = 1.0
    s = oracle.band_sum(cfg, out)
    max_shift = max(int(oracle.band_shifts(cfg, d).max()) for d in range(3))
    assert s.shape == (3, n_out - max_shift)
    for d in range(3):
        assert s[d, j0] == cfg.n_chan and s[d].sum() == cfg.n_chan
    rng = np.random.default_rng(3)
    r = rng.normal(size=(3, cfg.n_chan, n_out))
    s = oracle.band_sum(cfg, r)
    assert np.allclose(s[1], r[1].sum(0)[: s.shape[1]], rtol=0, atol=1e-12)
    # brute force for the dispersed rows, written out index by index
    sh0 = oracle.band_shifts(cfg, 0)
    for j in (0, 17, s.shape[1] - 1):
        assert abs(s[0, j] - sum(r[0, c, j + sh0[c]] for c in range(cfg.n_chan))) < 1e-12


def test_p17_band_sum_raises_the_pulse_above_a_single_channel():
    """Science sanity for the whole chain (statistical): coherent dedispersion per channel + alignment + band sum of
    the tiny workload gives a folded pulse whose signal-to-noise beats a single channel's by roughly sqrt(C), and
    summing WITHOUT the alignment (DM 0 shifts) smears it away."""
    w = datagen.WORKLOADS["tiny"]
    x = datagen.generate(w)
    cfg = oracle.OracleConfig(w.n_chan, w.bw_hz, w.f_center_hz, (w.pulse_dm,), w.n_fft, w.n_int)
    head, tail, L = oracle.framing(cfg)
    out = oracle.dedisp(cfg, x, n_threads=os.cpu_count() or 1)

    def snr(series):
        t = (head + np.arange(series.size) * w.n_int + 0.5 * w.n_int) / w.chan_width_hz
        nbin = 39
        b = np.minimum((np.mod(t, w.pulse_period_s) / w.pulse_period_s * nbin).astype(int), nbin - 1)
        prof = np.bincount(b, series, nbin) / np.maximum(np.bincount(b, None, nbin), 1)
        off = np.sort(prof)[: nbin // 2]
        return (prof.max() - np.median(prof)) / off.std()

    aligned = oracle.band_sum(cfg, out)[0]
    cfg0 = oracle.OracleConfig(w.n_chan, w.bw_hz, w.f_center_hz, (0.0,), w.n_fft, w.n_int)
    unaligned = oracle.band_sum(cfg0, out)[0]
    single = out[0, w.n_chan - 1]
    assert snr(aligned) > 4.0 * snr(single)           # sqrt(64) = 8 in the ideal case
    assert snr(aligned) > 3.0 * snr(unaligned)


# ----------------------------------------------------------------------------- P18: folding (NEXT-3)
def test_p18_fold_closed_forms_and_numpy_bincount():
    """(a) a constant series folds to sum == count; (b) with dt = period/n_bins exactly, sample j falls in bin
    j mod n_bins, so a comb of period n_bins puts everything in one bin; (c) an independent implementation
    (numpy mod + bincount) gives the same bins and sums on random data with an awkward period."""
    oracle.build()
    s, n = oracle.fold(np.ones(1000), 0.0, 1.0, 64.0, 64)
    assert np.array_equal(s, n.astype(float)) and n.sum() == 1000 and n.max() - n.min() <= 1
    comb = np.zeros(64 * 20)
    comb[5::64] = 3.0
    s, n = oracle.fold(comb, 0.0, 0.25, 16.0, 64)           # 0.25 and 16 are exact in binary
    assert s[5] == 60.0 and s.sum() == 60.0 and np.all(n == 20)
    rng = np.random.default_rng(18)
    x = rng.normal(size=50_000) + 10.0
    t0, dt, P, nb = 0.00123, 64e-6, 5.0e-3 * 1.000137, 39
    s, n = oracle.fold(x, t0, dt, P, nb)
    t = t0 + np.arange(x.size) * dt
    ph = t / P - np.floor(t / P)
    b = np.minimum((ph * nb).astype(int), nb - 1)
    assert np.array_equal(n, np.bincount(b, minlength=nb))
    assert np.allclose(s, np.bincount(b, x, nb), rtol=1e-12)


# ----------------------------------------------------------------------------- frozen oracle output
def load_frozen_case():
    import importlib.util
    here = os.path.join(os.path.dirname(__file__), "golden")
    spec = importlib.util.spec_from_file_location("make_oracle_golden", os.path.join(here, "make_oracle_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    vals = np.loadtxt(os.path.join(here, "oracle_small_case.txt"))
    with open(os.path.join(here, "oracle_small_case.txt")) as fh:
        shape = [int(v) for v in [l for l in fh if l.startswith("# shape")][0].split()[2:]]
    return mod, vals.reshape(shape)


def test_oracle_output_is_frozen():
    """The oracle still produces the stored values (written by tests/golden/make_oracle_golden.py, which calls only
    oracle/ and datagen/): its arithmetic has not drifted.  1e-12 relative leaves room for libm differences only."""
    mod, frozen = load_frozen_case()
    _, _, out = mod.compute()
    assert out.shape == frozen.shape
    assert np.abs(out / frozen - 1.0).max() < 1e-12


# ----------------------------------------------------------------------------- P19: physical sign pin (independent of Eq. 3)
def _dispersed_band_impulse(C, B, F, dm, T, t0_s, A):
    """A whole-band impulse that went through the ISM, built from the DELAY LAW alone (a component at
    sky frequency f arrives D*DM/f^2 late), then split into C critically sampled channels by one FFT (an ideal
    brick-wall channeliser; channel c covers [F-B/2 + c dv, F-B/2 + (c+1) dv), R3, baseband frequency rising with sky
    frequency, R5).  The transfer function is exp(-i phi) with (1/2 pi) dphi/df = delay, delays measured
    against the top band edge: phi(f) = -2 pi D DM (1/f + f/f_top^2).  Returns complex [T][C]."""
    M = C * T
    nu = np.fft.fftfreq(M, d=1.0 / B)                       # baseband frequency of the whole band, sky = F + nu
    f_top = F + B / 2
    X = A * np.exp(-2j * np.pi * nu * t0_s)                 # impulse at t0
    X = X * np.exp(+2j * np.pi * D_HZ * dm * (1.0 / (F + nu) + nu / f_top ** 2))
    Xs = np.fft.fftshift(X)                                 # ascending sky frequency
    chans = [np.fft.ifft(np.fft.ifftshift(Xs[c * T:(c + 1) * T])) for c in range(C)]
    return np.stack(chans, axis=1)


def test_p19_physically_dispersed_band_impulse_collapses_with_one_positive_dm():
    """The pin that ties the chirp sign (R1), the framing roles (R9) and the band alignment (R16) to physics rather
    than to each other: an impulse dispersed by the delay law (no use of Eq. 3) must, with ONE plan at DM = +0.5,
    (a) collapse inside every channel, (b) sit at the arrival time of the channel centre, and (c) line up in the band
    sum.  The opposite DM sign must smear it further."""
    C, B, F, dm, T, N = 8, 1e6, 100e6, 0.5, 4096, 256
    dv = B / C
    A = 800.0
    t0 = 1500.25 / dv
    z = _dispersed_band_impulse(C, B, F, dm, T, t0, A)
    x = _to_int8(z)
    cfg = oracle.OracleConfig(C, B, F, (dm,), N, 1)
    head, tail, L = oracle.framing(cfg)
    out = oracle.dedisp(cfg, x)[0]                                        # [C][n_out], n_int = 1
    fcs = np.array([oracle.chan_freq(cfg, c) for c in range(C)])
    arrive = (t0 + D_HZ * dm * (fcs ** -2.0 - (F + B / 2) ** -2.0)) * dv - head   # output sample index
    undisp = np.abs(z) ** 2
    for c in range(C):
        pk = int(out[c].argmax())
        assert abs(pk - arrive[c]) <= 1.0, (c, pk, arrive[c])             # (b)
        frac = out[c, pk - 2: pk + 3].sum() / out[c].sum()
        # (a) collapsed: a band-limited impulse half a sample off the grid keeps 2*(sinc^2(.5)+sinc^2(1.5))+sinc^2(2.5)
        # = 0.916 of its energy in 5 samples, one on the grid keeps all of it; measured 0.921 ... 0.998
        assert frac > 0.90, (c, frac)
        assert out[c].max() > 6.0 * undisp[:, c].max()                    # ... from a smear of ~65 samples
    s = oracle.band_sum(cfg, out[None])[0]                                # (c)
    pk = int(s.argmax())
    assert s[pk - 2: pk + 3].sum() > 0.90 * s.sum()
    assert s.max() > 0.5 * C * A * A
    # negative control: the opposite sign doubles the smear instead of removing it
    cfg_n = oracle.OracleConfig(C, B, F, (-dm,), N, 1)
    out_n = oracle.dedisp(cfg_n, x)[0]
    for c in range(C):
        assert out_n[c].max() < 0.6 * undisp[:, c].max() + 50.0


# ----------------------------------------------------------------------------- P20: the sampled-unit and unpack entry points
def test_p20_dedisp_units_equals_the_rows_of_dedisp():
    """oracle.dedisp_units is the only reference of the full-size GPU tests: every (channel, block) unit of a 3-channel,
    4-block, 3-DM case must equal the matching slice of oracle.dedisp exactly (same arithmetic, different indexing),
    voltages included (their squared sums reproduce the intensities)."""
    cfg = cfg_tiny(n_chan=3, bw_hz=0.75e6, f_center_hz=317.375e6, dm=(10.0, -6.0, 3.0), n_int=8)
    head, tail, L = oracle.framing(cfg)
    x = datagen.uniform_int8(4 * L + head + tail + 5, 3, seed=20)
    full = oracle.dedisp(cfg, x)
    per = L // cfg.n_int
    assert full.shape == (3, 3, 4 * per)
    chans = [c for c in range(3) for b in range(4)]
    blocks = [b for c in range(3) for b in range(4)]
    order = np.random.default_rng(20).permutation(len(chans))           # not in storage order
    chans, blocks = np.asarray(chans)[order], np.asarray(blocks)[order]
    units, volt = oracle.dedisp_units(cfg, x, chans, blocks, n_threads=3, want_voltage=True)
    assert units.shape == (12, 3, per) and volt.shape == (12, 3, L)
    for i, (c, b) in enumerate(zip(chans, blocks)):
        for d in range(3):
            assert np.array_equal(units[i, d], full[d, c, b * per:(b + 1) * per]), (i, c, b, d)
            p = (np.abs(volt[i, d]) ** 2).reshape(per, cfg.n_int).sum(1)
            assert np.allclose(p, units[i, d], rtol=1e-12, atol=0)
    # the DM = +10 and DM = -6 rows really differ (a stride bug that repeats one DM would pass the loop above otherwise)
    assert np.abs(units[:, 0] - units[:, 1]).max() > 1.0


def test_p20_unpack_block_is_the_framed_slice_of_the_input():
    cfg = cfg_tiny(n_chan=5, bw_hz=1.25e6, f_center_hz=317.625e6, n_int=4)
    head, tail, L = oracle.framing(cfg)
    x = datagen.uniform_int8(3 * L + head + tail, 5, seed=21)
    nb = oracle.n_blocks(cfg, x.shape[0])
    assert nb == 3
    for c in (0, 2, 4):
        for b in (0, nb - 1):
            got = oracle.unpack_block(cfg, x, c, b)
            assert got.dtype == np.float64 and got.shape == (cfg.n_fft, 2)
            assert np.array_equal(got, x[b * L: b * L + cfg.n_fft, c, :].astype(np.float64))
    assert (x == -128).any()


# ----------------------------------------------------------------------------------------------------------------
# P21 (R18): per-channel-group framing.  A group of channels framed for its OWN smear (P:L121,
# the length to discard is the dispersion time in the band; it falls as f^-3) gives the same
# dedispersed series as the whole-band framing, shifted by the whole number (head_whole - head_group)/n_int of outputs
# ----------------------------------------------------------------------------------------------------------------
def test_p21_group_framing_retimes_to_the_whole_band_axis():
    n_int = 4
    whole = oracle.OracleConfig(8, 16e6, 60e6, (0.001,), 1024, n_int)       # 52 ... 68 MHz: smear falls 2.2x across it
    head_w, tail_w, L_w = oracle.framing(whole)
    x = datagen.noise_only(12 * 1024, 8, seed=31)
    ref = oracle.dedisp(whole, x)
    # an impulse in every channel at one instant: the position is fixed by the sample grid, not by a correlation
    xi = np.zeros((6 * 1024, 8, 2), dtype=np.int8)
    t_imp = 2500
    xi[t_imp, :, 0] = 100
    ref_i = oracle.dedisp(whole, xi)
    heads = []
    for g in range(2):
        c0, n = 4 * g, 4
        cfg = oracle.OracleConfig(n, n * 2e6, 60e6 - 8e6 + (c0 + 0.5 * n) * 2e6, (0.001,), 1024, n_int)
        head, tail, L = oracle.framing(cfg)
        heads.append(head)
        assert head <= head_w and tail <= tail_w and L >= L_w and (head_w - head) % n_int == 0
        off = (head_w - head) // n_int
        out = oracle.dedisp(cfg, np.ascontiguousarray(x[:, c0:c0 + n]))
        m = min(ref.shape[2], out.shape[2] - off)
        a, b = ref[:, c0:c0 + n, :m], out[:, :, off:off + m]
        rel = np.sqrt(((a - b) ** 2).sum() / (a ** 2).sum())
        rel_off = np.sqrt(((a[:, :, 1:] - b[:, :, :-1]) ** 2).sum() / (a ** 2).sum())
        assert rel < 0.02 < 0.2 < rel_off, (g, rel, rel_off)   # aligned: wrap-around differences only (see P5)
        # the dedispersed energy of the impulse peaks in the same output sample on the common axis, for every channel
        out_i = oracle.dedisp(cfg, np.ascontiguousarray(xi[:, c0:c0 + n]))
        for c in range(n):
            assert int(np.argmax(out_i[0, c])) - off == int(np.argmax(ref_i[0, c0 + c]))
    assert heads[1] < heads[0] == head_w                         # the low group sets the band's framing
