"""fp64 oracle of the paper's OWN mode: full-band coherent dedispersion (Fig. 4,
P:L173-179).  No sub-banding: the GSB spectra are inverse transformed back to the real
Nyquist-sampled voltage series, ONE long real FFT of N points covers the whole band, the chirp of Eq. 3 is
applied with the LOWER BAND EDGE as its reference, and the overlap-save method returns the dedispersed series.

TEST INFRASTRUCTURE ONLY (like the rest of oracle/): plain numpy in fp64, the paper's steps in the paper's order, the
library FFT (numpy.fft, pocketfft in fp64) serving as the FFT step.  No product code imports this module; no CUDA
kernel for this mode exists yet, so nothing here has been shaped by one.

Steps (Fig. 4):
  1. inverse transform   every GSB spectrum (C complex int8 bins of a 2C-point real FFT) -> 2C real samples
  2. long FFT            blocks of N real samples, N = the smallest power of 2 > 2 x (dispersion time in samples)
  3. chirp               N/2 bins x taper(f_l) exp(-2 pi i psi), psi = D DM f_l^2 / ((f_l + f_o) f_o^2): "the inverse of the
                         third term" that Eq. 3 prints
  4. inverse FFT         back to N real samples
  5. overlap-save        D = length of the impulse response is lost per block and "prefixed to the next block"
  6. detect + integrate  square, sum n_int samples

Readings:
  R19  which bins a GSB spectrum holds: bins 0 .. C-1 of the 2C-point real FFT (bin k at f_o + k B/C); the Nyquist bin is
       not recorded and is taken as 0; the imaginary part of bin 0 carries nothing for a real series and is ignored.
       Normalisation 1/(2C) on the inverse, so a spectrum made by an unnormalised forward FFT returns the original samples.
  R20  which end is discarded: with the lower edge as reference every other frequency of the band arrived EARLIER than
       f_o and the correction delays it (group delay of exp(-2 pi i psi) is +d psi/d f_l >= 0): an output sample needs up
       to D PAST input samples, so the first D outputs of a block are invalid ("discarded from the beginning");
       P:L270's "at the end" describes the same bookkeeping from the input side (the last D inputs of a block are
       read again as the first D of the next).  D = ceil(smear x 2B) rounded up to a multiple of n_int.
  R21  baseband order: upper sideband, bin k of the long FFT is f_l = k 2B/N above f_o ("deviation from the lower
       edge"); the bin at f_l = B (Nyquist) gets the same formula.
"""
from __future__ import annotations

import numpy as np

D_HZ2_S = 4.148808e15  # P:L117 "4.148808 x 10^9" in MHz/us units = 4.148808e15 Hz^2 s per pc cm^-3 (R8)


def smear_seconds(dm: float, f_lo_hz: float, f_hi_hz: float) -> float:
    """Dispersion time in the band = length of the impulse response: D DM (1/f_lo^2 - 1/f_hi^2)."""
    return D_HZ2_S * abs(dm) * (1.0 / f_lo_hz ** 2 - 1.0 / f_hi_hz ** 2)


def nfft_rule(smear_samples: float) -> int:
    """the smallest power of 2 greater than twice the number of samples of the dispersion time."""
    n = 1
    while n <= 2.0 * smear_samples:
        n *= 2
    return n


def framing(bw_hz: float, f_lo_hz: float, dms, n_fft: int, n_int: int):
    """(D, L): samples lost per block (R20) and valid samples per block; ValueError if the transform is too short."""
    fs = 2.0 * bw_hz
    d = max(int(np.ceil(smear_seconds(dm, f_lo_hz, f_lo_hz + bw_hz) * fs)) for dm in dms)
    d = -(-d // n_int) * n_int
    if d >= n_fft or (n_fft - d) % n_int:
        raise ValueError(f"transform of {n_fft} too short for an overlap of {d}")
    return d, n_fft - d


def gsb_inverse(spec_int8: np.ndarray) -> np.ndarray:
    """Step 1: int8 [n_spec][C][2] (re, im) -> float64 [n_spec * 2C] real voltage series (R19)."""
    s = np.asarray(spec_int8)
    assert s.dtype == np.int8 and s.ndim == 3 and s.shape[2] == 2
    n_spec, C = s.shape[0], s.shape[1]
    half = np.zeros((n_spec, C + 1), dtype=np.complex128)
    half[:, :C] = s[:, :, 0].astype(np.float64) + 1j * s[:, :, 1].astype(np.float64)
    half[:, 0] = half[:, 0].real            # bin 0 of a real series is real
    return np.fft.irfft(half, n=2 * C, axis=1).reshape(-1)  # irfft carries the 1/(2C)


def chirp(bw_hz: float, f_lo_hz: float, dm: float, n_fft: int, taper: str = "none") -> np.ndarray:
    """Step 3: the chirp function on the N/2 + 1 bins of the long real FFT (Eq. 3 P:L114 inverted)."""
    k = np.arange(n_fft // 2 + 1, dtype=np.float64)
    fl = k * (2.0 * bw_hz / n_fft)                                   # R21
    psi = D_HZ2_S * dm * fl * fl / ((fl + f_lo_hz) * f_lo_hz ** 2)   # cycles
    psi -= np.floor(psi)
    h = np.exp(-2j * np.pi * psi)
    if taper == "hann":        # same windows as the channelised path (R6), centred on the band
        h = h * np.cos(np.pi * (fl - 0.5 * bw_hz) / bw_hz) ** 2
    elif taper == "welch":
        h = h * (1.0 - (2.0 * (fl - 0.5 * bw_hz) / bw_hz) ** 2)
    elif taper != "none":
        raise ValueError(taper)
    return h


def dedisp_series(v: np.ndarray, bw_hz: float, f_lo_hz: float, dms, n_fft: int, n_int: int, taper: str = "none",
                  want_voltage: bool = False, fft_dtype=np.float64):
    """Steps 2-6 on the real voltage series v: float64 [n_dm][nb * L / n_int] intensities (and the valid dedispersed
    voltages [n_dm][nb * L] when asked).  Block b reads v[b L : b L + N]; its first D outputs are dropped (R20), so
    output sample j covers input times [D + j n_int, D + (j + 1) n_int).
    fft_dtype=np.float32 runs the two long FFTs and the chirp product in single precision (scipy.fft keeps the input
    precision): the experiment behind P:L151 / P:L219 / Fig. 8, not part of the oracle proper."""
    v = np.asarray(v, dtype=np.float64)
    D, L = framing(bw_hz, f_lo_hz, dms, n_fft, n_int)
    nb = 0 if v.size < n_fft else (v.size - D) // L
    out = np.zeros((len(dms), nb * L // n_int))
    volt = np.zeros((len(dms), nb * L)) if want_voltage else None
    if fft_dtype == np.float64:
        rfft, irfft, cdt = np.fft.rfft, np.fft.irfft, np.complex128
    else:
        import scipy.fft as sf
        rfft, irfft, cdt = sf.rfft, sf.irfft, np.complex64
    hs = [chirp(bw_hz, f_lo_hz, dm, n_fft, taper).astype(cdt) for dm in dms]
    for b in range(nb):
        spec = rfft(v[b * L: b * L + n_fft].astype(fft_dtype))       # step 2
        for d, h in enumerate(hs):
            y = irfft(spec * h, n=n_fft)                              # steps 3, 4 (1/N on the inverse, R7)
            valid = np.asarray(y[D:], dtype=np.float64)              # step 5
            if want_voltage:
                volt[d, b * L:(b + 1) * L] = valid
            out[d, b * L // n_int:(b + 1) * L // n_int] = (valid * valid).reshape(-1, n_int).sum(1)   # step 6
    return (out, volt) if want_voltage else out


def fullband(spec_int8: np.ndarray, bw_hz: float, f_lo_hz: float, dms, n_fft: int, n_int: int, taper: str = "none"):
    """The whole path of Fig. 4 on GSB spectra int8 [n_spec][C][2]."""
    return dedisp_series(gsb_inverse(spec_int8), bw_hz, f_lo_hz, dms, n_fft, n_int, taper)
