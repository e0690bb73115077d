"""Seeded synthetic GMRT-shaped voltage-beam inputs (shared by the oracle tests,
the CUDA parity tests, smoke() and bench.py).

This module holds NONE of the dedispersion method's arithmetic: it simulates
the sky + the GSB recorder.  It imports neither `oracle` nor the product
package.  The inputs stand in for the paper's GMRT observations (B0329+54,
B1937+21 ... P:L49), which are not available; DESIGN.md states the
recipe.

Recipe per frequency channel c (independent Philox stream keyed (seed, c)):
  noise   n[t] = sigma * (g1 + i g2)                      sigma = 20 counts per component
  pulse   p[t] = a * sigma * gate(t) * (g3 + i g4)        amplitude-modulated noise, gate = 1 while
                                                          ((t/dv - delay_c) mod P) < W
  ISM     p' = IFFT( FFT(p) * exp(-i*phi) )               ONE zero-padded whole-series transform, H = exp(-i*phi)
                                                          as PAPER.md P:L107 defines the ISM transfer function
          phi(f) = -2*pi*D*DM*[ 1/(f_c+f) - 1/f_c + f/f_c^2 ]  cold-plasma phase of PAPER.md Eq. 1 (its dispersive
                                                          part is -2*pi*D*DM/f) minus the constant and linear terms
                                                          (P:L112): low frequencies arrive later
  record  re, im = clip(rint(n + p'), -127, 127) as int8, layout [t][chan][2]
delay_c = D*DM*(1/f_c^2 - 1/f_top^2) is the inter-channel dispersion delay, kept so the band looks
like a real observation (the hot path does not remove it).
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass, replace
from typing import Sequence, Tuple

import numpy as np
import scipy.fft

D_HZ2_S = 4.148808e15  # P:L117, in Hz^2 s per pc cm^-3


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config: observing set-up + injected pulsar + transform sizes."""
    name: str
    n_chan: int
    bw_hz: float
    f_center_hz: float
    duration_s: float
    dm_trials: Tuple[float, ...]
    n_fft: int
    n_int: int
    pulse_period_s: float
    pulse_width_s: float
    pulse_amp_sigma: float
    pulse_dm: float
    seed: int
    sigma: float = 20.0
    chunk_s: float = 0.0  # >0: streamed from pinned host memory in chunks of this length

    @property
    def chan_width_hz(self) -> float:
        return self.bw_hz / self.n_chan

    @property
    def n_samp(self) -> int:
        """Complex samples per channel (one per 1/dv seconds)."""
        return int(round(self.duration_s * self.chan_width_hz))

    def scaled(self, duration_s: float) -> "Workload":
        return replace(self, duration_s=duration_s)


# BASELINE.json configs[0..4]; seeds: configs[0] says "seed 0", the others take their index.
WORKLOADS = {
    "tiny": Workload("tiny", 64, 16e6, 325e6, 0.25, (10.0,), 1024, 16, 5e-3, 50e-6, 3.0, 10.0, 0),
    "gmrt16": Workload("gmrt16", 256, 16e6, 325e6, 8.0, (57.0,), 2048, 8, 33e-3, 1e-3, 2.0, 57.0, 1),
    "gmrt32": Workload("gmrt32", 512, 32e6, 325e6, 16.0, (71.0,), 4096, 4, 1.6e-3, 30e-6, 2.0, 71.0, 2,
                       chunk_s=1.0),
    "lowfreq": Workload("lowfreq", 512, 16e6, 150e6, 16.0, (150.0,), 16384, 32, 250e-3, 5e-3, 2.0, 150.0, 3),
    "wideband": Workload("wideband", 2048, 400e6, 400e6, 8.0,
                         tuple(90.0 + 2.5 * i for i in range(8)), 16384, 64, 5e-3, 100e-6, 2.0, 100.0, 4),
}
WORKLOAD_ORDER = ("tiny", "gmrt16", "gmrt32", "lowfreq", "wideband")


def chan_freqs_hz(w: Workload) -> np.ndarray:
    dv = w.chan_width_hz
    return w.f_center_hz - 0.5 * w.bw_hz + (np.arange(w.n_chan) + 0.5) * dv


def _next_pow2(n: int) -> int:
    p = 1
    while p < n:
        p <<= 1
    return p


def _ism_phase(dm: float, f_c: float, f: np.ndarray) -> np.ndarray:
    """Cold-plasma propagation phase phi (radians) of PAPER.md Eq. 1 relative to the channel centre, with the constant
    and the linear (pure delay) terms removed (Eq. 1-2).  Eq. 1's dispersive part is
    -2 pi (L f_p^2 / 2c) / f = -2 pi D DM / f; the ISM transfer function is exp(-i phi), whose group delay
    (1/2 pi) dphi/df = D DM / f^2 is the dispersion delay law of P:L39-41."""
    return -2.0 * np.pi * D_HZ2_S * dm * (1.0 / (f_c + f) - 1.0 / f_c + f / (f_c * f_c))


def _gen_channel(w: Workload, c: int, f_c: float, f_top: float, t0: int, n: int, clip: bool = True) -> np.ndarray:
    """int8 [n][2] for channel c, samples t0 .. t0+n-1 of the full series (the full series is
    always synthesised so that any window is consistent; windows are cut afterwards)."""
    T = w.n_samp
    dv = w.chan_width_hz
    rng = np.random.Generator(np.random.Philox(key=w.seed, counter=[0, 0, 0, c]))
    noise = rng.standard_normal((T, 2), dtype=np.float32) * np.float32(w.sigma)
    delay = D_HZ2_S * w.pulse_dm * (1.0 / (f_c * f_c) - 1.0 / (f_top * f_top))
    tt = np.arange(T, dtype=np.float64) / dv - delay
    gate = np.mod(tt, w.pulse_period_s) < w.pulse_width_s
    idx = np.nonzero(gate)[0]
    g = rng.standard_normal((idx.size, 2))
    if idx.size and w.pulse_amp_sigma > 0.0:
        lo, hi = f_c - 0.5 * dv, f_c + 0.5 * dv
        smear = D_HZ2_S * abs(w.pulse_dm) * (1.0 / (lo * lo) - 1.0 / (hi * hi)) * dv
        pad = int(np.ceil(smear)) + 8
        nfft = _next_pow2(T + 2 * pad)
        p = np.zeros(nfft, dtype=np.complex128)
        p[pad + idx] = w.pulse_amp_sigma * w.sigma * (g[:, 0] + 1j * g[:, 1])
        f = scipy.fft.fftfreq(nfft, d=1.0 / dv)
        P = scipy.fft.fft(p)
        P *= np.exp(-1j * _ism_phase(w.pulse_dm, f_c, f))
        p = scipy.fft.ifft(P)[pad:pad + T]
        noise[:, 0] += p.real.astype(np.float32)
        noise[:, 1] += p.imag.astype(np.float32)
    v = np.rint(noise[t0:t0 + n])
    if clip:
        np.clip(v, -127, 127, out=v)
    return v.astype(np.int8)


def generate(w: Workload, chans: Sequence[int] | None = None, t0: int = 0, n_samp: int | None = None,
             n_threads: int | None = None) -> np.ndarray:
    """int8 [n_samp][len(chans)][2], time-major like the GSB voltage-beam blocks.
    `chans` defaults to all channels; channel c always gets the same stream whatever subset is asked."""
    T = w.n_samp
    n = T - t0 if n_samp is None else n_samp
    assert 0 <= t0 and t0 + n <= T
    chans = list(range(w.n_chan)) if chans is None else list(chans)
    fcs = chan_freqs_hz(w)
    f_top = w.f_center_hz + 0.5 * w.bw_hz
    out = np.empty((n, len(chans), 2), dtype=np.int8)
    n_threads = n_threads or min(32, os.cpu_count() or 1)

    def work(i):
        out[:, i, :] = _gen_channel(w, chans[i], float(fcs[chans[i]]), f_top, t0, n)

    if n_threads <= 1 or len(chans) == 1:
        for i in range(len(chans)):
            work(i)
    else:
        with ThreadPoolExecutor(n_threads) as ex:
            list(ex.map(work, range(len(chans))))
    return out


def noise_only(n_samp: int, n_chan: int, seed: int, sigma: float = 20.0) -> np.ndarray:
    """White Gaussian int8 noise [n_samp][n_chan][2], clipped to +-127 (BASELINE configs' noise part)."""
    rng = np.random.Generator(np.random.Philox(key=seed))
    v = np.rint(rng.standard_normal((n_samp, n_chan, 2), dtype=np.float32) * np.float32(sigma))
    np.clip(v, -127, 127, out=v)
    return v.astype(np.int8)


def uniform_int8(n_samp: int, n_chan: int, seed: int) -> np.ndarray:
    """Every int8 value including -128, uniformly (edge-case input for the unpack)."""
    rng = np.random.Generator(np.random.Philox(key=seed))
    return rng.integers(-128, 128, size=(n_samp, n_chan, 2), dtype=np.int8)
