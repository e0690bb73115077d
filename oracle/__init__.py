"""ctypes front-end of the fp64 CPU oracle (oracle/dedisp_oracle.c).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  The product package
(paper_1509_00186_b200) never imports this module, and this module never
imports the product package.

All arithmetic lives in the C file; this module only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass, field
from typing import Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dedisp_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no fast-math; -fcx-limited-range only selects the
    textbook (ac-bd, ad+bc) complex product instead of the NaN-recovering libcall)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fcx-limited-range", "-fPIC", "-shared", "-pthread",
             "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Cfg(C.Structure):
    _fields_ = [("n_chan", C.c_int), ("bw_hz", C.c_double), ("f_center_hz", C.c_double),
                ("n_dm", C.c_int), ("dm", C.POINTER(C.c_double)), ("n_fft", C.c_int),
                ("n_int", C.c_int), ("taper", C.c_int)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, ip, llp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.POINTER(C.c_longlong)
        cp = C.POINTER(_Cfg)
        L.oracle_dft_naive.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int]
        L.oracle_dft_naive.restype = None
        L.oracle_fft.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.oracle_fft_radix2.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.oracle_chan_width.argtypes = [cp]; L.oracle_chan_width.restype = C.c_double
        L.oracle_chan_freq.argtypes = [cp, C.c_int]; L.oracle_chan_freq.restype = C.c_double
        L.oracle_bin_freq.argtypes = [cp, C.c_int]; L.oracle_bin_freq.restype = C.c_double
        L.oracle_chirp_phase_cycles.argtypes = [C.c_double] * 3
        L.oracle_chirp_phase_cycles.restype = C.c_double
        L.oracle_taper.argtypes = [C.c_int, C.c_double, C.c_double]; L.oracle_taper.restype = C.c_double
        L.oracle_chirp.argtypes = [cp, C.c_int, C.c_int, C.c_void_p]; L.oracle_chirp.restype = None
        L.oracle_framing.argtypes = [cp, ip, ip, ip]
        L.oracle_smear_seconds.argtypes = [C.c_double] * 3; L.oracle_smear_seconds.restype = C.c_double
        L.oracle_nfft_rule.argtypes = [C.c_double]; L.oracle_nfft_rule.restype = C.c_longlong
        L.oracle_n_blocks.argtypes = [cp, C.c_longlong, C.c_int, C.c_int, C.c_int]
        L.oracle_n_blocks.restype = C.c_longlong
        L.oracle_dedisp.argtypes = [cp, C.c_void_p, C.c_longlong, C.c_void_p, C.c_longlong, C.c_int]
        L.oracle_dedisp.restype = C.c_longlong
        L.oracle_dedisp_units.argtypes = [cp, C.c_void_p, C.c_longlong, C.c_void_p, C.c_void_p, C.c_int,
                                          C.c_void_p, C.c_void_p, C.c_int]
        L.oracle_dedisp_units.restype = C.c_longlong
        L.oracle_unpack_block.argtypes = [cp, C.c_void_p, C.c_int, C.c_longlong, C.c_int, C.c_void_p]
        L.oracle_unpack_block.restype = None
        L.oracle_band_shifts.argtypes = [cp, C.c_int, C.c_void_p]
        L.oracle_band_shifts.restype = None
        L.oracle_band_sum.argtypes = [cp, C.c_void_p, C.c_longlong, C.c_longlong, C.c_void_p, C.c_longlong]
        L.oracle_band_sum.restype = C.c_longlong
        L.oracle_fold.argtypes = [C.c_void_p, C.c_longlong, C.c_double, C.c_double, C.c_double, C.c_int, C.c_void_p,
                                  C.c_void_p]
        L.oracle_fold.restype = None
        _lib = L
    return _lib


TAPER = {"none": 0, "hann": 1, "welch": 2}


@dataclass
class OracleConfig:
    """Parameters of the problem as the paper states them (observing
    frequency, bandwidth, DM) plus the channelisation and transform sizes."""
    n_chan: int
    bw_hz: float
    f_center_hz: float
    dm: Sequence[float]
    n_fft: int
    n_int: int
    taper: str = "none"
    _dm_arr: np.ndarray = field(init=False, repr=False)

    def __post_init__(self):
        self._dm_arr = np.ascontiguousarray(np.asarray(self.dm, dtype=np.float64).reshape(-1))

    def c(self) -> _Cfg:
        return _Cfg(self.n_chan, self.bw_hz, self.f_center_hz, len(self._dm_arr),
                    self._dm_arr.ctypes.data_as(C.POINTER(C.c_double)), self.n_fft, self.n_int,
                    TAPER[self.taper])

    @property
    def n_dm(self) -> int:
        return len(self._dm_arr)


def _cplx(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.complex128))


def dft_naive(x, sign: int = -1) -> np.ndarray:
    x = _cplx(x); out = np.empty_like(x)
    lib().oracle_dft_naive(x.ctypes.data, out.ctypes.data, x.size, sign)
    return out


def fft(x, sign: int = -1, force_radix2: bool = False) -> np.ndarray:
    """Unnormalised transform, kernel exp(sign*2*pi*i*k*n/N)."""
    y = _cplx(x).copy()
    f = lib().oracle_fft_radix2 if force_radix2 else lib().oracle_fft
    if f(y.ctypes.data, y.size, sign) != 0:
        raise ValueError("oracle fft: n must be a power of two")
    return y


def chan_width(cfg: OracleConfig) -> float:
    return lib().oracle_chan_width(C.byref(cfg.c()))


def chan_freq(cfg: OracleConfig, c: int) -> float:
    return lib().oracle_chan_freq(C.byref(cfg.c()), c)


def bin_freq(cfg: OracleConfig, k: int) -> float:
    return lib().oracle_bin_freq(C.byref(cfg.c()), k)


def chirp_phase_cycles(dm: float, f_c_hz: float, f_hz: float) -> float:
    return lib().oracle_chirp_phase_cycles(dm, f_c_hz, f_hz)


def taper(kind: str, f_hz: float, dv_hz: float) -> float:
    return lib().oracle_taper(TAPER[kind], f_hz, dv_hz)


def chirp(cfg: OracleConfig, d: int, c: int) -> np.ndarray:
    H = np.empty(cfg.n_fft, dtype=np.complex128)
    lib().oracle_chirp(C.byref(cfg.c()), d, c, H.ctypes.data)
    return H


def framing(cfg: OracleConfig):
    """(head, tail, L) of reading R9; raises when the transform is too short."""
    h, t, l = C.c_int(), C.c_int(), C.c_int()
    rc = lib().oracle_framing(C.byref(cfg.c()), C.byref(h), C.byref(t), C.byref(l))
    if rc != 0:
        raise ValueError(f"oracle framing invalid: head={h.value} tail={t.value} L={l.value}")
    return h.value, t.value, l.value


def smear_seconds(dm: float, f_lo_hz: float, f_hi_hz: float) -> float:
    return lib().oracle_smear_seconds(dm, f_lo_hz, f_hi_hz)


def nfft_rule(smear_samples: float) -> int:
    return lib().oracle_nfft_rule(smear_samples)


def n_blocks(cfg: OracleConfig, n_samp: int) -> int:
    h, t, l = framing(cfg)
    return lib().oracle_n_blocks(C.byref(cfg.c()), n_samp, h, t, l)


def _check_in(cfg: OracleConfig, x: np.ndarray) -> np.ndarray:
    x = np.ascontiguousarray(x)
    if x.dtype != np.int8 or x.ndim != 3 or x.shape[1] != cfg.n_chan or x.shape[2] != 2:
        raise ValueError("input must be int8 [T][n_chan][2]")
    return x


def dedisp(cfg: OracleConfig, x: np.ndarray, n_threads: int = 1) -> np.ndarray:
    """One-shot oracle: int8 [T][C][2] -> float64 [n_dm][C][n_out]."""
    x = _check_in(cfg, x)
    h, t, l = framing(cfg)
    nb = n_blocks(cfg, x.shape[0])
    nout = nb * (l // cfg.n_int)
    out = np.zeros((cfg.n_dm, cfg.n_chan, max(nout, 0)), dtype=np.float64)
    if nout == 0:
        return out
    rc = lib().oracle_dedisp(C.byref(cfg.c()), x.ctypes.data, x.shape[0], out.ctypes.data, nout, n_threads)
    if rc != nout:
        raise RuntimeError(f"oracle_dedisp failed: {rc}")
    return out


def dedisp_units(cfg: OracleConfig, x: np.ndarray, chans, blocks, n_threads: int = 1,
                 want_voltage: bool = False):
    """Sampled (channel, block) units -> [n_units][n_dm][L/n_int] (and the complex
    dedispersed voltages [n_units][n_dm][L] when want_voltage)."""
    x = _check_in(cfg, x)
    h, t, l = framing(cfg)
    chans = np.ascontiguousarray(np.asarray(chans, dtype=np.int32))
    blocks = np.ascontiguousarray(np.asarray(blocks, dtype=np.int64))
    assert chans.shape == blocks.shape and chans.ndim == 1
    nu = chans.size
    out = np.zeros((nu, cfg.n_dm, l // cfg.n_int), dtype=np.float64)
    volt = np.zeros((nu, cfg.n_dm, l), dtype=np.complex128) if want_voltage else None
    rc = lib().oracle_dedisp_units(C.byref(cfg.c()), x.ctypes.data, x.shape[0], chans.ctypes.data,
                                   blocks.ctypes.data, nu, out.ctypes.data,
                                   volt.ctypes.data if want_voltage else None, n_threads)
    if rc < 0:
        raise RuntimeError(f"oracle_dedisp_units failed: {rc}")
    return (out, volt) if want_voltage else out


def unpack_block(cfg: OracleConfig, x: np.ndarray, c: int, b: int) -> np.ndarray:
    x = _check_in(cfg, x)
    h, t, l = framing(cfg)
    dst = np.empty((cfg.n_fft, 2), dtype=np.float64)
    lib().oracle_unpack_block(C.byref(cfg.c()), x.ctypes.data, c, b, l, dst.ctypes.data)
    return dst


def band_shifts(cfg: OracleConfig, d: int) -> np.ndarray:
    """Whole-output-sample delays of every channel relative to the earliest one (NEXT-3, reading R16)."""
    sh = np.zeros(cfg.n_chan, dtype=np.int64)
    lib().oracle_band_shifts(C.byref(cfg.c()), d, sh.ctypes.data)
    return sh


def band_sum(cfg: OracleConfig, out: np.ndarray) -> np.ndarray:
    """out float64 [n_dm][n_chan][n_out] -> aligned band sum float64 [n_dm][n_series]."""
    out = np.ascontiguousarray(out, dtype=np.float64)
    assert out.ndim == 3 and out.shape[0] == cfg.n_dm and out.shape[1] == cfg.n_chan
    n_out = out.shape[2]
    series = np.zeros((cfg.n_dm, n_out), dtype=np.float64)
    n_ser = lib().oracle_band_sum(C.byref(cfg.c()), out.ctypes.data, n_out, n_out, series.ctypes.data, n_out)
    return np.ascontiguousarray(series[:, :n_ser])


def fold(series, t0_s: float, dt_s: float, period_s: float, n_bins: int):
    """Fold a time series at `period_s` (reading R17): (sum per phase bin, samples per phase bin)."""
    series = np.ascontiguousarray(series, dtype=np.float64).reshape(-1)
    s = np.zeros(n_bins, dtype=np.float64)
    n = np.zeros(n_bins, dtype=np.int64)
    lib().oracle_fold(series.ctypes.data, series.size, t0_s, dt_s, period_s, n_bins, s.ctypes.data, n.ctypes.data)
    return s, n

