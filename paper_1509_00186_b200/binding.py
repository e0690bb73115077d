"""ctypes binding of libdedisp (include/dedisp.h).  Argument marshalling only: every step of the path runs in the
library's CUDA kernels.  There is no CPU fallback: if the library is missing or fails to load, importing raises."""
from __future__ import annotations

import ctypes as C
import os
from typing import Sequence

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libdedisp.so")

OK, EINVAL, ENOMEM, ECUDA, ESHORT, ENODEV, ETOOBIG = 0, -1, -2, -3, -4, -5, -6
TAPER = {"none": 0, "hann": 1, "welch": 2}

# every symbol include/dedisp.h declares (tests check that the library exports all of them)
SYMBOLS = (
    "dedisp_framing", "dedisp_plan", "dedisp_plan_shard", "dedisp_shard_time_offset", "dedisp_get_info", "dedisp_out_samples", "dedisp_reserve", "dedisp_execute",
    "dedisp_execute_add", "dedisp_execute_static",
    "dedisp_stream_begin", "dedisp_stream_push", "dedisp_stream_sync", "dedisp_stream_end", "dedisp_profile_enable",
    "dedisp_profile_read", "dedisp_band_samples", "dedisp_band_shifts", "dedisp_band_sum", "dedisp_fold", "dedisp_destroy",
    "dedisp_strerror", "dedisp_last_cuda_error", "dedisp_debug_unpack", "dedisp_debug_chirp", "dedisp_debug_voltage",
    "dedisp_ubench_fp32",
    "dedisp_fullband_framing", "dedisp_fullband_plan", "dedisp_fullband_get_framing", "dedisp_fullband_out_samples",
    "dedisp_fullband_execute", "dedisp_fullband_debug_series", "dedisp_fullband_destroy",
)


class Info(C.Structure):
    _fields_ = [("n_chan", C.c_int), ("n_dm", C.c_int), ("n_fft", C.c_int), ("n_int", C.c_int),
                ("head", C.c_int), ("tail", C.c_int), ("L", C.c_int),
                ("chan_width_hz", C.c_double), ("max_smear_samples", C.c_double), ("nfft_rule", C.c_int)]


class DedispError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        msg = _lib.dedisp_strerror(code).decode()
        if code == ECUDA:
            msg += f" [cudaError {_lib.dedisp_last_cuda_error()}]"
        super().__init__(f"{where}: {msg} ({code})")


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python paper_1509_00186_b200/build.py` "
                          "(the CUDA library is the product; there is no fallback)")
    L = C.CDLL(LIB_PATH)
    dp, ip, vp, ll = C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_void_p, C.c_longlong
    L.dedisp_framing.argtypes = [C.c_int, C.c_double, C.c_double, dp, C.c_int, C.c_int, C.c_int, ip, ip, ip]
    L.dedisp_plan.argtypes = [C.POINTER(vp), C.c_int, C.c_double, C.c_double, dp, C.c_int, C.c_int, C.c_int, C.c_uint]
    L.dedisp_plan_shard.argtypes = [C.POINTER(vp), C.c_int, C.c_double, C.c_double, dp, C.c_int, C.c_int, C.c_int, C.c_uint,
                                    C.c_int, C.c_int, C.c_uint]
    L.dedisp_shard_time_offset.argtypes = [vp]
    L.dedisp_shard_time_offset.restype = ll
    llp = C.POINTER(ll)
    L.dedisp_fullband_framing.argtypes = [C.c_double, C.c_double, dp, C.c_int, ll, C.c_int, ip, llp]
    L.dedisp_fullband_plan.argtypes = [C.POINTER(vp), C.c_int, C.c_double, C.c_double, dp, C.c_int, ll, C.c_int, C.c_uint]
    L.dedisp_fullband_get_framing.argtypes = [vp, ip, llp, ip, ip]
    L.dedisp_fullband_out_samples.argtypes = [vp, ll]
    L.dedisp_fullband_out_samples.restype = ll
    L.dedisp_fullband_execute.argtypes = [vp, vp, ll, vp, ll, vp]
    L.dedisp_fullband_debug_series.argtypes = [vp, vp, ll, vp, vp]
    L.dedisp_fullband_destroy.argtypes = [vp]
    L.dedisp_get_info.argtypes = [vp, C.POINTER(Info)]
    L.dedisp_out_samples.argtypes = [vp, ll]
    L.dedisp_out_samples.restype = ll
    L.dedisp_reserve.argtypes = [vp, ll]
    L.dedisp_execute.argtypes = [vp, vp, ll, vp, ll, vp]
    L.dedisp_execute_add.argtypes = [vp, vp, ll, vp, ll, vp]
    L.dedisp_execute_static.argtypes = [vp, vp, ll, vp, ll, vp]
    L.dedisp_stream_begin.argtypes = [vp, ll]
    L.dedisp_stream_push.argtypes = [vp, vp, ll, vp, ll, C.POINTER(ll)]
    L.dedisp_stream_sync.argtypes = [vp]
    L.dedisp_stream_end.argtypes = [vp]
    L.dedisp_profile_enable.argtypes = [vp, C.c_int]
    L.dedisp_profile_read.argtypes = [vp, dp, dp, ip]
    L.dedisp_band_samples.argtypes = [vp, ll]
    L.dedisp_band_samples.restype = ll
    L.dedisp_band_shifts.argtypes = [vp, C.c_int, C.POINTER(ll)]
    L.dedisp_band_sum.argtypes = [vp, vp, ll, ll, vp, ll, vp]
    L.dedisp_fold.argtypes = [vp, ll, C.c_double, C.c_double, C.c_double, C.c_int, vp, vp, vp]
    L.dedisp_destroy.argtypes = [vp]
    L.dedisp_ubench_fp32.argtypes = [C.c_int, C.c_int, dp, dp]
    L.dedisp_strerror.argtypes = [C.c_int]
    L.dedisp_strerror.restype = C.c_char_p
    L.dedisp_last_cuda_error.argtypes = []
    L.dedisp_debug_unpack.argtypes = [vp, vp, ll, C.c_int, ll, vp, vp]
    L.dedisp_debug_chirp.argtypes = [vp, C.c_int, C.c_int, vp]
    L.dedisp_debug_voltage.argtypes = [vp, vp, ll, C.c_int, ll, vp, vp]
    return L


_lib = _load()


def lib() -> C.CDLL:
    return _lib


def _check(rc: int, where: str) -> None:
    if rc != OK:
        raise DedispError(rc, where)


def _dm_array(dm: Sequence[float]):
    dm = [float(v) for v in dm]
    return (C.c_double * len(dm))(*dm), len(dm)


def dedisp_framing(n_chan: int, bw_hz: float, f_center_hz: float, dm: Sequence[float], n_fft: int, n_int: int):
    """(head, tail, L) of the overlap-save framing; host arithmetic only (no GPU needed)."""
    arr, n = _dm_array(dm)
    h, t, l = C.c_int(), C.c_int(), C.c_int()
    _check(_lib.dedisp_framing(n_chan, bw_hz, f_center_hz, arr, n, n_fft, n_int, C.byref(h), C.byref(t), C.byref(l)),
           "dedisp_framing")
    return h.value, t.value, l.value


def dedisp_plan(n_chan: int, bw_hz: float, f_center_hz: float, dm: Sequence[float], n_fft: int, n_int: int,
                taper: str = "none") -> "Plan":
    return Plan(n_chan, bw_hz, f_center_hz, dm, n_fft, n_int, taper)


SHARD_FULL_INPUT, SHARD_OWN_FRAMING = 1, 2


def dedisp_plan_shard(n_chan_total: int, bw_hz_total: float, f_center_hz_total: float, dm: Sequence[float], n_fft: int,
                      n_int: int, chan0: int, n_chan: int, taper: str = "none", full_input: bool = False,
                      own_framing: bool = False) -> "Plan":
    """Plan for channels chan0 .. chan0 + n_chan - 1 of the band (dedisp.h: dedisp_plan_shard)."""
    return Plan(n_chan_total, bw_hz_total, f_center_hz_total, dm, n_fft, n_int, taper,
                shard=(chan0, n_chan, (SHARD_FULL_INPUT if full_input else 0) | (SHARD_OWN_FRAMING if own_framing else 0)))


UBENCH_FORMS = ("plain 2xFADD2", "times-i 2xFADD2 (lane-swapped operand)", "twiddle conventional FMUL2+FFMA2+2xFADD2",
                "twiddle folded 3xFFMA2 (v=2a-u)", "twiddle folded, rotated by i", "twiddle folded 4xFFMA2",
                "immediate twiddle folded 3xFFMA2", "immediate twiddle conventional")


def dedisp_ubench_fp32(form: int, iters: int = 4096):
    """(SM sub-partition cycles per butterfly, ms of the launch) for instruction form `form` (see dedisp.h)."""
    cyc, ms = C.c_double(), C.c_double()
    _check(_lib.dedisp_ubench_fp32(form, iters, C.byref(cyc), C.byref(ms)), "dedisp_ubench_fp32")
    return cyc.value, ms.value


def dedisp_fold(d_series, t0_s: float, dt_s: float, period_s: float, n_bins: int, stream=None):
    """Fold a 1-D CUDA float32 series at period_s: returns (sum per bin float32 [n_bins], count per bin int32 [n_bins])."""
    import torch
    assert d_series.is_cuda and d_series.dtype == torch.float32 and d_series.is_contiguous() and d_series.dim() == 1
    s = torch.empty(n_bins, dtype=torch.float32, device=d_series.device)
    n = torch.empty(n_bins, dtype=torch.int32, device=d_series.device)
    st = torch.cuda.current_stream(d_series.device).cuda_stream if stream is None else stream
    _check(_lib.dedisp_fold(d_series.data_ptr(), d_series.numel(), t0_s, dt_s, period_s, n_bins, s.data_ptr(),
                            n.data_ptr(), st), "dedisp_fold")
    return s, n


class Plan:
    """Owns a dedisp_plan_t.  Methods take torch tensors (or raw pointers) and pass pointers through."""

    def __init__(self, n_chan, bw_hz, f_center_hz, dm, n_fft, n_int, taper="none", shard=None):
        self._h = C.c_void_p()
        arr, n = _dm_array(dm)
        if shard is None:
            _check(_lib.dedisp_plan(C.byref(self._h), n_chan, bw_hz, f_center_hz, arr, n, n_fft, n_int, TAPER[taper]),
                   "dedisp_plan")
            self.in_chan = n_chan
        else:
            chan0, n_shard, sflags = shard
            _check(_lib.dedisp_plan_shard(C.byref(self._h), n_chan, bw_hz, f_center_hz, arr, n, n_fft, n_int,
                                          TAPER[taper], chan0, n_shard, sflags), "dedisp_plan_shard")
            self.in_chan = n_chan if sflags & SHARD_FULL_INPUT else n_shard  # channels per row of execute()'s input
        self.time_offset = int(_lib.dedisp_shard_time_offset(self._h))
        info = Info()
        _check(_lib.dedisp_get_info(self._h, C.byref(info)), "dedisp_get_info")
        self.info = info
        self.n_chan, self.n_dm, self.n_fft, self.n_int = info.n_chan, info.n_dm, info.n_fft, info.n_int
        self.head, self.tail, self.L = info.head, info.tail, info.L

    # -- sizes ------------------------------------------------------------------------------------------------
    def out_samples(self, n_samp: int) -> int:
        return int(_lib.dedisp_out_samples(self._h, n_samp))

    def n_blocks(self, n_samp: int) -> int:
        return self.out_samples(n_samp) // (self.L // self.n_int)

    def reserve(self, n_samp: int) -> None:
        _check(_lib.dedisp_reserve(self._h, n_samp), "dedisp_reserve")

    # -- one-shot ---------------------------------------------------------------------------------------------
    def execute(self, d_in, d_out=None, stream=None, add: bool = False):
        """d_in: CUDA int8 tensor [n_samp][n_chan][2]; returns/fills CUDA float32 [n_dm][n_chan][n_out].
        add=True: dedisp_execute_add, the intensities are added to d_out (second polarisation)."""
        import torch
        assert d_in.is_cuda and d_in.dtype == torch.int8 and d_in.is_contiguous()
        assert d_in.dim() == 3 and d_in.shape[1] == self.in_chan and d_in.shape[2] == 2
        assert not add or d_out is not None, "add=True needs the first polarisation's output"
        n_samp = d_in.shape[0]
        n_out = self.out_samples(n_samp)
        if d_out is None:
            d_out = torch.empty((self.n_dm, self.n_chan, max(n_out, 0)), dtype=torch.float32, device=d_in.device)
        assert d_out.is_cuda and d_out.dtype == torch.float32 and d_out.is_contiguous()
        assert d_out.dim() == 3 and d_out.shape[0] == self.n_dm and d_out.shape[1] == self.n_chan
        st = torch.cuda.current_stream(d_in.device).cuda_stream if stream is None else stream
        fn = _lib.dedisp_execute_add if add else _lib.dedisp_execute
        _check(fn(self._h, d_in.data_ptr(), n_samp, d_out.data_ptr(), d_out.shape[2], st), "dedisp_execute")
        return d_out

    def execute_static(self, d_in, d_out, stream=None):
        """dedisp_execute_static: execute() without any allocation (the scratch is a static 64 MiB device array shared
        by all calls; DedispError(ETOOBIG) beyond it).  d_out must be given: this call creates nothing."""
        import torch
        assert d_in.is_cuda and d_in.dtype == torch.int8 and d_in.is_contiguous()
        assert d_in.dim() == 3 and d_in.shape[1] == self.in_chan and d_in.shape[2] == 2
        assert d_out.is_cuda and d_out.dtype == torch.float32 and d_out.is_contiguous()
        assert d_out.dim() == 3 and d_out.shape[0] == self.n_dm and d_out.shape[1] == self.n_chan
        st = torch.cuda.current_stream(d_in.device).cuda_stream if stream is None else stream
        _check(_lib.dedisp_execute_static(self._h, d_in.data_ptr(), d_in.shape[0], d_out.data_ptr(), d_out.shape[2], st),
               "dedisp_execute_static")
        return d_out

    def execute_ptr(self, in_ptr: int, n_samp: int, out_ptr: int, out_stride: int, stream: int = 0) -> None:
        _check(_lib.dedisp_execute(self._h, in_ptr, n_samp, out_ptr, out_stride, stream), "dedisp_execute")

    # -- streaming --------------------------------------------------------------------------------------------
    def stream_begin(self, max_chunk_samp: int) -> None:
        _check(_lib.dedisp_stream_begin(self._h, max_chunk_samp), "dedisp_stream_begin")

    def stream_push(self, h_in, h_out, col0: int = 0) -> int:
        """h_in: pinned int8 [n][C][2]; h_out: pinned float32 [n_dm][C][stride], this chunk's outputs land in columns
        [col0, col0 + returned count) of every row.  Returns the number of outputs per (dm, chan) this chunk completed."""
        import torch
        assert not h_in.is_cuda and h_in.dtype == torch.int8 and h_in.is_contiguous()
        assert h_in.dim() == 3 and h_in.shape[1] == self.n_chan and h_in.shape[2] == 2
        assert not h_out.is_cuda and h_out.dtype == torch.float32 and h_out.is_contiguous()
        assert h_out.dim() == 3 and h_out.shape[0] == self.n_dm and h_out.shape[1] == self.n_chan
        assert 0 <= col0 <= h_out.shape[2]
        n = C.c_longlong(0)
        # the library checks out_stride >= n_out; the room left behind col0 is checked here
        rc = _lib.dedisp_stream_push(self._h, h_in.data_ptr(), h_in.shape[0], h_out.data_ptr() + 4 * col0,
                                     h_out.shape[2], C.byref(n))
        _check(rc, "dedisp_stream_push")
        assert col0 + n.value <= h_out.shape[2], "h_out too short for this chunk's outputs"
        return int(n.value)

    def stream_sync(self) -> None:
        _check(_lib.dedisp_stream_sync(self._h), "dedisp_stream_sync")

    def stream_end(self) -> None:
        _check(_lib.dedisp_stream_end(self._h), "dedisp_stream_end")

    # -- sub-band alignment + band sum ------------------------------------------------------------------------
    def band_samples(self, n_out: int) -> int:
        return int(_lib.dedisp_band_samples(self._h, n_out))

    def band_shifts(self, d: int):
        import numpy as np
        sh = (C.c_longlong * self.n_chan)()
        _check(_lib.dedisp_band_shifts(self._h, d, sh), "dedisp_band_shifts")
        return np.asarray(list(sh), dtype=np.int64)

    def band_sum(self, d_out, d_series=None, stream=None):
        """d_out: CUDA float32 [n_dm][n_chan][n_out] (from execute) -> CUDA float32 [n_dm][n_series]."""
        import torch
        assert d_out.is_cuda and d_out.dtype == torch.float32 and d_out.is_contiguous()
        assert d_out.dim() == 3 and d_out.shape[0] == self.n_dm and d_out.shape[1] == self.n_chan
        n_out = d_out.shape[2]
        n_ser = self.band_samples(n_out)
        if d_series is None:
            d_series = torch.empty((self.n_dm, max(n_ser, 0)), dtype=torch.float32, device=d_out.device)
        assert d_series.is_cuda and d_series.dtype == torch.float32 and d_series.is_contiguous()
        assert d_series.dim() == 2 and d_series.shape[0] == self.n_dm
        st = torch.cuda.current_stream(d_out.device).cuda_stream if stream is None else stream
        _check(_lib.dedisp_band_sum(self._h, d_out.data_ptr(), n_out, n_out, d_series.data_ptr(), d_series.shape[1], st),
               "dedisp_band_sum")
        return d_series

    # -- kernel timing ----------------------------------------------------------------------------------------
    def profile_enable(self, on: bool = True) -> None:
        _check(_lib.dedisp_profile_enable(self._h, 1 if on else 0), "dedisp_profile_enable")

    def profile_read(self):
        """(ms in the corner-turn kernel, ms in the fused kernel, calls) summed since the last read."""
        a, b, n = C.c_double(), C.c_double(), C.c_int()
        _check(_lib.dedisp_profile_read(self._h, C.byref(a), C.byref(b), C.byref(n)), "dedisp_profile_read")
        return a.value, b.value, n.value

    # -- test hooks -------------------------------------------------------------------------------------------
    def debug_unpack(self, d_in, chan: int, block: int):
        import torch
        out = torch.empty((self.n_fft, 2), dtype=torch.float32, device=d_in.device)
        st = torch.cuda.current_stream(d_in.device).cuda_stream
        _check(_lib.dedisp_debug_unpack(self._h, d_in.data_ptr(), d_in.shape[0], chan, block, out.data_ptr(), st),
               "dedisp_debug_unpack")
        return out

    def debug_chirp(self, d: int, chan: int):
        import numpy as np
        h = np.empty((self.n_fft, 2), dtype=np.float32)
        _check(_lib.dedisp_debug_chirp(self._h, d, chan, h.ctypes.data), "dedisp_debug_chirp")
        return h[:, 0] + 1j * h[:, 1]

    def debug_voltage(self, d_in, chan: int, block: int):
        import torch
        out = torch.empty((self.n_dm, self.L, 2), dtype=torch.float32, device=d_in.device)
        st = torch.cuda.current_stream(d_in.device).cuda_stream
        _check(_lib.dedisp_debug_voltage(self._h, d_in.data_ptr(), d_in.shape[0], chan, block, out.data_ptr(), st),
               "dedisp_debug_voltage")
        return out

    # -- lifetime ---------------------------------------------------------------------------------------------
    def destroy(self) -> None:
        if self._h:
            _lib.dedisp_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()


def dedisp_fullband_framing(bw_hz: float, f_lo_hz: float, dm: Sequence[float], n_fft: int, n_int: int):
    """(D, L) of the full-band mode (dedisp.h: dedisp_fullband_framing); host arithmetic only."""
    arr, n = _dm_array(dm)
    d, l = C.c_int(), C.c_longlong()
    _check(_lib.dedisp_fullband_framing(bw_hz, f_lo_hz, arr, n, n_fft, n_int, C.byref(d), C.byref(l)),
           "dedisp_fullband_framing")
    return d.value, l.value


class FullbandPlan:
    """Owns a dedisp_fullband_t: the paper's own full-band mode (dedisp.h).  Argument marshalling only."""

    def __init__(self, n_chan, bw_hz, f_lo_hz, dm, n_fft, n_int, taper="none"):
        self._h = C.c_void_p()
        arr, n = _dm_array(dm)
        _check(_lib.dedisp_fullband_plan(C.byref(self._h), n_chan, bw_hz, f_lo_hz, arr, n, n_fft, n_int, TAPER[taper]),
               "dedisp_fullband_plan")
        d, l, n1, n2 = C.c_int(), C.c_longlong(), C.c_int(), C.c_int()
        _check(_lib.dedisp_fullband_get_framing(self._h, C.byref(d), C.byref(l), C.byref(n1), C.byref(n2)),
               "dedisp_fullband_get_framing")
        self.n_chan, self.n_dm, self.n_fft, self.n_int = n_chan, n, n_fft, n_int
        self.D, self.L, self.n1, self.n2 = d.value, l.value, n1.value, n2.value

    def out_samples(self, n_spec: int) -> int:
        return int(_lib.dedisp_fullband_out_samples(self._h, n_spec))

    def execute(self, d_spec, d_out=None, stream=None):
        """d_spec: CUDA int8 [n_spec][n_chan][2] -> CUDA float32 [n_dm][n_out]."""
        import torch
        assert d_spec.is_cuda and d_spec.dtype == torch.int8 and d_spec.is_contiguous()
        assert d_spec.dim() == 3 and d_spec.shape[1] == self.n_chan and d_spec.shape[2] == 2
        n_out = self.out_samples(d_spec.shape[0])
        if d_out is None:
            d_out = torch.empty((self.n_dm, max(n_out, 0)), dtype=torch.float32, device=d_spec.device)
        assert d_out.is_cuda and d_out.dtype == torch.float32 and d_out.is_contiguous() and d_out.shape[0] == self.n_dm
        st = torch.cuda.current_stream(d_spec.device).cuda_stream if stream is None else stream
        _check(_lib.dedisp_fullband_execute(self._h, d_spec.data_ptr(), d_spec.shape[0], d_out.data_ptr(),
                                            d_out.shape[1], st), "dedisp_fullband_execute")
        return d_out

    def debug_series(self, d_spec):
        import torch
        out = torch.empty(d_spec.shape[0] * 2 * self.n_chan, dtype=torch.float32, device=d_spec.device)
        st = torch.cuda.current_stream(d_spec.device).cuda_stream
        _check(_lib.dedisp_fullband_debug_series(self._h, d_spec.data_ptr(), d_spec.shape[0], out.data_ptr(), st),
               "dedisp_fullband_debug_series")
        return out

    def destroy(self):
        if self._h:
            _lib.dedisp_fullband_destroy(self._h)
            self._h = C.c_void_p()

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
