"""B200-native channelised overlap-save coherent dedispersion (De & Gupta, arXiv:1509.00186).

The product is libdedisp.so (CUDA, sm_100a) behind the C ABI of include/dedisp.h; this package is the thin ctypes
binding with the same names.  Importing fails loudly when the library has not been built."""
from .binding import (DedispError, FullbandPlan, Info, LIB_PATH, Plan, SYMBOLS, TAPER, UBENCH_FORMS, dedisp_fold, dedisp_framing,
                      dedisp_fullband_framing, dedisp_plan, dedisp_plan_shard, dedisp_ubench_fp32, lib)

__all__ = ["DedispError", "FullbandPlan", "Info", "LIB_PATH", "Plan", "SYMBOLS", "TAPER", "UBENCH_FORMS", "dedisp_fold", "dedisp_framing",
           "dedisp_fullband_framing", "dedisp_plan", "dedisp_plan_shard", "dedisp_ubench_fp32", "lib"]
