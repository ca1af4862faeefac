"""paper_2509_21754_b200 -- B200-native (sm_100a) FITrig hot path: tLISI map + candidate detection.

Thin ctypes binding over the C ABI of include/fitrig.h (argument marshalling only; every step of the
path runs in the CUDA kernels of csrc/).  PyTorch is used by callers for device memory and streams.
"""
from .binding import (  # noqa: F401
    BRANCH_FREQUENCY, BRANCH_IMAGE, INTERP_BICUBIC, INTERP_BILINEAR, INTERP_MAKIMA, INTERP_SPLINE, REF_ABS, REF_FLOOR, REF_LITERAL, Candidate, Context, FitrigError, Plan,
    choose_accumulate, choose_accumulate_static, exported_symbols, last_error, lib_path, load_library, plan_query, version,
)
