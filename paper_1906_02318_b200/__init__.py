"""B200-native (sm_100a) MPMI-SC tick: thin Python binding over the C-ABI library libmpmi.so.

Argument marshalling only -- every step of the path (sampler, lift, rollout, safe test, selection)
runs in the CUDA kernels under csrc/.  There is no CPU fallback: importing `mpmi` without the
built library raises.
"""
from .mpmi import (Context, Result, MpmiError, load_library, library_path, SAMPLER_PHILOX,  # noqa: F401
                   SAMPLER_GRID, LIFT_MONO, LIFT_RFF, DUMP_NONE, DUMP_PHYS, DUMP_LIFTED)
