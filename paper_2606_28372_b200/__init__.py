"""paper_2606_28372_b200 -- B200-native batched constraint-aware evolutionary auto-tuning steps.

Thin Python binding over the C ABI of ``include/cao.h`` (``libcao.so``, hand-written CUDA for sm_100a).
It only marshals arguments: PyTorch provides device memory and streams, every step of the hot path
(enumeration, operators, snap, validity, repair, lookup, selection) runs in the library's kernels.
There is no CPU fallback: importing :mod:`.api` objects without the built library raises.
"""
from .api import (Space, Runs, HParams, Variant, ALGOS, CaoError, lib, launch_count, test_philox, test_exp_neg, test_curand_philox, int_peak,
                  profile_enable, profile_read)  # noqa: F401
