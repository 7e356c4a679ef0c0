"""paper_1207_2367_b200 -- B200-native hot path of the HiGPUs method (arXiv 1207.2367).

Direct O(m N) FP64 evaluation of softened Newtonian gravity (acceleration, jerk, snap) with
the 6th-order Hermite predictor/corrector and block time steps around it, as hand-written
sm_100a CUDA kernels behind a C-ABI (include/nb.h, libnb.so).  This package is only the thin
binding: argument marshalling, no arithmetic.  There is no CPU fallback.
"""
from .nb import *  # noqa: F401,F403
from .nb import __all__  # noqa: F401
