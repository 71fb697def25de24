"""B200-native SFFT subtraction (arxiv 2509.18544's difference-imaging hot path).

The product is libsfft.so (C ABI in include/sfft.h, CUDA kernels in csrc/); `sfft` is its thin
ctypes binding and `starfield` the seeded synthetic input generators.
"""
from . import starfield  # noqa: F401
from .sfft import SfftError, SfftPlan, load_library, probe_fp64, solve_static, version  # noqa: F401
