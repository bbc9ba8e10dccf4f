"""paper_2307_16758_b200 -- B200-native (sm_100a, fp64) explicit shallow-water time step on
unstructured triangle meshes: the data-parallel hot path of arxiv 2307.16758 as a C-ABI CUDA
library (include/swe_b200.h, csrc/) plus this thin ctypes binding.  No CPU fallback."""
from .binding import *  # noqa: F401,F403
from .binding import lib, create_from_config, SweError, SIGNATURES, SCHEMES, BC_KINDS, KERNEL_KINDS
