"""B200-native bit-packed checkerboard Metropolis sweep of the 3D +-J Edwards-Anderson spin glass (arXiv 1411.0127).

`binding` wraps the C-ABI library `libising_b200.so` (include/ising.h); `synth` makes the seeded synthetic
inputs; `build` compiles the library in-tree for sm_100a.  The compute path is CUDA only.
"""
from . import synth  # noqa: F401
from .binding import LAYOUT_AUTO, LAYOUT_BATCH, LAYOUT_SAMPLE_PACKED, MINSTD, MT19937_SHARED, PHILOX, PHILOX_SHARED, PR_SHARED, Ising, IsingError, IsingSlab  # noqa: F401
