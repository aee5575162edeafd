"""paper_2504_07948_b200 -- B200-native (sm_100a) batched Slater-Jastrow electron-move engine.

The product is the C-ABI CUDA library ``libqmc_b200.so`` (sources in ``csrc/``, header in
``include/qmc.h``).  This package is its thin Python binding: the functions have the ABI's names and
only marshal arguments; PyTorch supplies device memory and streams.  There is no CPU fallback.

Build:  ``python -m paper_2504_07948_b200.build``
"""
from .binding import *  # noqa: F401,F403
from .binding import EXPORTED, LIB_PATH, QmcError, STAGES, System, Walkers, load_library  # noqa: F401
