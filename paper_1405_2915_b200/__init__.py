"""paper_1405_2915_b200 — B200-native SkePU-style data-parallel skeletons over smart containers.

The product is ``libskel.so`` (C ABI: ``include/skel.h``; CUDA kernels for sm_100a under ``csrc/``).
``binding`` is its thin ctypes front end; ``inputs`` holds the seeded synthetic input generators.
Importing the package loads the CUDA library and fails loudly if it has not been built.
"""
from . import inputs  # noqa: F401  (numpy only)
from . import binding as skel  # noqa: F401  (raises ImportError when libskel.so is missing)
from .binding import Context, Matrix, SkelError, SkelInstance, Vector  # noqa: F401
