"""paper_1405_2915_b200 — B200-native SkePU-style data-parallel skeletons over smart containers.

The product is ``libskel.so`` (C ABI: ``include/skel.h``; CUDA kernels for sm_100a under ``csrc/``).
``binding`` is its thin ctypes front end. Importing the package loads the CUDA library and fails
loudly if it has not been built. The seeded input generators live OUTSIDE the package
(``skel_inputs.py`` at the repo root, numpy only), so that the oracle's tests and the reference
arm of ``bench.py`` never map the library they check.
"""
from . import binding as skel  # noqa: F401  (raises ImportError when libskel.so is missing)
from .binding import Context, Future, Matrix, SkelError, SkelInstance, Vector  # noqa: F401
