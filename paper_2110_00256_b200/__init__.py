"""B200-native (sm_100a) implementation of the PICSAR-QED Monte Carlo hot path (arXiv 2110.00256).

``Context`` wraps the C ABI of ``include/picsarqed.h`` (``libpicsarqed.so``, hand-written CUDA);
``workloads`` holds the seeded synthetic input generators.  There is no CPU fallback.
"""
from . import workloads  # noqa: F401
from .binding import (F32, F64, LEPTON, NOALLOC_MAX_N, PHOTON, UNITS_HL_MEV, UNITS_LIBRARY, UNITS_NORM_LAMBDA, UNITS_NORM_OMEGA,  # noqa: F401
                      UNITS_SI, TAB_BW_P, TAB_LNG, TAB_LNT, TAB_QS_LNP, Context,  # noqa: F401
                      PicsarQedError, Species, TableParams, lib)
from .build import build, lib_path  # noqa: F401
