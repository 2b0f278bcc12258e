"""B200-native hot path of CHORUS-MHD (arxiv 2502.17805): SD residual of compressible MHD + GLM on curved hexahedra
and the SSPRK(5,3) update, as hand-written CUDA kernels for sm_100a behind a C ABI (include/chorus.h)."""
from . import inputs  # noqa: F401
from .binding import Chorus, ChorusError, get_operators, fp64_peak, diagnostics_static, lib, SYMBOLS, LIB_PATH  # noqa: F401
