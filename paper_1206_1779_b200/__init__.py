"""B200-native residual + analytic Newton matrix of the ghost/gluon DSEs (arXiv:1206.1779).

Public API: the C ABI of include/dse.h (libdse_b200.so) and its thin binding `binding.Dse`.
"""
from .binding import Dse, DseError, DseParams, params_from_workload, load_library, DSE_FLAG_GEOMETRY_CACHE, DSE_FLAG_ANGULAR_TANH_SINH, DSE_FLAG_RADIAL_SPLIT, DSE_FLAG_USER_TABLES, DSE_FLAG_CONST_COEF, DSE_FLAG_PER_SYSTEM_KERNELS  # noqa: F401
