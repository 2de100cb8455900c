"""paper_2110_14557_b200 -- B200-native (sm_100a) hot path of the SLDG Vlasov-Poisson solver
(Einkemmer & Moriggl, arXiv 2110.14557): thin ctypes binding over the C-ABI in include/sldg.h.

Argument marshalling only; every step of the path runs in the CUDA kernels under csrc/.
There is no CPU fallback: if the library is missing or no CUDA device is present, calls raise.
"""
from .binding import Sldg, SldgError, lib, library_path, EXPORTS, AB, gauss_legendre, sipg_matrices, plan_query, plan_query_step_to, density_static, density_static_max_x  # noqa: F401
