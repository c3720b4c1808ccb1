"""paper_2606_07777_b200 -- B200-native dual-gradient hot path of the ridge-regularised matching-LP solver
(arxiv/paper_2606_07777).  The product is the C-ABI library `libdualip_b200.so` (include/dualip.h); this
package is its thin ctypes binding.  There is no CPU fallback: using the binding without the built library
or without a CUDA device raises.
"""
from .binding import (DualipError, Problem, Opts, Scalars, Info, lib_path, load_library,  # noqa: F401
                      PROJ_SIMPLEX_INEQ, PROJ_BOX, PROJ_BOXCUT, PROJ_SIMPLEX_EQ,
                      RED_AUTO, RED_SMEM, RED_GLOBAL, RED_CSC, PRECOND_NONE, PRECOND_JACOBI, STEP_FIXED, STEP_ADAPTIVE,
                      EXPORTED_SYMBOLS, grad_static, STATIC_MAX_DUALS, ETOOBIG, ESTALE, EHOOK)
