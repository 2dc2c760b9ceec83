"""B200-native (sm_100a) bundle-adjustment hot path after arxiv 2605.30583 ("Caspar").

One Levenberg-Marquardt iteration = per-observation residual + Jacobian linearization of a
9-parameter camera and a 3-D point, then a matrix-free block-Jacobi preconditioned CG solve on the
point-eliminated (Schur) normal equations.  The product is the C-ABI library
`libcaspar_ba.so` (include/caspar_ba.h, csrc/); this package only marshals arguments to it.
"""
from .binding import (CasparBA, CasparError, PcgInfo, Stats, Step, StepInfo, EXPORTED_SYMBOLS,  # noqa: F401
                      load_library, library_path, plan_layout, cost_static, STATIC_MAX_CAMERAS)
from .binding import RESIDUALS, JC, JP, U, V, G, SCHUR_RHS, DELTA, PRECONDITIONER  # noqa: F401
from .binding import OK, EINVAL, ECUDA, ENOMEM, ENUMERIC, ESTATE  # noqa: F401
from . import sharding  # noqa: F401
