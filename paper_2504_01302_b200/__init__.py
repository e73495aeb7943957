"""glad-b200: batched joint lensing + dynamics log-likelihood (arXiv 2504.01302) as hand-written
sm_100a CUDA kernels behind the C ABI in include/glad.h.  `Glad` is the thin Python binding."""
from .binding import (EXPORTS, LIGHT_CHAMELEON, LIGHT_SERSIC, FLAG_BIN_INVALID, FLAG_DYN_INVALID, FLAG_LENS_INVALID, FLAG_PIXSRC_NOT_PD, LENS_NOALLOC_MAX_B, NDYN, NLENS, NPROF, PROFILE_CHAMELEON, PROFILE_NFW_CSE, PROFILE_EPL, PROFILE_SERSIC, Glad,  # noqa: F401
                      GladError, bh_theta2, load)
from .build import build  # noqa: F401
from .sharding import gather_loglike, shard_range  # noqa: F401
