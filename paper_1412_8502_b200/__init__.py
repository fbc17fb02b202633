"""B200-native (sm_100a) nuclear-pasta molecular dynamics hot path of arXiv:1412.8502.

`Sim` wraps the C-ABI CUDA library declared in include/pasta.h; `inputs` holds the seeded synthetic
workloads.  Importing this package loads neither torch nor the CUDA library.
"""
from . import inputs  # noqa: F401
from .binding import (CLUSTERS_NOALLOC_MAX_N, Env, Params, PastaError, Sim, clusters_noalloc,  # noqa: F401
                      default_params, library_path, load, shard_bounds)
