"""B200-native (sm_100a) nuclear-pasta molecular dynamics hot path of arXiv:1412.8502.

`Sim` wraps the C-ABI CUDA library declared in include/pasta.h; `inputs` holds the seeded synthetic
workloads.  Importing this package loads neither torch nor the CUDA library.
"""
from . import inputs  # noqa: F401
from .binding import Env, Params, PastaError, Sim, default_params, library_path, load, shard_bounds  # noqa: F401
