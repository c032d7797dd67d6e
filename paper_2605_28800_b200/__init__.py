"""B200-native (sm_100a) TDGL hot path of arxiv/paper_2605_28800: C-ABI library libfe_b200 + ctypes binding.

    from paper_2605_28800_b200 import Grid, fe_rhs, fe_step, ...

The CUDA library is required (build it with `python -m paper_2605_28800_b200.build`); there is no CPU path.
"""
from .binding import *            # noqa: F401,F403
from .binding import Grid, FeError, load, lib_path, SYMBOLS   # noqa: F401
