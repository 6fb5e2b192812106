"""ExpertFlow MoE expert layer over a GPU expert cache -- B200-native (sm_100a) C-ABI library + thin binding.

The compute lives in ``libef.so`` (``csrc/``, declared in ``include/ef.h``).  This package only marshals
arguments.  There is no CPU fallback: if the library is missing or no CUDA device is present, calls fail.
"""
from .binding import (EfError, EfContext, EfConfig, CacheStats, load_library, library_path,  # noqa: F401
                      exported_symbols, DECLARED_SYMBOLS, DIAG_SYMBOLS, EF_OPT_SPLITK, EF_OPT_WAVE_BYTES,
                      EF_OPT_CHUNK_MIN_BYTES, EF_OPT_FUSED_WAVES, EF_OPT_TOKEN_SCHED_PATH, EF_OPT_COPY_ORDER, EF_OPT_EARLY_RELEASE)
from .layer import MoELayerRunner, DualBatchRunner  # noqa: F401
