"""B200-native Barnes-Hut force pipeline of arxiv/paper_1106_1900 (Bonsai): CUDA library + thin binding.

``csrc/`` holds the sm_100a kernels and the C ABI of ``include/bh.h``; ``binding.py`` marshals arguments.
Nothing here imports ``oracle/`` (test infrastructure); there is no CPU fallback.
"""
from .binding import (BarnesHut, BhDomainBox, BhError, BhStats, LIB_PATH, STAGES, SYMBOLS, decode_domain_box,  # noqa: F401
                      direct_forces, domain_box_static, domain_box_static_max_n, load_library, probe_fp32, workspace_bytes)
from .pipeline import HostStepPipeline  # noqa: F401
from .sharded import ShardedBarnesHut, balanced_bounds, keep_own_rows, share_bounds, share_mask  # noqa: F401
