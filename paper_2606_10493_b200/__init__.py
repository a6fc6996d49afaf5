"""B200-native stream-loading-prefill MoE layer (arxiv/paper_2606_10493, §3.1).

`binding` wraps the C-ABI library `libslpmoe.so` (include/slp_moe.h) one-to-one; `inputs` holds
the seeded synthetic-input generators.  The library is loaded on first use and the load fails
loudly if it has not been built (`python __graft_entry__.py` builds it); there is no CPU or
PyTorch fallback for any step of the path.
"""

from . import inputs, sharding, smallep  # noqa: F401
from .binding import (  # noqa: F401
    SlpMoeLayer, SlpError, lib, library_path, measure_h2d_gbs, query_plan, finalize_partial, EXPORTED_SYMBOLS,
    permute_static, permute_static_rows,
)
