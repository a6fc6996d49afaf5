"""CPU oracle for the stream-loading-prefill MoE layer (TEST INFRASTRUCTURE ONLY).

This package is a plain, slow, obviously-correct numpy implementation of what the hot path
computes (restated in DESIGN.md §3).  It is written from the paper
(`/root/reference/PAPER.md`, cited per function as PAPER.md:<line>) and shares no code with the
CUDA path under `paper_2606_10493_b200/`: neither imports the other.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import it.  The product path never does.

Parity pins (what each function is checked against, other than itself) are listed in
DESIGN.md §3.3 and implemented in `tests/test_oracle_*.py`.  The *output values* of a whole
layer are "parity unpinned" by the paper (it prints no activations); they are pinned only by the
closed forms / special cases / brute-force checks listed there.
"""

from .e4m3 import e4m3_decode, e4m3_encode_rne, E4M3_MAX  # noqa: F401
from .moe_layer import (  # noqa: F401
    bf16_bits_to_f64,
    f64_to_bf16_bits,
    quantize_rows_1x128,
    dequantize_rows_1x128,
    dequantize_weight_128x128,
    router,
    permutation,
    expert_ffn,
    moe_layer,
)
