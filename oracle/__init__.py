"""ORACLE package — test infrastructure only (see chunk_attention.py header). Never imported by the
product path (`paper_2606_15319_b200`), which fails loudly when its CUDA library is missing."""
from .chunk_attention import (attend_rows, chunk_attention, error_metrics, gather_kv, kv_append,  # noqa: F401
                              kv_transfer, lse_merge, to_f64, token_positions, token_slots, visible_tokens)
from . import fp8_attention  # noqa: F401  (NEXT-3: e4m3 quantiser, quantising append, attention over dequantised operands)
