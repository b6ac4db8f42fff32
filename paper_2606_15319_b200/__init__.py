"""B200-native ragged, paged chunk attention (slack_kv_append / slack_plan / slack_chunk_attention).

The CUDA extension (csrc/ -> libslack.so) is loaded lazily by `paper_2606_15319_b200.binding`;
importing the package alone (e.g. for `workloads`) needs neither a GPU nor the built library.
"""
__all__ = ["workloads", "metrics", "binding", "build"]
