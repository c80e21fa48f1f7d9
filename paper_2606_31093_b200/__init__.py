"""kvtier: B200-native paged-KV tier transfer (pack / unpack / offload / reload).

The hot path of Omni-Flow's Data Flow layer (sec. 4.1.1, sec. 4.1.2)
as hand-written sm_100a CUDA behind a C ABI (include/kvtier.h).  ``kvtier`` is the thin ctypes
binding (argument marshalling only); ``workloads`` holds the seeded input generators.
Importing the package does not load the CUDA library; ``paper_2606_31093_b200.kvtier`` does and
fails loudly when it is missing.
"""
__all__ = ["kvtier", "workloads"]
