"""B200-native paged-KV mixed-batch attention (kv_append, batch_attention, step timer).

The product path is the C-ABI library ``libpa_b200.so`` (include/pa.h) built from ``csrc/``;
``binding`` only marshals arguments.  There is no CPU fallback: every entry point raises if the
CUDA library is missing.  ``synth`` (seeded inputs) is importable without a GPU.
"""
__all__ = ["binding", "synth"]
