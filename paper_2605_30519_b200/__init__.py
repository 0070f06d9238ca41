"""B200-native OmniMem hot path (arxiv/paper_2605_30519): paged KV cache, block-key pooling,
Query-Shared KV Selection with Adaptive Window Exclusion, and Per-Head Scattered KV Access
attention, behind the C-ABI declared in ``include/omnimem.h``.

``paper_2605_30519_b200.binding`` is the thin Python binding (argument marshalling only);
``paper_2605_30519_b200.synth`` holds the seeded workload generators.  Importing this package
does not load the CUDA library; ``binding.load()`` does and fails loudly if it is missing.
"""
__all__ = ["binding", "synth"]
