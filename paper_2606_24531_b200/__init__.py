"""B200-native (sm_100a) block-parallel decode of the ACEAPEX-style two-layer codec of
arxiv/paper_2606_24531: per-block 32-lane interleaved rANS (entropy layer) and absolute-offset
LZ copies (match layer), plus the single-coordinate seek. See DESIGN.md and FORMAT.md.

``paper_2606_24531_b200.binding`` is the thin ctypes binding over the C-ABI library
(``include/aceapex.h``); ``paper_2606_24531_b200.workloads`` holds the seeded input generators.
"""
__all__ = ["binding", "workloads"]
