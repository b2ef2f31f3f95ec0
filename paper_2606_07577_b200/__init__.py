"""B200-native OmniMem per-chunk KV-cache compression step (arxiv/paper_2606_07577).

`paper_2606_07577_b200.omnimem` is the thin Python binding of the C-ABI library
(include/omnimem.h); `paper_2606_07577_b200.inputs` draws the seeded synthetic workloads.
The binding loads `libomnimem.so` on first use and raises if it is missing: there is no CPU fallback.
"""
__all__ = ["inputs", "omnimem"]
