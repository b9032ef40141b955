"""ebic-b200: B200-native fitness evaluation + row-bitmask extraction for EBIC (arXiv 1807.09932).

`workloads` is importable without the CUDA library; everything in `binding` needs
`libebic.so` (built by `paper_1807_09932_b200/csrc/build.py` or `__graft_entry__.build()`)
and fails loudly if it is missing -- there is no CPU fallback.
"""
__all__ = ["workloads", "binding", "sharded"]
