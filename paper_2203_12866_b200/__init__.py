"""cosenu-b200: the COSEnu (arXiv 2203.12866) RK4 hot path as hand-written sm_100a CUDA behind a C ABI.

Importing the package does not load the CUDA library; `paper_2203_12866_b200.binding` does, and
fails loudly if it is missing.  There is no CPU fallback.
"""
