"""paper_1809_00995_b200 -- B200-native (sm_100a) hot path of arXiv 1809.00995: the Abelian-Higgs string
network leapfrog update and its diagnostics.  The product is the C-ABI library csrc/libahs.so (include/ahs.h);
`binding` is its thin ctypes mirror.  Nothing in this package imports oracle/ (test infrastructure)."""

__all__ = ["binding", "build", "synthetic"]
__version__ = "0.1"
