"""B200-native weighted-NMF hot path of arXiv 2309.04623 (fit -> project -> subtract).

The compute lives in hand-written sm_100a CUDA kernels behind the C-ABI library
declared in include/nmf.h; `paper_2309_04623_b200.nmf` is a thin ctypes binding
(argument marshalling only).  There is no CPU fallback: importing the binding on
a box without the built library raises.
"""
