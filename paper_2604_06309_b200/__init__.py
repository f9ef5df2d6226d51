"""B200-native (sm_100a, fp64) DMFE history-integral path of arxiv/paper_2604_06309.

The product is the C-ABI library `libdmfe.so` (include/dmfe.h, csrc/); `dmfe.py` is the thin
ctypes binding of the same names.  There is no CPU fallback: every entry point raises if the
CUDA library is missing."""
