"""B200-native hot path of the MPR prediction method (arxiv/paper_1910_08448).

`mpr` is the ctypes binding of the C-ABI CUDA library (include/mpr.h); `inputs` holds the seeded
synthetic input generators (none of the method's arithmetic); `build` compiles libmpr.so.
"""
