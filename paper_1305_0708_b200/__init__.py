"""paper_1305_0708_b200 -- B200-native tree-level |M|^2 (hot path of arXiv:1305.0708).

csrc/   device function library, generated per-process kernels, the C-ABI (libhg.so; include/hg.h)
gen/    process generator: diagram enumeration, colour-flow algebra, CUDA emitter, flop counter
api.py  ctypes binding with the names of the C ABI
build.py  nvcc build of libhg.so for sm_100a
"""
