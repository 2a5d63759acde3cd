"""feds-b200: selective-encryption fragmentation of 8-bit images (arXiv 1512.02951 section 6) on one B200.

The product is the C-ABI CUDA library `libfeds.so` (include/feds.h, sources in csrc/); `binding` is its thin
ctypes wrapper. Build with `python -m paper_1512_02951_b200.build`. Importing `binding` without the built library
raises: there is no CPU fallback.
"""
