"""B200-native 2-D BGK-UGKS time step (arXiv:1810.08137): thin Python binding of libugks.

The product is the C-ABI library ``libugks.so`` (include/ugks.h; CUDA for sm_100a in csrc/).  This package only
marshals arguments: torch supplies device memory and the stream, every step of the path runs in the CUDA kernels.
There is no CPU fallback: if the extension is missing or no GPU is present, calls raise.
"""
from .binding import Ugks, UgksError, jit_check, lib, library_path, residual_noalloc  # noqa: F401
