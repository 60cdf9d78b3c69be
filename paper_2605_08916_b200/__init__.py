"""B200-native Diffusion Restore hot path (arXiv 2605.08916): thin Python binding over libdr.so (include/dr.h).

Every step of the path runs in the CUDA kernels of csrc/; this package only marshals arguments.  PyTorch is
used for device memory and streams.  There is no CPU fallback: importing `binding` raises if libdr.so is missing.
"""
from .binding import *  # noqa: F401,F403
