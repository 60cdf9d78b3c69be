"""B200-native Diffusion Restore hot path (arXiv 2605.08916): thin Python binding over libdr.so (include/dr.h).

Every step of the path runs in the CUDA kernels of csrc/; this package only marshals arguments.  PyTorch is
used for device memory and streams.  There is no CPU fallback: the first use of any name of the binding loads
libdr.so and raises ImportError if it is missing.  (`paper_2605_08916_b200.build` stays importable on a fresh
checkout, where the library does not exist yet.)
"""
import importlib

_SUBMODULES = ("build", "binding", "sharding")


def __getattr__(name):
    if name in _SUBMODULES:
        return importlib.import_module(f"{__name__}.{name}")
    binding = importlib.import_module(f"{__name__}.binding")   # raises ImportError when libdr.so is missing
    try:
        return getattr(binding, name)
    except AttributeError:
        raise AttributeError(f"module {__name__!r} has no attribute {name!r}") from None
