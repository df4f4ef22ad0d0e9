"""paper_1206_0919_b200 -- B200-native dimensionally split relativistic SHASTA (arXiv:1206.0919).

`Shasta` (paper_1206_0919_b200.shasta) is the thin binding over the C-ABI library
`csrc/libshasta.so` (include/shasta.h).  Importing the package does not load CUDA; the
binding fails loudly when the library is missing -- there is no CPU fallback.
"""

__all__ = ["Shasta", "inputs"]


def __getattr__(name):
    if name == "Shasta":
        from .shasta import Shasta
        return Shasta
    raise AttributeError(name)
