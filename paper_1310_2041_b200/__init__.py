"""paper_1310_2041_b200 -- B200-native short-range force pipeline of GALAMOST-style polymer MD.

The product is `libgm.so` (hand-written CUDA for sm_100a behind the C ABI of include/gm.h); this
package is its thin ctypes binding.  There is no CPU fallback: importing `gm` fails loudly if the
library has not been built (`python -m paper_1310_2041_b200.build`).
"""
from . import gm  # noqa: F401
from .gm import System  # noqa: F401
