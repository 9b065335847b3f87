"""B200-native GPU stage of FusionANNS (arxiv 2409.16576): thin Python binding of the
C-ABI library declared in include/fann.h.  Every step of the path runs in the CUDA
kernels of csrc/; this package only marshals arguments.  Importing it does not load
the library; the first call does, and fails loudly if libfann.so is missing."""
from .binding import *  # noqa: F401,F403  (every fann_* mirror, FannIndex, FannError, the constants)
from .binding import library_path, load_library  # noqa: F401
