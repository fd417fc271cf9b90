"""B200-native GBEES prediction step (arXiv 2508.13986): thin ctypes binding over libgbees.so.

Every step of the path runs in the hand-written CUDA kernels behind the C ABI of include/gbees.h;
this package only marshals arguments. There is no CPU fallback: importing `binding` without the
built extension raises.
"""
from .binding import Gbees, GbeesError, HashTable, lib_path  # noqa: F401
