"""B200-native TTT global-context-memory hot path (Scal3R, arxiv/paper_2604_08542).

The product is the C-ABI library `libttt_b200.so` (include/ttt.h); this package is the thin
Python binding over it (argument marshalling only — every step of the path runs in the CUDA
kernels). PyTorch is used for device memory and streams. There is no CPU fallback: importing
`binding` raises if the library has not been built (`python -m paper_2604_08542_b200._build`).
"""
from .binding import (TTT, TTTError, TTT_BF16, TTT_F32, lib_path, load_library, version)  # noqa: F401
