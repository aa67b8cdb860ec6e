"""B200-native hot path of the GPU-aware OpenSHMEM auxiliary specification (arxiv/paper_2607_08006).

Thin ctypes binding over the C-ABI library `libshmemg.so` (include/shmemg.h): argument marshalling only,
every step of the path runs in the library's sm_100a kernels.  PyTorch is used for device memory and
streams.  There is no CPU fallback: importing `binding` raises if the library has not been built.
"""
from .binding import (CAP, CMP, ERR, OP, OP_DTYPE, SIGNAL, TEAM, Batch, ShmemgError, World, lib)  # noqa: F401
