"""DF-SSM per-token decode step for one B200: Python binding of the C-ABI library libdfssm.so.

Argument marshalling only -- every step of the path runs in the CUDA kernels of csrc/.
PyTorch is used for device memory and the stream.  There is no CPU fallback.
"""
from .binding import (DfssmError, Config, Model, Scheduler, lib, lib_path, TAPS, KCLASSES, EXPORTED_SYMBOLS,
                      dfssm_arena_bytes, head_noalloc, head_noalloc_scratch_need, NOALLOC_SCRATCH_BYTES)

__all__ = ["DfssmError", "Config", "Model", "Scheduler", "lib", "lib_path", "TAPS", "KCLASSES", "EXPORTED_SYMBOLS",
           "dfssm_arena_bytes", "head_noalloc", "head_noalloc_scratch_need", "NOALLOC_SCRATCH_BYTES"]
