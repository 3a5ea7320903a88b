"""paper_2001_02765_b200 -- B200 (sm_100a) direct self-gravity of a thin disk on block-structured AMR.

Thin ctypes binding over the C ABI of include/sg_disk.h (argument marshalling only; every step of
the path runs in the CUDA kernels of csrc/).  There is no CPU fallback: if libsg_disk.so is missing
the import of :mod:`.binding` fails loudly.
"""
from .binding import (SgDisk, SgError, lib_path, load_library, measure_fp64_peak, measure_fp64_mma_peak, version,  # noqa: F401
                      shard_range, EXPORTED_SYMBOLS, force_uniform_static)
