"""paper_1311_5582_b200 -- thin Python binding of libea_b200.so (include/ea.h).

Argument marshalling only: every step of the path (bit-packed store, checkerboard sweep,
parallel-tempering swap, energy / overlap reductions) runs in the hand-written sm_100a
kernels of csrc/.  PyTorch is used for device memory (the workspace tensor) and the stream.
There is no CPU fallback: importing works without a GPU (so the symbol table can be
checked), creating a simulation does not.
"""
from .binding import (EA, EA_KERNEL_AUTO, EA_KERNEL_GENERIC, EA_KERNEL_RESIDENT, EA_KERNEL_TILED, EA_KERNEL_STREAM,
                      EA_KERNEL_REPLICA, EA_LAYOUT_REALIZATION_BITS, EA_LAYOUT_REPLICA_BITS, EA_SWAP_MOVE, EA_SWAP_PERMUTE,
                      EAError, exported_symbols, lib, library_path, measure_int_peak)

__all__ = ["EA", "EAError", "lib", "library_path", "exported_symbols", "measure_int_peak", "EA_KERNEL_AUTO",
           "EA_KERNEL_GENERIC", "EA_KERNEL_RESIDENT", "EA_KERNEL_TILED", "EA_KERNEL_STREAM", "EA_KERNEL_REPLICA",
           "EA_LAYOUT_REALIZATION_BITS", "EA_LAYOUT_REPLICA_BITS", "EA_SWAP_PERMUTE", "EA_SWAP_MOVE"]
