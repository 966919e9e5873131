"""B200-native neBEM hot path (arxiv 2606.24154): thin Python binding over the C ABI of include/neb.h.

Argument marshalling only — every step of the path (frame tables, influence matrix, LU, triangular
solves, field evaluation, space-charge sums) runs in the CUDA kernels of libneb.so.  There is no CPU
fallback: importing works without a GPU (so the library can be built and inspected), creating a
context does not.
"""
from .binding import (Neb, NebError, lib, lib_path, exported_symbols, NEB_RECT, NEB_TRI, NEB_WIRE,  # noqa: F401
                      NEB_BC_DIRICHLET, NEB_BC_DIELECTRIC, STAGES)
