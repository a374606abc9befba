"""B200-native LIETS-QSGS growth path (arxiv/paper_2602_11734): thin Python binding of libliets.so.

Everything the method computes runs in the hand-written sm_100a kernels behind the C ABI of
``include/liets.h``; this package only marshals arguments.  PyTorch supplies device memory
(the workspace and output buffers) and the CUDA stream.  There is no CPU fallback: loading fails
loudly if the library has not been built, and every call fails without a CUDA device.
"""
from .liets import (Liets, LietsBatch, LietsError, lib, library_path, OK, FRONT_EMPTY, MAX_STEPS,  # noqa: F401
                    E_ARG, E_STATE, E_CAPACITY, E_CUDA,
                    BOUNDARY_WALL, BOUNDARY_PERIODIC, BOUNDARY_PERIODIC_XY, STORAGE_U8, STORAGE_TILE, STORAGE_FULL, LAW_CONSTANT, LAW_EQ1,
                    FORMAT_U8, FORMAT_BITS, S2_STATIC_MAX_LAGS, ORDER_INDEX, ORDER_KEYED, SPACING_SPARSE, SPACING_DENSE, EXPORTS)
