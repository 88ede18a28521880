"""B200-native NOLSM hot path (arXiv 2205.12182): thin Python binding over the C-ABI library
libnolsm.so (include/nolsm.h). Importing this package does not load the library; `Nolsm(...)` does,
and raises if the CUDA extension is missing -- there is no CPU fallback."""
from .binding import (DTYPE_F32, DTYPE_F64, ENGINE_AUTO, ENGINE_PERSISTENT, ENGINE_ROUNDS, GEMM_AUTO, GEMM_SIMT, GEMM_UMMA, ITER_EQ6, ITER_LOWDIN, PREC_FP16_FP32, PREC_FP32, Nolsm,
                      NolsmError, NolsmOptions, NolsmStats, lib_path, load_library)

__all__ = ["Nolsm", "NolsmError", "NolsmOptions", "NolsmStats", "load_library", "lib_path", "PREC_FP16_FP32",
           "PREC_FP32", "DTYPE_F64", "DTYPE_F32", "GEMM_AUTO", "GEMM_UMMA", "GEMM_SIMT", "ENGINE_AUTO", "ENGINE_PERSISTENT", "ENGINE_ROUNDS", "ITER_EQ6", "ITER_LOWDIN"]
