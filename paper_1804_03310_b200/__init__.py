"""B200-native phaseless-AFQMC walker step (arXiv:1804.03310): C-ABI CUDA library + ctypes binding."""
from .binding import (AFQMC_ECUDA, AFQMC_EINVAL, AFQMC_ENOMEM, AFQMC_EUNSUPPORTED, AFQMC_OK, FLAG_KILLED,
                      FLAG_NONFINITE, FLAG_SINGULAR, LIB_PATH, SYMBOLS, AfqmcContext, AfqmcError, AfqmcParams,
                      afqmc_peak_probe, afqmc_query_bytes, load_library, make_params)

__all__ = ["AfqmcContext", "AfqmcError", "AfqmcParams", "afqmc_peak_probe", "afqmc_query_bytes", "load_library", "make_params",
           "LIB_PATH", "SYMBOLS", "AFQMC_OK", "AFQMC_EINVAL", "AFQMC_EUNSUPPORTED", "AFQMC_ECUDA", "AFQMC_ENOMEM",
           "FLAG_SINGULAR", "FLAG_NONFINITE", "FLAG_KILLED"]
