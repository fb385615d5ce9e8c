"""pCMD forward model, Hess diagram and log-likelihood (arXiv:1904.00011) on B200.

The product is libpcmd.so (include/pcmd.h); this package is the thin Python binding.  It never
imports oracle/ and has no CPU fallback: without the CUDA library and a GPU it raises."""
from .binding import (Pcmd, PcmdError, lib, LIKE_POISSON, LIKE_GAUSS, LIKE_GAUSS_LITERAL,  # noqa: F401
                      exported_symbols, philox, pipe_bench, params_from_paper)
