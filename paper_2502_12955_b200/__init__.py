"""B200 (sm_100a) lattice Boltzmann hot path of CooLBM (arXiv 2502.12955): a C-ABI CUDA library
(include/lbm.h, csrc/) and this thin binding.  No CPU fallback; see DESIGN.md."""
from .lbm import (LBM, LbmError, LbmParams, SYMBOLS, LIB_PATH, lattice_table, lib, make_params,  # noqa: F401
                  D2Q9, D3Q19, BGK, SC1, SC2, SC2_ADE, BGK_T)
