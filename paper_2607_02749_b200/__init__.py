"""paper_2607_02749_b200 -- B200-native batched VQE energy engine (hot path of Graph-VQE, arxiv/paper_2607_02749).

Thin Python binding over the C-ABI library libgvqe.so (include/gvqe.h); see DESIGN.md.
"""
from .binding import (  # noqa: F401
    Gvqe, GvqeError, GvqeLayout, load, lib_path, EXPORTS, argmax_noalloc, NOALLOC_MAX_AMPLITUDES, cobyla_minimize,
    GVQE_OK, GVQE_ERR_INVALID_ARG, GVQE_ERR_NO_HAMILTONIAN, GVQE_ERR_WORKSPACE, GVQE_ERR_UNSUPPORTED, GVQE_ERR_CUDA,
    GVQE_C64, GVQE_C128,
)
from .build import build  # noqa: F401
