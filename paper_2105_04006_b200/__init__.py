"""B200-native batched Lomb-Scargle periodogram (arXiv 2105.04006 hot path).

The product is the C-ABI CUDA library `liblsp_b200.so` (include/lsp.h, sources under csrc/); this package is
its thin Python binding.  There is no CPU fallback: the calls fail loudly without the library or a GPU.
"""
from .binding import (  # noqa: F401
    EXPORTS,
    LspConfig,
    LSP_FLAG_PAGEABLE_STAGED,
    LSP_STATIC_SCRATCH_BYTES,
    LspError,
    Plan,
    load_library,
    lsp_best_merge,
    lsp_best_period,
    lsp_best_period_static,
    lsp_destroy,
    lsp_periodogram_batched,
    lsp_periodogram_batched_host,
    lsp_periodogram_generalized,
    lsp_periodogram_generalized_host,
    lsp_plan_create,
    lsp_version,
)
