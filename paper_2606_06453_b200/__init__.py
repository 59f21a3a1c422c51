"""B200-native sparse decode hot path of arxiv/paper_2606_06453 (Vortex): C-ABI library
libvortex_b200.so (csrc/, include/vortex_b200.h) plus this thin binding.  No CPU fallback."""
from .binding import (Context, KvPool, PageTable, VortexError, alloc_summary, context_for, load_library,
                      tables_for, EXPORTS, LIB_PATH, VX_STEP_UPDATE_SUMMARY, VX_STEP_APPROX_TOPK, VX_OPT_MLA_STEP,
                      VX_MLA_STEP_AUTO, VX_MLA_STEP_FUSED, VX_MLA_STEP_CHAINED, VX_MLA_STEP_FLAT,
                      VX_OPT_MLA_FLAT_SPLITS, VX_OPT_MLA_FLAT_WAVES)

__all__ = ["Context", "KvPool", "PageTable", "VortexError", "alloc_summary", "context_for",
           "load_library", "tables_for", "EXPORTS", "LIB_PATH", "VX_STEP_UPDATE_SUMMARY", "VX_STEP_APPROX_TOPK",
           "VX_OPT_MLA_STEP", "VX_MLA_STEP_AUTO", "VX_MLA_STEP_FUSED", "VX_MLA_STEP_CHAINED", "VX_MLA_STEP_FLAT",
           "VX_OPT_MLA_FLAT_SPLITS", "VX_OPT_MLA_FLAT_WAVES"]
