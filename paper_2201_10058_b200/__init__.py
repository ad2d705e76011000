"""B200-native GENGA kick + close-encounter pre-check (arXiv 2201.10058, eq. 3 / eq. 62-63 / App. A).

The product is the C-ABI library libgenga_kick.so (include/genga_kick.h, csrc/); this package is
its thin ctypes binding.  It never imports oracle/ and has no CPU fallback."""
from .binding import (kick_list_static, STATIC_EXPORTS, STATIC_MAX_BODIES, E_STATIC_MAX, GengaKick, GengaKickConfig, GengaKickPlan, GengaKickError, lib, make_plan, make_plan_tp2, make_plan_sym, make_plan_tprows, plan_sym_row_begin,
                      plan_sym_row_of, plan_cta_range, plan_iblock_ctas, strerror, EXPORTS, STEP_EXPORTS, GROUP_EXPORTS, BS_EXPORTS, SENC_EXPORTS, GengaSencConfig, STATUS_BAD_PAIR, STATUS_GROUP_TOO_LARGE, STATUS_BS_NOT_CONVERGED, LIB_PATH, STATUS_COINCIDENT, STATUS_CAND_OVERFLOW, STATUS_FX_RANGE, STATUS_UNBOUND,
                      OK, E_NULL, E_ALIGN, E_SIZE, E_LEVEL, E_CUDA, E_NOMEM, ORDER_AUTO, ORDER_CALLER, ORDER_SORTED)

__all__ = ["kick_list_static", "STATIC_EXPORTS", "STATIC_MAX_BODIES", "E_STATIC_MAX", "GengaKick", "GengaKickConfig", "GengaKickPlan", "GengaKickError", "lib", "make_plan", "make_plan_tp2", "make_plan_sym", "make_plan_tprows",
           "plan_sym_row_begin", "plan_sym_row_of", "plan_cta_range", "plan_iblock_ctas", "strerror", "EXPORTS", "STEP_EXPORTS", "GROUP_EXPORTS", "BS_EXPORTS", "SENC_EXPORTS", "GengaSencConfig", "STATUS_BAD_PAIR", "STATUS_GROUP_TOO_LARGE", "STATUS_BS_NOT_CONVERGED", "LIB_PATH", "STATUS_COINCIDENT", "STATUS_CAND_OVERFLOW", "STATUS_FX_RANGE", "STATUS_UNBOUND",
           "ORDER_AUTO", "ORDER_CALLER", "ORDER_SORTED", "OK", "E_NULL", "E_ALIGN", "E_SIZE", "E_LEVEL", "E_CUDA", "E_NOMEM"]
