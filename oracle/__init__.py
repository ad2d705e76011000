"""CPU oracle of the GENGA kick + encounter pre-check.  TEST INFRASTRUCTURE ONLY.

Importable only from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference legs.
The arithmetic lives in genga_kick_oracle.c (plain C, binary64 per pair, long double sums) and
genga_step_oracle.c (Rcrit / HC / FG, long double), genga_detect_oracle.c (detection), genga_group_oracle.c (grouping), genga_bs_oracle.c (Bulirsch-Stoer); this
module is argument marshalling via ctypes.  It imports nothing from the CUDA package.
"""
from .oracle import (OracleResult, ListKickResult, K_of_y, K, weight, weight_bs, kick, kick_list, pair_set, num_threads,
                     lib_path)

from . import step
from . import group
from . import bs
from . import detect

__all__ = ["step", "group", "bs", "detect", "OracleResult", "K_of_y", "K", "weight", "weight_bs", "kick", "kick_list", "ListKickResult", "pair_set", "num_threads", "lib_path"]
