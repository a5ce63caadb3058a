"""B200-native brute-force incoherent de-dispersion (arxiv 1111.6399, ARTEMIS hot path).

``out[d][t] = sum_c in[c][t + s(c,d)]`` for every trial DM of a plan (§2).
The product is the C-ABI library ``libdedisp_b200.so`` (``include/dedisp.h``); this
package is its thin ctypes binding plus the config/synthetic-input modules.
"""
from .configs import CONFIGS, SurveyConfig, shrink, paper_sweep  # noqa: F401
from .api import (Plan, Stream, DedispError, shift_table_host, lib,  # noqa: F401,E402
                  KERNEL_AUTO, KERNEL_NAIVE, KERNEL_TILED, KERNEL_SUBBAND, detect, detect_static, CAND_DTYPE)
