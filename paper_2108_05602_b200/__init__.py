"""paper_2108_05602_b200 - B200-native (sm_100a) cross-spectrum fringe search, the data-parallel hot
path of VOLKS2 (arXiv 2108.05602).  The product is libvolks_b200.so (C-ABI, include/volks.h);
this package is its thin binding."""
from .binding import (CAND_DTYPE, DETECTION_DTYPE, PEAK_DTYPE, PULSE_DTYPE, Plan, VolksError,  # noqa: F401
                      allif_search, baseline_match, bin_to_physical, cal_phasors, dm_shifts, fringe_search, lib, make_options, measure_fp32_peak, plan_create_raw, search_noalloc,
                      volks_options, window_match)
