"""B200-native forward Monte Carlo shortwave photon tracer (arxiv 2208.05247 §2.3).

The product is the C-ABI library declared in include/rt.h (CUDA kernels for sm_100a in csrc/);
this package is its thin Python binding.  No CPU fallback exists."""
from .binding import (Grid, Tallies, RtError, rt_counters, lib, philox_words, tally_to_flux, counters_of, W0, LIB_PATH, EXPORTS,  # noqa: F401
                      FATE_ATM_ABS, FATE_SFC_ABS, FATE_TOD_EXIT, FATE_CAPPED, FATE_ROULETTE, MODE_ANALOG, MODE_WEIGHTED,
                      majorant_no_alloc, NO_ALLOC_MAX_CELLS, selftest_ieee)
