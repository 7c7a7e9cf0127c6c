"""B200-native batched evaluation of algorithmic Matsubara integration (arXiv 2311.17189).

The product is the C-ABI library ``libami_b200.so`` (``include/ami.h``); this package is its
thin Python binding.  Importing the package does not load the library; the first call does and
raises if it has not been built."""
from .binding import (AmiError, AmiTable, PLAN_AUTO, PLAN_FLAT, PLAN_REG, PLAN_TREE, PLAN_UNORDERED, EXPORTS, LIB_PATH,  # noqa: F401
                      fp64_peak_probe, kernel_launches, lib, search_sum_order, read_graph, label_graph, ORDER_FEWEST_TERMS,
                      ORDER_FEWEST_OPS, BAND_TIGHT_BINDING, BAND_FREE, tally_static, tally_static_setup,
                      TALLY_STATIC_MAX_ROWS)
