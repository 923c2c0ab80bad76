"""paper_2011_13926_b200 — B200-native (sm_100a, fp64) radiative-transfer step of the AP/WB M1 scheme of
arXiv 2011.13926 (ARK-RT).  The product is libark_m1.so (C ABI in include/ark_m1.h, CUDA sources in csrc/);
this package only builds it (build.py) and binds it (binding.py)."""
from .binding import (ArkM1, load_library, version, fastmath_errors, fp64_issue_rate, ArkM1Group, ArkM1_3D, ArkHostTransport, gloo_host_transport, nccl_unique_id, slab_range, noalloc_setup, noalloc_max_cells, count_unrealizable_noalloc, SYMBOLS, LIB_PATH,  # noqa: F401
                      BC_PERIODIC, BC_DIRICHLET, BC_OUTFLOW, XLO, XHI, YLO, YHI)
