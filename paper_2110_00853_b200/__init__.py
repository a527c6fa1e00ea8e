"""B200-native nodal-DG right-hand side for atmospheric LES (hot path of arXiv 2110.00853).

The product is the CUDA library ``libcm_dg.so`` (C ABI in ``include/cm_dg.h``); this package is a thin
ctypes binding with the same entry-point names.  PyTorch is used only for device memory and streams.
There is no CPU fallback: importing ``binding`` fails loudly if the library has not been built
(``python -m paper_2110_00853_b200.build``), and ``cm_dg_setup`` fails without a CUDA device.
"""
from .binding import (CmDg, CmDgError, cm_dg_coords, cm_dg_destroy, cm_dg_diagnostics, cm_dg_diagnostics_static, cm_dg_gradient,  # noqa: F401
                      cm_dg_last_error, cm_dg_layout, cm_dg_lsrk_step, cm_dg_lsrk_step_host, cm_dg_lsrk_step_table, cm_dg_filter,
                      cm_dg_metrics, cm_dg_profiles,
                      cm_dg_profile_begin, cm_dg_profile_end, cm_dg_rhs, cm_dg_rhs_host, cm_dg_setup, library_path)  # noqa: F401
