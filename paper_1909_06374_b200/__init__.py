"""paper_1909_06374_b200 -- B200-native light-curve generator (hot path of Sartori et al. 2019).

The product is the C-ABI CUDA library libagnvar.so (include/agnvar.h, csrc/); this package is its thin
Python binding plus the seeded workload descriptions.  No CPU fallback exists: importing a call without
the compiled library raises.
"""
from .binding import (AGNVAR_ERDF_BPL, AGNVAR_ERDF_LOGNORMAL, AGNVAR_F32, AGNVAR_F64, AgnvarError,  # noqa: F401
                      agnvar_e13_iterate, agnvar_erdf_sample_sorted, agnvar_erdf_table, agnvar_philox_u32, agnvar_periodogram, agnvar_psd_bpl,
                      agnvar_tk_generate, agnvar_structure_function, agnvar_delta_m_prob, agnvar_ensemble_sf, agnvar_moments, agnvar_slice_sample_sorted, agnvar_structure_function_static, static_scratch_bytes, static_scratch_need, free_workspace, launch_count, lib, strerror, trace_begin, trace_end, version, workspace_bytes)
from .pipeline import generate_light_curves  # noqa: F401
from . import workloads  # noqa: F401
