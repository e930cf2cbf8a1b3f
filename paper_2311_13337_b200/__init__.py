"""tvbx: B200-native batched TVB-AdEx parameter-sweep integrator (arxiv 2311.13337 hot path).

The product is the C-ABI library `libtvbx.so` (include/tvbx.h; sources in csrc/); this package is
its thin Python binding.  See DESIGN.md.
"""
from .binding import (Connectome, Sweep, TvbxError, build, default_params, lib, sweep_from_config, trim_memory, diag_tf_closed2,  # noqa: F401
                      PARAM_IDS, N_PARAMS, TVBX_F32, TVBX_F64, TVBX_FC_AUTO, TVBX_FC_FP32, TVBX_FC_TF32, LIB_PATH, EXPORTS)
