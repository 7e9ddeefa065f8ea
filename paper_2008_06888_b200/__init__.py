"""B200-native tropical tensor-network sweep for spin-glass ground states (arXiv 2008.06888).

The product is the C-ABI CUDA library ``libttn.so`` (include/ttn.h, csrc/); this package is the
thin binding with the same names.  There is no CPU path.
"""
from .ttn import (  # noqa: F401
    TROPICAL_F32, COUNTING_F32_F64, TROPICAL_I16, CALL_ENERGY, CALL_COUNT, CALL_CONFIG, CALL_ENERGY_I16, CALL_ENERGY_Z2, CALL_COUNT_Z2, CALL_ENERGY_I16_Z2, CALL_CONFIG_Z2, EXPORTS,
    TTNError, Plan, lib, workspace_bytes, alloc_workspace, plan_describe,
    sweep_energy, sweep_energy_i16, sweep_count, ground_config, potts3_sweep_energy, potts3_sweep_count,
    chimera_workspace_bytes, chimera_sweep_energy_i16, chimera_count_workspace_bytes, chimera_sweep_count,
    sweep_energy_noalloc, NOALLOC_SCRATCH_BYTES,
)
